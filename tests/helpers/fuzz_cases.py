"""Seeded random test cases for the fuzz parity test (tests/test_gpu_fuzz.py): a network, initial
counts, library options and run limits per seed.  Input construction only -- no arithmetic of the
method.  The recipe varies what the fixed configs keep constant:

  * generator: random mass-action (configs 3/5a recipe) or protein-interaction (config 4 recipe),
    M from 2 to ~8e4 (log-uniform), 1 to 100 reactions per species;
  * rates: as generated / 30 % zeros / 10^U(-6,3) / all equal (near-ties) / one decimal digit;
  * reactant coefficients: as generated, or a fifth of them raised to sigma = 3;
  * counts: as generated / 0..3 (mostly zero propensities, early absorption) / sparse / 0..1e6 / 0..29;
  * options: kernel (candidate-first / plain), exchange (cluster / L2), CTAs per trajectory,
    state in shared / global memory, prefetch bits, X replicas, refresh mode.
"""
import math

import numpy as np

import rt_workloads as W

BUNDLE_CTAS = [0, 1, 2, 3, 5, 7, 12, 13, 16, 17, 37, 74, 148]


def make_case(seed, max_reactions=80_000):
    """Returns (net, x0, options, max_firings, trajectory)."""
    r = np.random.default_rng(1_000_003 * seed + 17)
    kind = r.choice(["rma", "rma", "rma", "ppi"])
    M = min(int(10 ** r.uniform(0.3, 4.9)), max_reactions)
    N = max(1, int(M / 10 ** r.uniform(0.0, 2.0)))
    if kind == "rma":
        net, x0 = W.random_mass_action(N, M, seed=seed)
    else:
        net, x0 = W.protein_interaction(max(8, N), max(4, M // 2), seed=seed)
    net = dict(net)
    M, N = int(net["n_reactions"]), int(net["n_species"])
    rate = np.array(net["rate"], dtype=np.float64)
    mode = r.integers(0, 6)
    if mode == 1:
        rate[r.random(M) < 0.3] = 0.0
    elif mode == 2:
        rate = 10.0 ** r.uniform(-6, 3, size=M)
    elif mode == 3:
        rate[:] = 0.5
    elif mode == 4:
        rate = np.round(rate, 1) + 0.1
    net["rate"] = rate
    sigma = np.array(net["react_sigma"], dtype=np.int32)
    cubic = False
    if r.random() < 0.25 and len(sigma):
        sel = r.random(len(sigma)) < 0.2
        sigma[sel] = 3
        cubic = bool(sel.any())
    net["react_sigma"] = sigma
    xm = r.integers(0, 5)
    if xm == 1:
        x0 = r.integers(0, 4, size=N).astype(np.int64)
    elif xm == 2:
        x0 = (r.random(N) < 0.2).astype(np.int64) * r.integers(1, 50, size=N)
    elif xm == 3 and not cubic:
        x0 = r.integers(0, 1_000_000, size=N).astype(np.int64)
    elif xm == 4:
        x0 = r.integers(0, 30, size=N).astype(np.int64)
    if cubic:
        x0 = np.minimum(x0, 2000)          # counts stay below the 2^21-1 bound of sigma = 3
    opts = []
    if r.random() < 0.5:
        opts.append(("pipeline", int(r.integers(0, 2))))
    if r.random() < 0.5:
        opts.append(("exchange", int(r.integers(0, 2))))
    if r.random() < 0.7:
        opts.append(("bundle_ctas", int(r.choice(BUNDLE_CTAS))))
    if r.random() < 0.25:
        opts.append(("state_mode", 1))
    if r.random() < 0.3:
        opts.append(("prefetch", int(r.integers(0, 8))))
    if r.random() < 0.15:
        opts.append(("x_replicas", int(r.choice([2, 4]))))
    if r.random() < 0.1:
        opts.append(("refresh_mode", 1))
    firings = int(10 ** r.uniform(2.0, 3.4))
    return net, np.ascontiguousarray(x0, dtype=np.int64), opts, firings, int(r.integers(0, 1000))


# The simplest path through the library: one CTA, pass-then-reduce kernel, state streamed from
# global memory, every propensity recomputed every firing (the paper's own scheme), no prefetch.
REFERENCE_OPTIONS = [("pipeline", 0), ("bundle_ctas", 1), ("state_mode", 1), ("prefetch", 0),
                     ("refresh_mode", 1)]

INF = math.inf


# ---- cases for the other entry points and modes (tests/test_gpu_fuzz.py, second test) ---------
SIMPLE_OPTIONS = [("pipeline", 0), ("bundle_ctas", 1), ("state_mode", 1), ("prefetch", 0)]
MODES = ["ensemble", "ensemble", "resume", "residual", "schedule", "exponential"]


def make_mode_case(seed):
    """A dict: mode, net, x0, options, firings, trajectory, plus what the mode needs.  Relative
    quantities (fractions of the run's duration) are resolved by the test once it knows that
    duration; nothing here depends on the method."""
    r = np.random.default_rng(7919 * seed + 3)
    mode = MODES[int(r.integers(0, len(MODES)))]
    c = dict(mode=mode, seed=seed)
    if mode == "ensemble":
        which = int(r.integers(0, 3))          # 0: <= 4 reactions (register kernel), 1: <= 64, 2: bundle kernel
        if which == 0:
            net, x0 = W.random_mass_action(int(r.integers(1, 5)), int(r.integers(1, 5)), seed=seed)
            x0 = r.integers(0, 300, size=len(x0)).astype(np.int64)
        elif which == 1:
            net, x0 = W.random_mass_action(int(r.integers(1, 33)), int(r.integers(1, 65)), seed=seed)
            if r.random() < 0.4:
                x0 = r.integers(0, 40, size=len(x0)).astype(np.int64)
        else:
            net, x0, _, _, _ = make_case(seed, max_reactions=20_000)
        opts = []
        if which == 1 and r.random() < 0.3:
            opts.append(("ensemble_path", 2))
        if which == 0 and r.random() < 0.3:
            opts.append(("tiny_kernel", 0))
        if which == 2:
            if r.random() < 0.5:
                opts.append(("pipeline", int(r.integers(0, 2))))
            if r.random() < 0.5:
                opts.append(("exchange", int(r.integers(0, 2))))
            if r.random() < 0.5:
                opts.append(("bundle_ctas", int(r.choice([0, 1, 2, 3, 7, 13, 16]))))
        c.update(net=dict(net), x0=np.ascontiguousarray(x0, dtype=np.int64), options=opts,
                 n_traj=int(r.choice([1, 2, 31, 33, 64, 200])) if which < 2 else int(r.integers(1, 24)),
                 firings=int(10 ** r.uniform(1.5, 3.0)), traj_first=int(r.integers(0, 5000)),
                 t_end_fraction=float(r.uniform(0.3, 1.2)) if r.random() < 0.4 else None,
                 drop_firing_limit=bool(r.random() < 0.5))
        return c
    net, x0, opts, firings, traj = make_case(seed, max_reactions=40_000)
    opts = [o for o in opts if o[0] != "refresh_mode"]
    c.update(net=net, x0=x0, options=opts, firings=min(firings, 1500), trajectory=traj)
    M = int(net["n_reactions"])
    if mode in ("resume", "residual"):
        c["split"] = float(r.uniform(0.1, 0.9))
    elif mode == "schedule":
        nb = int(r.integers(1, 8))
        c["break_fractions"] = np.sort(r.uniform(0.0, 1.1, size=nb))
        if r.random() < 0.2:
            c["break_fractions"][0] = 0.0
        c["factor"] = r.choice([0.0, 0.5, 1.0, 2.0, 3.7], size=nb)
        c["mask"] = None if r.random() < 0.5 else (r.random(M) < 0.5).astype(np.uint8)
    else:
        c["lambda_times_duration"] = r.choice([0.0, 1.0, -1.0, 0.3, -2.5], size=M)
    return c
