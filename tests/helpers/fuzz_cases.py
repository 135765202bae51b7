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
