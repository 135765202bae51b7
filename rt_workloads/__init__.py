"""Seeded synthetic workloads (BASELINE.json configs 1-5) as plain numpy CSR arrays.

This module holds NONE of the method's arithmetic (no propensity, no waiting time, no RNG
draw of the simulation): it only builds networks and initial counts.  It is the one module
both the CUDA path's callers (tests, bench.py) and the oracle's callers use, so that both
sides see byte-identical inputs.  It imports neither side.

A network is a dict:
    n_species N, n_reactions M,
    react_ptr  int64[M+1], react_species int32[nnz_r], react_sigma int32[nnz_r]   (sigma_jk >= 1)
    stoich_ptr int64[M+1], stoich_species int32[nnz_v], stoich_v int32[nnz_v]     (v_jk != 0)
    rate float64[M]                                                                 (c_k)
Rows are sorted by species index; no species appears twice in a row.

The paper's only workload is the Lotka file of Table 4 = config 2; the
other networks follow BASELINE.json `configs` and SURVEY.md 8(d); recipes restated in DESIGN.md.
"""
import numpy as np

__all__ = ["birth_death", "lotka_volterra", "random_mass_action", "protein_interaction",
           "from_reactions", "CONFIGS", "make_config"]


def from_reactions(n_species, reactions):
    """Build a network dict from a python list of (reactants {j: sigma}, products {j: coef}, c)."""
    rp, rs, rg = [0], [], []
    sp, ss, sv = [0], [], []
    rate = []
    for reactants, products, c in reactions:
        for j in sorted(reactants):
            rs.append(j)
            rg.append(reactants[j])
        rp.append(len(rs))
        net = {}
        for j, s in reactants.items():
            net[j] = net.get(j, 0) - s
        for j, s in products.items():
            net[j] = net.get(j, 0) + s
        for j in sorted(net):
            if net[j] != 0:
                ss.append(j)
                sv.append(net[j])
        sp.append(len(ss))
        rate.append(c)
    return dict(n_species=int(n_species), n_reactions=len(reactions),
                react_ptr=np.asarray(rp, dtype=np.int64),
                react_species=np.asarray(rs, dtype=np.int32),
                react_sigma=np.asarray(rg, dtype=np.int32),
                stoich_ptr=np.asarray(sp, dtype=np.int64),
                stoich_species=np.asarray(ss, dtype=np.int32),
                stoich_v=np.asarray(sv, dtype=np.int32),
                rate=np.asarray(rate, dtype=np.float64))


def birth_death(c1=10.0, c2=0.1):
    """Config 1: 0 -> X (c1), X -> 0 (c2); X0 = 0."""
    net = from_reactions(1, [({}, {0: 1}, c1), ({0: 1}, {}, c2)])
    return net, np.zeros(1, dtype=np.int64)


def lotka_volterra(c1=10.0, c2=0.01, c3=10.0, y1=1000, y2=1000):
    """Config 2 (= PAPER.md:277-287, Table 4): Y1->2Y1, Y1+Y2->2Y2, Y2->0; X0=(1000,1000)."""
    net = from_reactions(2, [({0: 1}, {0: 2}, c1),
                             ({0: 1, 1: 1}, {1: 2}, c2),
                             ({1: 1}, {}, c3)])
    return net, np.asarray([y1, y2], dtype=np.int64)


def _csr_from_coo(M, row, col, val, drop_zero):
    """Sum duplicate (row, col) entries, optionally drop zeros, return CSR sorted by (row, col)."""
    key = row.astype(np.int64) * np.int64(1 << 32) + col.astype(np.int64)
    order = np.argsort(key, kind="stable")
    key, val = key[order], val[order]
    if key.size:
        first = np.empty(key.size, dtype=bool)
        first[0] = True
        np.not_equal(key[1:], key[:-1], out=first[1:])
        starts = np.flatnonzero(first)
        val = np.add.reduceat(val.astype(np.int64), starts)
        key = key[starts]
    if drop_zero:
        keep = val != 0
        key, val = key[keep], val[keep]
    r = (key >> 32).astype(np.int64)
    c = (key & np.int64(0xFFFFFFFF)).astype(np.int32)
    ptr = np.zeros(M + 1, dtype=np.int64)
    np.add.at(ptr, r + 1, 1)
    np.cumsum(ptr, out=ptr)
    return ptr, c, val.astype(np.int32)


def random_mass_action(n_species, n_reactions, seed=7):
    """Configs 3 / 5a: each reaction has 0-2 distinct uniform reactant species with sigma in
    {1,2}, and 1-2 uniform product species (coefficient 1 each); v = products - reactants with
    zero entries dropped; c_k = 10^U(-3,0); x0 uniform integers in [100, 1000]."""
    rng = np.random.default_rng(seed)
    N, M = int(n_species), int(n_reactions)
    n_react = rng.integers(0, 3, size=M)
    r1 = rng.integers(0, N, size=M)
    r2 = rng.integers(0, N - 1, size=M) if N > 1 else np.zeros(M, dtype=np.int64)
    r2 = r2 + (r2 >= r1)                     # distinct from r1
    if N == 1:
        n_react = np.minimum(n_react, 1)
    s1 = rng.integers(1, 3, size=M)
    s2 = rng.integers(1, 3, size=M)
    n_prod = rng.integers(1, 3, size=M)
    p1 = rng.integers(0, N, size=M)
    p2 = rng.integers(0, N, size=M)
    rate = 10.0 ** rng.uniform(-3.0, 0.0, size=M)
    x0 = rng.integers(100, 1001, size=N).astype(np.int64)

    k = np.arange(M, dtype=np.int64)
    m1, m2 = n_react >= 1, n_react >= 2
    rrow = np.concatenate([k[m1], k[m2]])
    rcol = np.concatenate([r1[m1], r2[m2]])
    rsig = np.concatenate([s1[m1], s2[m2]])
    react_ptr, react_species, react_sigma = _csr_from_coo(M, rrow, rcol, rsig, drop_zero=False)

    q2 = n_prod >= 2
    srow = np.concatenate([rrow, k, k[q2]])
    scol = np.concatenate([rcol, p1, p2[q2]])
    sval = np.concatenate([-rsig, np.ones(M, dtype=np.int64), np.ones(int(q2.sum()), dtype=np.int64)])
    stoich_ptr, stoich_species, stoich_v = _csr_from_coo(M, srow, scol, sval, drop_zero=True)

    net = dict(n_species=N, n_reactions=M, react_ptr=react_ptr, react_species=react_species,
               react_sigma=react_sigma, stoich_ptr=stoich_ptr, stoich_species=stoich_species,
               stoich_v=stoich_v, rate=rate)
    return net, x0


def protein_interaction(n_species=100_000, n_pairs=500_000, seed=4, gamma=2.5):
    """Config 4: n_pairs binding/unbinding pairs.  Species A_i, B_i, C_i drawn with weight
    proportional to rank^(-1/(gamma-1)) (power-law degree, exponent gamma), redrawn until
    distinct.  Reaction 2i: A+B -> C, c = 10^U(-4,-2); reaction 2i+1: C -> A+B, c = 10^U(-2,0).
    x0 uniform integers in [50, 500]."""
    rng = np.random.default_rng(seed)
    N, Q = int(n_species), int(n_pairs)
    w = np.arange(1, N + 1, dtype=np.float64) ** (-1.0 / (gamma - 1.0))
    cdf = np.cumsum(w)
    cdf /= cdf[-1]

    def draw(n):
        return np.minimum(np.searchsorted(cdf, rng.random(n), side="right"), N - 1)

    abc = np.stack([draw(Q), draw(Q), draw(Q)], axis=1)
    while True:
        bad = (abc[:, 0] == abc[:, 1]) | (abc[:, 0] == abc[:, 2]) | (abc[:, 1] == abc[:, 2])
        nb = int(bad.sum())
        if nb == 0:
            break
        abc[bad] = np.stack([draw(nb), draw(nb), draw(nb)], axis=1)
    c_bind = 10.0 ** rng.uniform(-4.0, -2.0, size=Q)
    c_unbind = 10.0 ** rng.uniform(-2.0, 0.0, size=Q)
    x0 = rng.integers(50, 501, size=N).astype(np.int64)

    M = 2 * Q
    i = np.arange(Q, dtype=np.int64)
    A, B, Cc = abc[:, 0], abc[:, 1], abc[:, 2]
    one = np.ones(Q, dtype=np.int64)
    rrow = np.concatenate([2 * i, 2 * i, 2 * i + 1])
    rcol = np.concatenate([A, B, Cc])
    rsig = np.concatenate([one, one, one])
    react_ptr, react_species, react_sigma = _csr_from_coo(M, rrow, rcol, rsig, drop_zero=False)
    srow = np.concatenate([2 * i, 2 * i, 2 * i, 2 * i + 1, 2 * i + 1, 2 * i + 1])
    scol = np.concatenate([A, B, Cc, A, B, Cc])
    sval = np.concatenate([-one, -one, one, one, one, -one])
    stoich_ptr, stoich_species, stoich_v = _csr_from_coo(M, srow, scol, sval, drop_zero=True)
    rate = np.empty(M, dtype=np.float64)
    rate[0::2] = c_bind
    rate[1::2] = c_unbind
    net = dict(n_species=N, n_reactions=M, react_ptr=react_ptr, react_species=react_species,
               react_sigma=react_sigma, stoich_ptr=stoich_ptr, stoich_species=stoich_species,
               stoich_v=stoich_v, rate=rate)
    return net, x0


# name -> (builder, run parameters).  Philox seeds: 1 and 7 are BASELINE.json's; 2, 4, 5 are
# SURVEY.md 8(d) proposals where BASELINE.json is silent.
CONFIGS = {
    "cfg1": dict(seed=1, n_traj=1000, t_end=1000.0, max_firings=1_000_000),
    "cfg2": dict(seed=2, n_traj=100_000, t_end=10.0, max_firings=5_000_000),
    "cfg3": dict(seed=7, n_traj=1, t_end=float("inf"), max_firings=100_000, trace=10_000),
    "cfg4": dict(seed=4, n_traj=1, t_end=float("inf"), max_firings=10_000, trace=10_000),
    "cfg5a": dict(seed=5, n_traj=1, t_end=float("inf"), max_firings=2_000, trace=2_000),
    "cfg5b": dict(seed=5, n_traj=64, t_end=float("inf"), max_firings=10_000),
}


def make_config(name, scale=1.0):
    """Network + x0 + run parameters of a BASELINE.json config.  `scale` < 1 shrinks N and M of
    the generated networks (cfg3/4/5a) by that factor for quick tests; the recipe is unchanged."""
    if name == "cfg1":
        net, x0 = birth_death()
    elif name == "cfg2":
        net, x0 = lotka_volterra()
    elif name in ("cfg3", "cfg5b"):
        net, x0 = random_mass_action(max(2, int(10_000 * scale)), max(2, int(100_000 * scale)), seed=7)
    elif name == "cfg4":
        net, x0 = protein_interaction(max(8, int(100_000 * scale)), max(4, int(500_000 * scale)), seed=4)
    elif name == "cfg5a":
        net, x0 = random_mass_action(max(2, int(1_000_000 * scale)), max(2, int(10_000_000 * scale)), seed=7)
    else:
        raise KeyError(name)
    return net, x0, dict(CONFIGS[name])
