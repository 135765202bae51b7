"""Random time algorithm of PAPER.md Table 1 (:251-256): EVERY step draws M fresh uniforms r_k,
sets Delta T_k = ln(1/r_k) (Eq.23, :156), solves Delta t_k = Delta T_k / a_k (Eq.24 with a_k
constant between firings, :160) and fires the channel with the smallest Delta t_k (Eq.25, :164).
No internal clock is carried over -- this is the memoryless variant the next-reaction form
(oracle/) must agree with in distribution (pin P10 of SURVEY.md 8(c)).  Vectorised over
independent trajectories with numpy; own generator, own propensity code; shares nothing with
oracle/ or the CUDA path."""
import numpy as np


def _h(X, species, sigma):
    out = np.ones(X.shape[0], dtype=np.float64)
    for j, s in zip(species, sigma):
        x = X[:, j].astype(np.float64)
        term = x
        for i in range(1, s):
            term = term * (x - i) / (i + 1)
        out = out * np.maximum(term, 0.0)
    return out


def rta_table1(net, x0, n_traj, t_end, seed, max_steps=10_000_000):
    """X(t_end) for n_traj independent Table-1 trajectories, [n_traj, N] int64 (a step that would
    pass t_end is not applied: reading G8)."""
    rng = np.random.default_rng(seed)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    rp, rs, rg = net["react_ptr"], net["react_species"], net["react_sigma"]
    sp, ss, sv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    V = np.zeros((M, N), dtype=np.int64)
    for k in range(M):
        for e in range(sp[k], sp[k + 1]):
            V[k, ss[e]] = sv[e]
    X = np.tile(np.asarray(x0, dtype=np.int64), (n_traj, 1))
    t = np.zeros(n_traj)
    alive = np.ones(n_traj, dtype=bool)
    for _ in range(max_steps):
        idx = np.flatnonzero(alive)
        if idx.size == 0:
            break
        Xa = X[idx]
        a = np.stack([net["rate"][k] * _h(Xa, rs[rp[k]:rp[k + 1]], rg[rp[k]:rp[k + 1]])
                      for k in range(M)], axis=1)
        r = 1.0 - rng.random((idx.size, M))                  # in (0, 1]
        dT = np.log(1.0 / r)
        with np.errstate(divide="ignore", invalid="ignore"):
            dt = np.where(a > 0, dT / a, np.inf)
        mu = dt.argmin(axis=1)
        dmin = dt[np.arange(idx.size), mu]
        tn = t[idx] + dmin
        stop = ~np.isfinite(dmin) | (tn > t_end)
        go = ~stop
        gi = idx[go]
        X[gi] += V[mu[go]]
        t[gi] = tn[go]
        alive[idx[stop]] = False
    else:
        raise RuntimeError("rta_table1: max_steps exhausted")
    return X
