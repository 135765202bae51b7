"""Brute-force Gillespie direct method (Gillespie 1977; Eq.21-22 with reading G10:
Delta t = ln(1/r) / sum_k a_k), vectorised over independent trajectories with numpy.

Used only to pin the oracle in distribution (the paper's claim that the random-time algorithm
is an exact SSA).  It shares no code with oracle/ or the CUDA path, uses numpy's
own generator, and evaluates propensities with math.comb-style integer arithmetic.
"""
import numpy as np


def _h(X, species, sigma):
    """prod_j C(X_j, sigma_j) for every trajectory; X is [n_traj, N] int64."""
    out = np.ones(X.shape[0], dtype=np.float64)
    for j, s in zip(species, sigma):
        x = X[:, j]
        if s == 1:
            b = x
        elif s == 2:
            b = x * (x - 1) // 2
        elif s == 3:
            b = x * (x - 1) * (x - 2) // 6
        else:
            raise ValueError(s)
        out = out * np.maximum(b, 0)
    return out


def direct_method(net, x0, n_traj, t_end, seed, max_steps=10_000_000):
    """Return X(t_end) for n_traj independent direct-method trajectories, [n_traj, N] int64,
    and the number of firings of every reaction, [n_traj, M]."""
    rng = np.random.default_rng(seed)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    rp, rs, rg = net["react_ptr"], net["react_species"], net["react_sigma"]
    sp, ss, sv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    V = np.zeros((M, N), dtype=np.int64)
    for k in range(M):
        for e in range(sp[k], sp[k + 1]):
            V[k, ss[e]] = sv[e]
    X = np.tile(np.asarray(x0, dtype=np.int64), (n_traj, 1))
    R = np.zeros((n_traj, M), dtype=np.int64)
    t = np.zeros(n_traj)
    alive = np.ones(n_traj, dtype=bool)
    for _ in range(max_steps):
        idx = np.flatnonzero(alive)
        if idx.size == 0:
            break
        Xa = X[idx]
        a = np.stack([net["rate"][k] * _h(Xa, rs[rp[k]:rp[k + 1]], rg[rp[k]:rp[k + 1]])
                      for k in range(M)], axis=1)
        a0 = a.sum(axis=1)
        dead = a0 <= 0
        with np.errstate(divide="ignore", invalid="ignore"):
            dt = -np.log(1.0 - rng.random(idx.size)) / a0
        tn = t[idx] + dt
        stop = dead | (tn > t_end)
        u = rng.random(idx.size) * a0
        mu = (np.cumsum(a, axis=1) <= u[:, None]).sum(axis=1)
        mu = np.minimum(mu, M - 1)
        go = ~stop
        gi = idx[go]
        X[gi] += V[mu[go]]
        R[gi, mu[go]] += 1
        t[gi] = tn[go]
        alive[idx[stop]] = False
    else:
        raise RuntimeError("direct_method: max_steps exhausted")
    return X, R
