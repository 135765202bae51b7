"""The parallel next-reaction random time algorithm of PAPER.md Table 3 (:262-272) in its LITERAL
(Delta t_k, p_k) form, as a test-side cross-check of the oracle's residual reading (G4):

    Initialize.  Compute a_k, set Delta t_k = ln(1/r_k)/a_k, set p_k = a_k
    while t < t_max:
        scan for Delta t_mu = min_k Delta t_k
        update species for reaction mu, set t = t + Delta t_mu
        recalculate a_k for every reaction,
        set Delta t_mu = ln(1/r)/a_mu, set Delta t_k = (p_k/a_k)(Delta t_k - Delta t_mu)   [k != mu]
        (p_k = a_k for the next step)

The rescale divides by the NEW a_k, so the form is only defined while every a_k stays > 0 (reading
G4: with a_k = 0 the remaining internal time is lost) -- the helper asserts that.  Vectorised over
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


def table3_literal(net, x0, n_traj, t_end, seed, max_steps=10_000_000):
    """X(t_end) for n_traj independent trajectories, [n_traj, N] int64 (a step that would pass t_end
    is not applied: reading G8)."""
    rng = np.random.default_rng(seed)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    rp, rs, rg = net["react_ptr"], net["react_species"], net["react_sigma"]
    sp, ss, sv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    rate = np.asarray(net["rate"], dtype=np.float64)
    V = np.zeros((M, N), dtype=np.int64)
    for k in range(M):
        for e in range(sp[k], sp[k + 1]):
            V[k, ss[e]] = sv[e]

    def propensities(X):
        return np.stack([rate[k] * _h(X, rs[rp[k]:rp[k + 1]], rg[rp[k]:rp[k + 1]]) for k in range(M)], axis=1)

    X = np.tile(np.asarray(x0, dtype=np.int64), (n_traj, 1))
    t = np.zeros(n_traj)
    a = propensities(X)
    assert (a > 0).all(), "Table 3's rescale form needs every a_k > 0"
    dt = -np.log(1.0 - rng.random((n_traj, M))) / a          # ln(1/r), r in (0, 1]
    p = a.copy()
    alive = np.ones(n_traj, dtype=bool)
    rows = np.arange(n_traj)
    for _ in range(max_steps):
        if not alive.any():
            break
        mu = np.argmin(dt, axis=1)
        dmin = dt[rows, mu]
        stop = alive & (t + dmin > t_end)
        alive &= ~stop
        go = np.flatnonzero(alive)
        if go.size == 0:
            break
        X[go] += V[mu[go]]
        t[go] += dmin[go]
        a_new = propensities(X[go])
        assert (a_new > 0).all(), "Table 3's rescale form needs every a_k > 0"
        d_go = (p[go] / a_new) * (dt[go] - dmin[go][:, None])
        d_go[np.arange(go.size), mu[go]] = -np.log(1.0 - rng.random(go.size)) / a_new[np.arange(go.size), mu[go]]
        dt[go] = d_go
        p[go] = a_new
    return X
