"""Pins of the oracle's smooth time-dependent-rate run (section 6, Eq.28, :224-231) with
c_k(t) = c_k exp(lambda_k t): closed forms, an exact law, limits that reduce to already-pinned
routines, and convergence of the piecewise-constant run towards it.  No GPU, no CUDA path."""
import math

import numpy as np
import pytest
from scipy import stats

import oracle
import rt_workloads as W

INF = math.inf


def _draws(seed, traj, k, n):
    return np.array([oracle.exp_draw(seed, traj, k, i) for i in range(n)])


@pytest.mark.parametrize("c,lam", [(3.0, 0.7), (40.0, -0.05), (0.2, 2.5)])
def test_single_channel_closed_form(c, lam):
    """One source channel 0 -> X with rate c exp(lam t): Eq.28 gives sum_{i<n} E_i =
    c (exp(lam t_n) - 1) / lam, i.e. t_n = log1p(lam sum E / c) / lam, and T(t_n) = sum E."""
    n, seed, traj = 60, 5, 2
    net = W.from_reactions(1, [({}, {0: 1}, c)])
    e = np.cumsum(_draws(seed, traj, 0, n + 1))
    if lam < 0:
        n = min(n, int(np.searchsorted(e, c / -lam)))     # total integral c/|lam| is finite
    r = oracle.run_rate_exp(net, [0], [lam], seed, traj, n, INF, n)
    assert r["firings"] == n
    np.testing.assert_allclose(r["trace_t"], np.log1p(lam * e[:n] / c) / lam, rtol=1e-12)
    assert r["T"][0] == pytest.approx(e[n - 1], rel=1e-12)
    assert r["P"][0] == pytest.approx(e[n], rel=1e-13)


def test_decaying_channel_goes_silent():
    """lam < 0: the whole future integral of the rate is c/|lam|.  The channel fires while its
    next internal firing time is below that and never again afterwards (dt = +inf -> ABSORBED)."""
    c, lam, seed, traj = 5.0, -1.0, 1, 0
    net = W.from_reactions(1, [({}, {0: 1}, c)])
    e = np.cumsum(_draws(seed, traj, 0, 200))
    n_expected = int(np.searchsorted(e, c / -lam))
    r = oracle.run_rate_exp(net, [0], [lam], seed, traj, 1000, INF, 1000)
    assert r["stop"] == oracle.STOP_ABSORBED and r["firings"] == n_expected
    assert r["t"] == r["trace_t"][-1]                    # absorbed: t stays at the last firing
    # a time limit before the channel goes silent: T(t_end) = c (1 - exp(-t_end)) (Eq.15 with
    # Eq.28's integrand), and the firings so far are those with sum E below it
    t_end = 0.5
    r = oracle.run_rate_exp(net, [0], [lam], seed, traj, 0, t_end)
    T_end = c * -math.expm1(lam * t_end)
    assert e[int(np.searchsorted(e, T_end))] < c / -lam   # (a firing is still pending at t_end)
    assert r["stop"] == oracle.STOP_T_END and r["T"][0] == pytest.approx(T_end, rel=1e-12)
    assert r["firings"] == int(np.searchsorted(e, T_end))


def test_independent_sources_merge_their_closed_forms():
    """M source channels with different lambda_k (growth, decay, zero) do not interact, so the trace
    is the sorted merge of M closed-form sequences.  Every channel's clock T_k is advanced in many
    partial intervals (one per firing of ANY channel): a wrong propensity, interval start or
    increment formula in the advance step shifts every later event of that channel."""
    seed, traj, n = 11, 3, 400
    c = [2.0, 9.0, 0.5, 4.0, 1.0]
    lam = [0.0, -0.02, 0.9, 0.3, -0.4]
    M = len(c)
    net = W.from_reactions(M, [({}, {k: 1}, c[k]) for k in range(M)])
    r = oracle.run_rate_exp(net, [0] * M, lam, seed, traj, n, INF, n)
    events = []
    for k in range(M):
        e = np.cumsum(_draws(seed, traj, k, n))
        if lam[k] == 0.0:
            tk = e / c[k]
        else:
            x = lam[k] * e / c[k]
            tk = np.where(x > -1.0, np.log1p(np.maximum(x, -0.999999999)) / lam[k], INF)
        events += [(float(t), k) for t in tk if math.isfinite(t)]
    events.sort()
    assert [k for _, k in events[:n]] == list(r["trace_mu"])
    np.testing.assert_allclose(r["trace_t"], [t for t, _ in events[:n]], rtol=1e-11)


def test_zero_lambda_is_the_constant_rate_run_bit_for_bit():
    net, x0, par = W.make_config("cfg3", scale=0.01)
    a = oracle.run(net, x0, 7, 0, 800, INF, 800)
    b = oracle.run_rate_exp(net, x0, np.zeros(net["n_reactions"]), 7, 0, 800, INF, 800)
    for key in ("trace_mu", "trace_t", "x", "T", "P", "fire_count"):
        assert np.array_equal(a[key], b[key]), key
    a = oracle.run(net, x0, 7, 0, 0, 0.004)
    b = oracle.run_rate_exp(net, x0, np.zeros(net["n_reactions"]), 7, 0, 0, 0.004)
    assert a["t"] == b["t"] == 0.004 and np.array_equal(a["T"], b["T"]) and np.array_equal(a["x"], b["x"])


def test_birth_death_with_decaying_birth_rate_is_poisson():
    """0 -> X at c1 exp(lam t), X -> 0 at c2 per molecule, X(0) = 0: a linear network stays Poisson
    with mean m(t) solving m' = c1 exp(lam t) - c2 m, i.e. m(t) = c1 (exp(lam t) - exp(-c2 t)) /
    (lam + c2); the birth count is Poisson(c1 (exp(lam t) - 1) / lam)."""
    c1, c2, lam, t_end, n_traj = 40.0, 0.5, -0.3, 4.0, 3000
    net = W.from_reactions(1, [({}, {0: 1}, c1), ({0: 1}, {}, c2)])
    xs, births = [], []
    for i in range(n_traj):
        r = oracle.run_rate_exp(net, [0], [lam, 0.0], 21, i, 0, t_end)
        assert r["stop"] == oracle.STOP_T_END and r["t"] == t_end
        xs.append(r["x"][0])
        births.append(r["fire_count"][0])
    x, b = np.array(xs, dtype=float), np.array(births, dtype=float)
    m = c1 * (math.exp(lam * t_end) - math.exp(-c2 * t_end)) / (lam + c2)
    nb = c1 * math.expm1(lam * t_end) / lam
    assert abs(x.mean() - m) < 3 * math.sqrt(m / n_traj)
    assert abs(x.var(ddof=1) - m) < 3 * m * math.sqrt(2.0 / (n_traj - 1)) + 3 * math.sqrt(m / n_traj)
    assert abs(b.mean() - nb) < 3 * math.sqrt(nb / n_traj)
    assert abs(b.var(ddof=1) - nb) < 3 * nb * math.sqrt(2.0 / (n_traj - 1)) + 3 * math.sqrt(nb / n_traj)
    # discrete law: empirical CDF against the Poisson CDF at the integers (Kolmogorov 1% point)
    grid = np.arange(0, 120)
    d = np.abs(np.searchsorted(np.sort(x), grid, side="right") / n_traj - stats.poisson.cdf(grid, m)).max()
    assert d < 1.63 / math.sqrt(n_traj)


def test_piecewise_constant_schedule_converges_to_it():
    """The piecewise-constant run (nrrta_run_sched, separately pinned) with a fine staircase
    f_i = exp(lam (b_i + b_{i+1}) / 2) approximates the smooth family: on a nonlinear network
    (Lotka-Volterra with every rate growing) the two agree in distribution at t_end."""
    net, x0 = W.lotka_volterra(y1=60, y2=40, c1=2.0, c2=0.02, c3=1.5)
    lam, t_end, n_traj, steps = 0.4, 2.0, 500, 400
    edges = np.linspace(0.0, t_end, steps + 1)
    tb = edges[:-1].copy()
    fa = np.exp(lam * 0.5 * (edges[:-1] + edges[1:]))
    xa, xb = [], []
    for i in range(n_traj):
        xa.append(oracle.run_rate_exp(net, x0, [lam] * 3, 31, i, 0, t_end)["x"])
        xb.append(oracle.run_sched(net, x0, 32, i, 0, t_end, t_break=tb, factor=fa)["x"])
    xa, xb = np.array(xa, dtype=float), np.array(xb, dtype=float)
    ps = sorted(stats.ks_2samp(xa[:, j], xb[:, j]).pvalue for j in range(2))
    assert ps[0] > 0.01 / 2 and ps[1] > 0.01
    for j in range(2):
        se = math.sqrt(xa[:, j].var(ddof=1) / n_traj + xb[:, j].var(ddof=1) / n_traj)
        assert abs(xa[:, j].mean() - xb[:, j].mean()) < 3 * se


def test_kurtz_identity_and_clock_invariants():
    net, x0, par = W.make_config("cfg3", scale=0.01)
    M = int(net["n_reactions"])
    rng = np.random.default_rng(5)
    lam = rng.choice([0.0, -30.0, 50.0, 8.0], size=M)
    r = oracle.run_rate_exp(net, x0, lam, 7, 1, 1500, INF, 1500)
    # Eq.5: X = X0 + sum_k R_k v_k
    x = np.array(x0, dtype=np.int64)
    sp, ss, sv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    for k in np.flatnonzero(r["fire_count"]):
        for e in range(sp[k], sp[k + 1]):
            x[ss[e]] += int(r["fire_count"][k]) * int(sv[e])
    assert np.array_equal(x, r["x"]) and (r["x"] >= 0).all()
    assert r["fire_count"].sum() == 1500 and (np.diff(r["trace_t"]) >= 0).all()
    assert (r["T"] <= r["P"] * (1 + 1e-12)).all()


def test_common_lambda_is_a_time_change_of_the_constant_rate_run():
    """Eq.28 with ONE lambda for every channel: int_0^t a_k(s) ds = a_k(X) * s(t) with the same
    s(t) = (exp(lambda t) - 1) / lambda for all k, so the run is the constant-rate run (same seed,
    hence same internal firing times P_k) under the time change s -> t(s) = log1p(lambda s) / lambda:
    same fired sequence, event times t(s_i).  With lambda < 0 internal time saturates at
    1 / |lambda|: the run fires exactly the constant-rate firings with s_i < 1 / |lambda|, then is
    ABSORBED.  (lambda is put BETWEEN two firing times: on one, the last argument is -1 +- rounding.)"""
    net, x0 = W.lotka_volterra(y1=80, y2=60, c1=1.5, c2=0.01, c3=1.0)
    M = int(net["n_reactions"])
    base = oracle.run(net, x0, 17, 3, 400, math.inf, 400)
    s = base["trace_t"]
    for n_keep, sign in ((150, -1.0), (300, -1.0), (400, +1.0)):
        if sign < 0:
            lam = -2.0 / float(s[n_keep - 1] + s[n_keep])           # 1/|lam| between firing n_keep-1 and n_keep
            o = oracle.run_rate_exp(net, x0, np.full(M, lam), 17, 3, 100000, math.inf, 400)
            assert o["stop"] == 3 and o["firings"] == n_keep         # ABSORBED
        else:
            lam = 0.5 / float(s[-1])
            o = oracle.run_rate_exp(net, x0, np.full(M, lam), 17, 3, n_keep, math.inf, 400)
            assert o["firings"] == n_keep
        np.testing.assert_array_equal(o["trace_mu"][:n_keep], base["trace_mu"][:n_keep])
        np.testing.assert_allclose(o["trace_t"][:n_keep], np.log1p(lam * s[:n_keep]) / lam, rtol=1e-9)
