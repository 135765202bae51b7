"""GPU parity: the CUDA path (through the C ABI of include/rt.h) against the CPU oracle on the
same seeded inputs.  Bar (BASELINE.json north_star): fired-reaction sequence and species counts
bit-exact for the first 1e4 firings, event times within 1e-12 relative."""
import math
import os

import numpy as np
import pytest

import rt_workloads as W
from helpers.tie_cases import tie_network, expected_trace

pytestmark = pytest.mark.gpu

RTOL_T = 1e-12


@pytest.fixture(scope="module")
def rt():
    import paper_2103_00405_b200 as rt
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    rt.lib()   # fails loudly if librt_b200.so is missing
    return rt


def _oracle():
    import oracle
    return oracle


def _check_run(rt, net, x0, seed, traj, max_firings, t_end, trace_cap, options=()):
    o = _oracle().run(net, x0, seed, traj, max_firings, t_end, trace_cap)
    with rt.Model(net) as m:
        for name, val in options:
            m.set_option(name, val)
        g = m.run(x0, seed, traj, max_firings, t_end, trace_cap, want_state=True)
        assert m.info("kernel_launches") >= 1
    assert g["firings"] == o["firings"]
    assert g["stop"] == o["stop"]
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)
    assert math.isclose(g["t"], o["t"], rel_tol=RTOL_T, abs_tol=0)
    # internal clocks: sums of a_k*dt, same order on both sides -> agree to ~firings ulp
    np.testing.assert_allclose(g["T"], o["T"], rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(g["P"], o["P"], rtol=1e-12, atol=0)
    return g, o


@pytest.mark.parametrize("refresh_mode", [0, 1])
@pytest.mark.parametrize("scale,firings", [(0.01, 3000), (0.0517, 2000)])
def test_cfg3_scaled_trace(rt, scale, firings, refresh_mode):
    """Random mass-action network at reduced N, M (ragged: M odd / not a tile multiple)."""
    net, x0, par = W.make_config("cfg3", scale=scale)
    _check_run(rt, net, x0, par["seed"], 0, firings, math.inf, firings,
               options=[("refresh_mode", refresh_mode)])


@pytest.mark.parametrize("pipeline", [1, 0])
@pytest.mark.parametrize("exchange", [0, 1])
@pytest.mark.parametrize("ctas", [1, 2, 7, 12, 16, 0])
def test_cfg3_bundle_shape_invariance(rt, ctas, exchange, pipeline):
    """Result must not depend on how many CTAs share the trajectory (determinism contract), nor on
    how they exchange their partial argmins -- as one thread-block cluster through distributed
    shared memory (exchange 0, bundles of 2..16 CTAs) or through slots in L2 (exchange 1) -- nor on
    the kernel: candidate-first (pipeline 1, rt_fast.cuh) or pass-then-reduce (0, rt_bundle.cuh)."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    _check_run(rt, net, x0, par["seed"], 3, 1500, math.inf, 1500,
               options=[("bundle_ctas", ctas), ("exchange", exchange), ("pipeline", pipeline)])
    with rt.Model(net) as m:
        m.set_option("bundle_ctas", ctas)
        m.set_option("exchange", exchange)
        m.set_option("pipeline", pipeline)
        m.run(x0, par["seed"], 3, 10)
        S = m.info("bundle_ctas")
        assert m.info("pipeline") == pipeline
        assert m.info("cluster_exchange") == (1 if exchange == 0 and 2 <= S <= 16 else 0)
        if ctas:
            assert S == ctas


@pytest.mark.parametrize("state_mode", [0, 1])
@pytest.mark.parametrize("ctas", [1, 3, 0])
def test_state_in_shared_vs_global_memory(rt, state_mode, ctas):
    """The (T,P,a) store lives in shared memory when a CTA's share fits, else in global memory
    (the HBM-streaming regime of cfg5a); both must give the oracle's path."""
    net, x0, par = W.make_config("cfg3", scale=0.03)
    _check_run(rt, net, x0, par["seed"], 1, 1200, math.inf, 1200,
               options=[("state_mode", state_mode), ("bundle_ctas", ctas)])


def _hub_network(n_species=40, n_reactions=5000, seed=3):
    """Every reaction reads hub species 0 (degree 5000 >> the hub threshold and, on one CTA,
    more refreshes per firing than one staging round holds); some rows have 3 reactants
    (general propensity path) and some change 6 species (CSR stoich path)."""
    rng = np.random.default_rng(seed)
    reactions = []
    for k in range(n_reactions):
        others = rng.choice(np.arange(1, n_species), size=6, replace=False)
        reactants = {0: 1}
        kind = k % 5
        if kind >= 1:
            reactants[int(others[0])] = 1 + (k % 2)
        if kind == 4:
            reactants[int(others[1])] = 1
        products = {0: 1, int(others[2]): 1}
        if kind == 3:
            products.update({int(others[3]): 1, int(others[4]): 2, int(others[5]): 1})
        reactions.append((reactants, products, float(10.0 ** rng.uniform(-4, -2))))
    return W.from_reactions(n_species, reactions), rng.integers(20, 60, size=n_species).astype(np.int64)


@pytest.mark.parametrize("ctas,state_mode,exchange", [(1, 0, 0), (1, 1, 0), (5, 0, 0), (5, 0, 1), (0, 0, 0), (0, 0, 1)])
def test_hub_species_general_rows_and_staging_overflow(rt, ctas, state_mode, exchange):
    net, x0 = _hub_network()
    for refresh_mode, pipeline in ((0, 1), (0, 0), (1, 1)):
        _check_run(rt, net, x0, 21, 0, 600, math.inf, 600,
                   options=[("bundle_ctas", ctas), ("state_mode", state_mode), ("pipeline", pipeline),
                            ("refresh_mode", refresh_mode), ("exchange", exchange)])


@pytest.mark.parametrize("ctas", [1, 0])
def test_extreme_rates_and_cubic_reactions(rt, ctas):
    """Rates from 1e-300 to 1e300 (outside the range where the approximate-quotient filter of the
    scan is proven, so the exact path must take over), zero and negative-zero rates, and
    trimolecular 3A -> B reactions (sigma = 3, count bound 2^21 - 1)."""
    rng = np.random.default_rng(11)
    n_species, reactions = 30, []
    for k in range(1500):
        j = [int(v) for v in rng.choice(n_species, size=3, replace=False)]
        kind = k % 6
        if kind == 0:
            reactions.append(({j[0]: 3}, {j[1]: 1}, float(10.0 ** rng.uniform(-6, -3))))
        elif kind == 1:
            reactions.append(({j[0]: 1, j[1]: 2}, {j[2]: 1}, float(10.0 ** rng.uniform(-300, -250))))
        elif kind == 2:
            reactions.append(({j[0]: 1}, {j[1]: 1}, float(10.0 ** rng.uniform(250, 300))))
        elif kind == 3:
            reactions.append(({j[0]: 1}, {j[1]: 2}, 0.0 if k % 12 == 3 else -0.0))
        else:
            reactions.append(({j[0]: 1, j[1]: 1}, {j[2]: 1, j[0]: 1}, float(10.0 ** rng.uniform(-2, 1))))
    net = W.from_reactions(n_species, reactions)
    x0 = rng.integers(5, 40, size=n_species).astype(np.int64)
    for state_mode in (0, 1):
        _check_run(rt, net, x0, 31, 2, 800, math.inf, 800,
                   options=[("bundle_ctas", ctas), ("state_mode", state_mode)])


def test_count_overflow_is_reported(rt):
    """0 -> X from the count bound: after the three deaths of the other species the first birth
    leaves [0, 2^31-1] -> RT_ERR_OVERFLOW at firing 4.  DESIGN.md 2 "Overflow": the offending
    firing is counted and traced, its X change is not applied -- on the bundle kernel, on the
    one-thread-per-trajectory kernel and in the oracle alike."""
    net = W.from_reactions(2, [({}, {0: 1}, 1.0), ({1: 1}, {}, 1.0)])
    x0 = np.array([2**31 - 1, 3], dtype=np.int64)
    o = _oracle().run(net, x0, 5, 0, 100, math.inf, 100, check=False)
    with rt.Model(net) as m:
        g = m.run(x0, 5, 0, 100, math.inf, 100, want_state=True, check=False)
        ens = []
        for path in (1, 2):
            m.set_option("ensemble_path", path)
            ens.append(m.ensemble(x0, 5, 0, 3, 100, math.inf, check=False))
            assert m.info("ensemble_path") == path
    assert g["code"] == rt.RT_ERR_OVERFLOW and g["status"] == rt.RT_ERR_OVERFLOW
    assert o["code"] == -5 and g["firings"] == o["firings"] == 4
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["x"], [2**31 - 1, 0])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    for e in ens:                      # row i of an ensemble == rt_run(trajectory i), errors included
        assert e["code"] == rt.RT_ERR_OVERFLOW and (e["status"] == rt.RT_ERR_OVERFLOW).all()
        for i in range(3):
            oi = _oracle().run(net, x0, 5, i, 100, math.inf, 0, check=False)
            np.testing.assert_array_equal(e["x"][i], oi["x"])
            assert e["firings"][i] == oi["firings"]


def test_network_without_any_reactant(rt):
    """A validated network with NO reactant entries at all (pure sources: empty react_species /
    react_sigma arrays): the single-channel closed form t_n = sum_i E_i / c (Eq.23-24,
    PAPER.md:156-160) through the bundle kernel and through the thread kernel."""
    c, n = 2.5, 200
    net = W.from_reactions(1, [({}, {0: 1}, c)])
    assert net["react_species"].size == 0
    g, o = _check_run(rt, net, np.array([0]), 13, 6, n, math.inf, n)
    e = [_oracle().exp_draw(13, 6, 0, i) for i in range(n)]
    np.testing.assert_allclose(g["trace_t"], np.cumsum(e) / c, rtol=1e-12)
    net3 = W.from_reactions(3, [({}, {0: 1}, 1.0), ({}, {1: 1, 2: 1}, 0.3), ({}, {2: 2}, 2.0)])
    _check_run(rt, net3, np.zeros(3, dtype=np.int64), 2, 0, 500, math.inf, 500)
    o = _oracle().ensemble(net3, np.zeros(3, dtype=np.int64), 2, 0, 40, 300, math.inf)
    with rt.Model(net3) as m:
        e = m.ensemble(np.zeros(3, dtype=np.int64), 2, 0, 40, 300, math.inf)
        assert m.info("ensemble_path") == 1
    np.testing.assert_array_equal(e["x"], o["x"])
    np.testing.assert_allclose(e["t"], o["t"], rtol=RTOL_T)


# ------------------------------------------------------------------ exact ties (reading G6)
def _check_tie(rt, M, coupled, formulation, options, n_more=40):
    """Exact finite ties from a checkpointed state (tests/helpers/tie_cases.py): an M-way tie at
    dt = 8, then M-1 firings that tie at dt = 0.  The expected trace 0, 1, ..., M-1 at t = 8.0
    follows by hand; the oracle is compared as well, past the end of the tie."""
    net, x0, T0, P0, n0 = tie_network(M, coupled=coupled)
    n = M + n_more
    o = _oracle().run_from(net, x0, 0.0, T0, P0, n0, 9, 1, n, math.inf, n, residual=bool(formulation))
    with rt.Model(net) as m:
        m.set_option("formulation", formulation)
        for name, val in options:
            m.set_option(name, val)
        if formulation:
            g = m.run_resume(x0, 0.0, -P0, np.zeros(M), n0, 9, 1, n, math.inf, n, want_state=True)
        else:
            g = m.run_resume(x0, 0.0, T0, P0, n0, 9, 1, n, math.inf, n, want_state=True)
    mu, tt = expected_trace(M)
    np.testing.assert_array_equal(g["trace_mu"][:M], mu)
    np.testing.assert_array_equal(g["trace_t"][:M], tt)
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)


@pytest.mark.parametrize("formulation", [0, 1])
@pytest.mark.parametrize("state_mode", [0, 1, 2])
@pytest.mark.parametrize("ctas", [1, 3, 7, 16, 0])
def test_exact_ties_go_to_the_lowest_index(rt, ctas, state_mode, formulation):
    """north_star: "argmin reduction over k with ties broken by lowest index".  The ties straddle
    the reactions of one thread (filter fallback: every approximate quotient of a thread is equal),
    lanes, warps and CTAs (REDUX lexmin, exchange slots), and with `coupled` every firing refreshes
    every hub reader inside the tie (fresh-candidate merge, warp-shared / cooperative re-scan)."""
    # state_mode 2 here: state in shared memory with the exchange through L2 (0: cluster / DSMEM)
    opts = [("bundle_ctas", ctas), ("state_mode", state_mode & 1), ("exchange", 1 if state_mode == 2 else 0)]
    _check_tie(rt, 5003, False, formulation, opts)
    _check_tie(rt, 4999, True, formulation, opts)


@pytest.mark.parametrize("ctas,exchange", [(1, 0), (3, 0), (3, 1), (16, 0), (0, 1)])
def test_exact_ties_plain_bundle_kernel(rt, ctas, exchange):
    """The same tie networks through the pass-then-reduce kernel (pipeline 0) with on-chip state."""
    opts = [("bundle_ctas", ctas), ("exchange", exchange), ("pipeline", 0)]
    for formulation in (0, 1):
        _check_tie(rt, 5003, False, formulation, opts)
        _check_tie(rt, 4999, True, formulation, opts)


def _check_resume_state(rt, net, x0, T0, P0, n, options):
    M = len(T0)
    n0 = np.zeros(M, dtype=np.uint64)
    o = _oracle().run_from(net, x0, 0.0, T0, P0, n0, 9, 1, n, math.inf, n)
    with rt.Model(net) as m:
        for name, val in options:
            m.set_option(name, val)
        g = m.run_resume(x0, 0.0, T0, P0, n0, 9, 1, n, math.inf, n, want_state=True)
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)
    np.testing.assert_allclose(g["T"], o["T"], rtol=1e-10, atol=1e-12)
    return g, o


@pytest.mark.parametrize("pipeline", [1, 0])
@pytest.mark.parametrize("ctas,exchange", [(1, 0), (4, 0), (4, 1), (0, 0)])
def test_near_ties_and_cancellation_defeat_the_filters(rt, ctas, exchange, pipeline):
    """Adversarial states for the approximate-quotient filters and for the candidate-first kernel's
    lagged candidates (rt_fast.cuh header).  (a) near-ties: every waiting time within 1e-9 .. 1e-6
    relative of every other one -- far inside the key tolerance, never equal -- so that no thread
    can rule anything out and every firing goes through the exact paths.  (b) catastrophic
    cancellation: internal times ~2^40 with residuals of order 1 (P - T keeps 2^-40 of P: outside
    the cancellation guard), as after a very long run, mixed with ordinary channels; one rounding
    of T + a*dt then moves a waiting time by more than the filters' margin, so a candidate kept
    across a firing without the guard could lose the argmin.  Both against oracle.run_from."""
    rng = np.random.default_rng(5)
    M = 4801
    net, x0, _, _, _ = tie_network(M, coupled=True)
    a0 = tie_network(M, coupled=True)[3] / 8.0            # a_k(X0), exact (see tie_cases.py)
    opts = [("bundle_ctas", ctas), ("exchange", exchange), ("pipeline", pipeline)]
    # (a) dt_k = 8 * (1 + eps_k), eps_k in [1e-9, 1e-6]
    eps = 10.0 ** rng.uniform(-9, -6, size=M)
    _check_resume_state(rt, net, x0, np.zeros(M), a0 * 8.0 * (1.0 + eps), 600, opts)
    # (b) every third channel carries a huge internal time; waiting times spread over a decade
    big = (np.arange(M) % 3 == 1)
    T0 = np.where(big, 2.0 ** 40 * (1.0 + rng.uniform(0, 1, size=M)), 0.0)
    P0 = T0 + a0 * 10.0 ** rng.uniform(-1, 0, size=M)
    g, o = _check_resume_state(rt, net, x0, T0, P0, 900, opts)
    assert big[g["trace_mu"]].sum() > 100 and (~big)[g["trace_mu"]].sum() > 100


def test_exact_ties_full_recompute_and_thread_kernel(rt):
    _check_tie(rt, 1201, True, 0, [("refresh_mode", 1)])
    # one-thread-per-trajectory kernel: no trace there, so the order shows in the counts --
    # after j firings exactly the channels 0..j-1 have fired once, all at t = 8.0
    M = 40
    net, x0, T0, P0, n0 = tie_network(M, coupled=True)
    with rt.Model(net) as m:
        m.set_option("ensemble_path", 1)
        for j in (1, 2, 17, M):
            g = m.run_resume(x0, 0.0, T0, P0, n0, 9, 1, j, math.inf, want_state=True)
            assert m.info("ensemble_path") == 1
            assert g["t"] == 8.0 and g["firings"] == j
            np.testing.assert_array_equal(g["fire_count"], (np.arange(M) < j).astype(np.uint64))
            o = _oracle().run_from(net, x0, 0.0, T0, P0, n0, 9, 1, j, math.inf)
            np.testing.assert_array_equal(g["x"], o["x"])
            np.testing.assert_allclose(g["P"], o["P"], rtol=1e-12)


@pytest.mark.parametrize("formulation,state_mode", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_resume_continues_bit_for_bit(rt, formulation, state_mode):
    """rt_run to n1 firings + rt_run_resume for n2 - n1 more == rt_run to n2 (include/rt.h), and
    both equal the oracle; also across a t_end stop."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    with rt.Model(net) as m:
        m.set_option("formulation", formulation)
        m.set_option("state_mode", state_mode)
        a = m.run(x0, 7, 4, 700, math.inf, 700, want_state=True)
        b = m.run_resume(a["x"], a["t"], a["T"], a["P"], a["fire_count"], 7, 4, 800, math.inf, 800,
                         want_state=True)
        c = m.run(x0, 7, 4, 1500, math.inf, 1500, want_state=True)
        t_end = float(c["trace_t"][1100]) * 1.0000001
        d = m.run_resume(a["x"], a["t"], a["T"], a["P"], a["fire_count"], 7, 4, 0, t_end, 4096)
    np.testing.assert_array_equal(b["trace_mu"], c["trace_mu"][700:])
    np.testing.assert_array_equal(b["trace_t"], c["trace_t"][700:])
    for key in ("x", "fire_count", "T", "P"):
        np.testing.assert_array_equal(b[key], c[key])
    assert b["t"] == c["t"] and b["firings"] == 800
    assert d["stop"] == rt.RT_STOP_T_END and d["t"] == t_end and d["firings"] == 401
    run = _oracle().run_residual if formulation else _oracle().run
    o = run(net, x0, 7, 4, 1500, math.inf, 1500)
    np.testing.assert_array_equal(c["trace_mu"], o["trace_mu"])


def test_resume_argument_checks(rt):
    net, x0 = W.lotka_volterra()
    z = np.zeros(3)
    n0 = np.zeros(3, dtype=np.uint64)
    with rt.Model(net) as m:
        assert m.run_resume(x0, 0.0, None, z, n0, 1, 0, 10, check=False)["code"] == rt.RT_ERR_NULL
        assert m.run_resume(x0, -1.0, z, z, n0, 1, 0, 10, check=False)["code"] == rt.RT_ERR_BAD_ARG
        assert m.run_resume(x0, 5.0, z, z, n0, 1, 0, 10, 2.0, check=False)["code"] == rt.RT_ERR_BAD_ARG
        bad = z.copy(); bad[1] = math.nan
        assert m.run_resume(x0, 0.0, bad, z, n0, 1, 0, 10, check=False)["code"] == rt.RT_ERR_BAD_ARG
        big = n0.copy(); big[2] = 2**32
        assert m.run_resume(x0, 0.0, z, z, big, 1, 0, 10, check=False)["code"] == rt.RT_ERR_BAD_ARG
        m.set_rate_schedule([0.5], [2.0])
        assert m.run_resume(x0, 0.0, z, z + 1, n0, 1, 0, 10, check=False)["code"] == rt.RT_ERR_UNSUPPORTED
        # the thread kernel implements neither schedules nor the residual form: forcing it must
        # fail loudly instead of returning constant-rate (T, P) results
        m.set_option("ensemble_path", 1)
        assert m.ensemble(x0, 2, 0, 4, 100, check=False)["code"] == rt.RT_ERR_UNSUPPORTED
        m.set_rate_schedule([], [])
        m.set_option("formulation", 1)
        assert m.ensemble(x0, 2, 0, 4, 100, check=False)["code"] == rt.RT_ERR_UNSUPPORTED
        m.set_option("formulation", 0)
        assert m.ensemble(x0, 2, 0, 4, 100)["code"] == rt.RT_OK


def test_cfg3_full_first_1e4(rt):
    """BASELINE config 3 at full size: first 1e4 firings bit-exact."""
    net, x0, par = W.make_config("cfg3")
    _check_run(rt, net, x0, par["seed"], 0, 10_000, math.inf, 10_000)     # one 16-CTA cluster
    _check_run(rt, net, x0, par["seed"], 0, 10_000, math.inf, 10_000, options=[("exchange", 1)])   # 148 CTAs, L2


def test_cfg4_scaled(rt):
    net, x0, par = W.make_config("cfg4", scale=0.02)
    _check_run(rt, net, x0, par["seed"], 0, 2000, math.inf, 2000)


def test_cfg4_full_first_1e4(rt):
    """BASELINE config 4 (M=1e6, the bench workload) in the launch shape bench.py times:
    the first 1e4 firings, fired sequence and counts bit-exact, times to 1e-12 (the oracle
    needs about a minute for its 1e10 reaction-steps)."""
    net, x0, par = W.make_config("cfg4")
    g, o = _check_run(rt, net, x0, par["seed"], 0, 10_000, math.inf, 10_000)
    assert g["firings"] == 10_000


def test_cfg5a_full_size_full_length(rt):
    """BASELINE config 5a (N=1e6, M=1e7: state streamed from global memory, 512-thread CTAs,
    cooperative re-scan) at full size and full length: all 2 000 firings of the (T, P) form,
    everything _check_run compares; the residual form (24 B per reaction) for its first 400.
    (The oracle needs ~2.5 min for its 2e10 reaction-steps; the two run on two host threads.)"""
    from concurrent.futures import ThreadPoolExecutor
    net, x0, par = W.make_config("cfg5a")
    n = par["max_firings"]
    assert n == 2000 and net["n_reactions"] == 10_000_000
    with ThreadPoolExecutor(2) as ex:
        fo = ex.submit(_oracle().run, net, x0, par["seed"], 0, n, math.inf, n)
        nr = 400
        fr = ex.submit(_oracle().run_residual, net, x0, par["seed"], 0, nr, math.inf, nr)
        with rt.Model(net) as m:
            g = m.run(x0, par["seed"], 0, n, math.inf, n, want_state=True)
            assert m.info("state_in_smem") == 0 and m.info("bundle_ctas") == m.info("num_sms")
            m.set_option("formulation", 1)
            gr = m.run(x0, par["seed"], 0, nr, math.inf, nr, want_state=True)
        o, orr = fo.result(), fr.result()
    assert g["firings"] == n and gr["firings"] == nr
    for a, b in ((g, o), (gr, orr)):
        assert a["firings"] == b["firings"] and a["stop"] == b["stop"]
        np.testing.assert_array_equal(a["trace_mu"], b["trace_mu"])
        np.testing.assert_array_equal(a["x"], b["x"])
        np.testing.assert_array_equal(a["fire_count"], b["fire_count"])
        np.testing.assert_allclose(a["trace_t"], b["trace_t"], rtol=RTOL_T, atol=0)
        assert math.isclose(a["t"], b["t"], rel_tol=RTOL_T, abs_tol=0)
    np.testing.assert_allclose(g["T"], o["T"], rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(g["P"], o["P"], rtol=1e-12, atol=0)
    np.testing.assert_allclose(-gr["T"], orr["R"], rtol=1e-10, atol=1e-12)


def test_cfg5b_full_size_ensemble(rt):
    """BASELINE config 5b: 64 trajectories of the M=1e5 network in the bench launch shape
    (several bundles with on-chip state); every row against the oracle for 2 500 firings, and
    trajectory 0 traced through rt_run in the same bundle shape."""
    net, x0, par = W.make_config("cfg5b")
    n, firings = 64, 2500
    o = _oracle().ensemble(net, x0, par["seed"], 0, n, firings, math.inf, n_threads=os.cpu_count() or 8)
    o0 = _oracle().run(net, x0, par["seed"], 0, firings, math.inf, firings)
    with rt.Model(net) as m:
        g = m.ensemble(x0, par["seed"], 0, n, firings, math.inf)
        assert m.info("ensemble_path") == 2 and m.info("state_in_smem") == 1
        shape = m.info("bundle_ctas")
        m.set_option("bundle_ctas", shape)
        g0 = m.run(x0, par["seed"], 0, firings, math.inf, firings)
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["firings"], o["firings"])
    np.testing.assert_array_equal(g["stop"], o["stop"])
    np.testing.assert_allclose(g["t"], o["t"], rtol=RTOL_T)
    np.testing.assert_array_equal(g0["trace_mu"], o0["trace_mu"])
    np.testing.assert_allclose(g0["trace_t"], o0["trace_t"], rtol=RTOL_T, atol=0)
    np.testing.assert_array_equal(g0["x"], g["x"][0])


def test_t_end_stop_and_absorption(rt):
    net, x0, par = W.make_config("cfg3", scale=0.01)
    g, o = _check_run(rt, net, x0, 11, 0, 0, 0.002, 4096)
    assert g["stop"] == rt.RT_STOP_T_END and g["t"] == 0.002
    # pure death from 5 molecules: absorbed after exactly 5 firings
    dnet = W.from_reactions(1, [({0: 1}, {}, 0.7)])
    g, o = _check_run(rt, dnet, np.array([5]), 3, 0, 0, 1e9, 16)
    assert g["stop"] == rt.RT_STOP_ABSORBED and g["firings"] == 5


def test_tiny_networks_on_bundle_path(rt):
    for builder in (W.birth_death, W.lotka_volterra):
        net, x0 = builder()
        _check_run(rt, net, x0, 5, 9, 2000, math.inf, 2000)


def test_ensemble_thread_path_matches_oracle(rt):
    """cfg1 / cfg2 ensembles (one thread per trajectory) against the oracle, row by row."""
    net, x0, par = W.make_config("cfg1")
    n = 67
    o = _oracle().ensemble(net, x0, par["seed"], 5, n, par["max_firings"], 50.0)
    with rt.Model(net) as m:
        g = m.ensemble(x0, par["seed"], 5, n, par["max_firings"], 50.0)
        assert m.info("ensemble_path") == 1
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["firings"], o["firings"])
    np.testing.assert_array_equal(g["stop"], o["stop"])
    np.testing.assert_allclose(g["t"], o["t"], rtol=RTOL_T)
    net, x0, par = W.make_config("cfg2")
    n = 45
    o = _oracle().ensemble(net, x0, par["seed"], 0, n, 20_000, 0.5)
    with rt.Model(net) as m:
        g = m.ensemble(x0, par["seed"], 0, n, 20_000, 0.5)
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["firings"], o["firings"])
    np.testing.assert_allclose(g["t"], o["t"], rtol=RTOL_T)


@pytest.mark.parametrize("tiny", [1, 0])
def test_tiny_networks_register_and_shared_memory_thread_kernels(rt, tiny):
    """One thread per trajectory, both kernels: rt_tiny_kernel (state in registers: at most 4
    reactions of at most 2 reactants over at most 4 species) and the general rt_thread_kernel give
    the oracle's rows -- stops by t_end, max_firings, absorption and count overflow, sigma = 2 and
    sigma = 3 reactants, a reaction without reactants, checkpointed single trajectories."""
    cases = []
    net, x0, par = W.make_config("cfg2")
    cases.append((net, x0, par["seed"], 33, 3000, 0.2))
    net, x0, par = W.make_config("cfg1")
    cases.append((net, x0, par["seed"], 40, 0, 30.0))
    # dimerisation 2A <-> B, trimer 3A -> C, source 0 -> A, decay C -> 0 (4 reactions, 3 species)
    net = W.from_reactions(3, [({0: 2}, {1: 1}, 0.02), ({1: 1}, {0: 2}, 1.0), ({0: 3}, {2: 1}, 1e-4),
                               ({}, {0: 1}, 5.0)])
    cases.append((net, np.array([60, 5, 0]), 7, 50, 500, math.inf))
    # pure death: absorbed
    net = W.from_reactions(2, [({0: 1}, {1: 1}, 1.0), ({1: 1}, {}, 2.0)])
    cases.append((net, np.array([30, 0]), 8, 25, 0, 1e9))
    for net, x0, seed, n, mf, t_end in cases:
        o = _oracle().ensemble(net, x0, seed, 2, n, mf, t_end)
        with rt.Model(net) as m:
            m.set_option("tiny_kernel", tiny)
            m.set_option("ensemble_path", 1)
            g = m.ensemble(x0, seed, 2, n, mf, t_end)
            assert m.info("ensemble_path") == 1 and m.info("tiny_kernel") == tiny
        np.testing.assert_array_equal(g["x"], o["x"])
        np.testing.assert_array_equal(g["firings"], o["firings"])
        np.testing.assert_array_equal(g["stop"], o["stop"])
        np.testing.assert_allclose(g["t"], o["t"], rtol=RTOL_T)
    # checkpoint / resume of one trajectory through the thread path
    net, x0, par = W.make_config("cfg2")
    with rt.Model(net) as m:
        m.set_option("tiny_kernel", tiny)
        m.set_option("ensemble_path", 1)
        a = m.run(x0, 3, 9, 700, math.inf, want_state=True)
        b1 = m.run(x0, 3, 9, 300, math.inf, want_state=True)
        b2 = m.run_resume(b1["x"], b1["t"], b1["T"], b1["P"], b1["fire_count"], 3, 9, 400, math.inf, want_state=True)
        assert m.info("tiny_kernel") == tiny
    o = _oracle().run(net, x0, 3, 9, 700, math.inf)
    np.testing.assert_array_equal(a["x"], o["x"])
    np.testing.assert_array_equal(b2["x"], a["x"])
    assert b2["t"] == a["t"]
    np.testing.assert_array_equal(b2["P"], a["P"])
    np.testing.assert_array_equal(b2["T"], a["T"])
    # count overflow on the thread path: the offending update is not applied
    net = W.from_reactions(1, [({}, {0: 1}, 1.0)])
    xmax = 2**31 - 1
    with rt.Model(net) as m:
        m.set_option("tiny_kernel", tiny)
        m.set_option("ensemble_path", 1)
        g = m.ensemble(np.array([xmax - 2]), 1, 0, 3, 10, math.inf, check=False)
    assert g["code"] == rt.RT_ERR_OVERFLOW
    np.testing.assert_array_equal(g["x"][:, 0], [xmax] * 3)
    np.testing.assert_array_equal(g["firings"], [3] * 3)


def test_ensemble_bundle_path_matches_run_and_oracle(rt):
    """cfg5b shape (several trajectories of one mid-size network): ensemble row i == rt_run(i)
    == oracle trajectory i; thread path and bundle path agree on a tiny network."""
    net, x0, par = W.make_config("cfg5b", scale=0.02)
    n = 5
    o = _oracle().ensemble(net, x0, par["seed"], 2, n, 800, math.inf)
    with rt.Model(net) as m:
        g = m.ensemble(x0, par["seed"], 2, n, 800, math.inf)
        assert m.info("ensemble_path") == 2
        one = m.run(x0, par["seed"], 4, 800)
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_allclose(g["t"], o["t"], rtol=RTOL_T)
    np.testing.assert_array_equal(one["x"], g["x"][2])
    net, x0 = W.lotka_volterra()
    with rt.Model(net) as m:
        a = m.ensemble(x0, 2, 0, 9, 3000, math.inf)
        m.set_option("ensemble_path", 2)
        b = m.ensemble(x0, 2, 0, 9, 3000, math.inf)
    np.testing.assert_array_equal(a["x"], b["x"])
    np.testing.assert_array_equal(a["t"], b["t"])


def test_prefix_property(rt):
    net, x0, par = W.make_config("cfg3", scale=0.01)
    with rt.Model(net) as m:
        a = m.run(x0, 7, 0, 500, trace_cap=500)
        b = m.run(x0, 7, 0, 1200, trace_cap=1200)
    np.testing.assert_array_equal(a["trace_mu"], b["trace_mu"][:500])
    np.testing.assert_array_equal(a["trace_t"], b["trace_t"][:500])


# ------------------------------------------------------------------ beyond the bit-exact horizon
def _ks_and_moments(a, b):
    """Two-sample KS p-value, and the differences of the means and of the variances in units of
    their standard errors (north_star: "means and variances within 3 standard errors").  The
    sampling variance of s^2 is (m4 - s^4 (n-3)/(n-1)) / n for any law with a fourth moment."""
    from scipy import stats
    p = stats.ks_2samp(a, b).pvalue
    se = math.sqrt(a.var(ddof=1) / len(a) + b.var(ddof=1) / len(b))

    def var_of_var(x):
        n, s2 = len(x), x.var(ddof=1)
        m4 = ((x - x.mean()) ** 4).mean()
        return max(m4 - s2 * s2 * (n - 3) / (n - 1), 0.0) / n
    se_v = math.sqrt(var_of_var(a) + var_of_var(b))
    return (p, abs(a.mean() - b.mean()) / max(se, 1e-300),
            abs(a.var(ddof=1) - b.var(ddof=1)) / max(se_v, 1e-300))


def _assert_within_3se(zs):
    """north_star's bar is "within 3 standard errors": a two-sided false-alarm rate of 0.27 % for ONE
    comparison.  A pre-registered family of m comparisons is held to the same 0.27 % family-wise
    (Holm step-down on the normal tail, exactly as the KS p-values are treated):
    the i-th largest excursion must satisfy 2(1 - Phi(z)) > 0.0027 / (m - i).  For m = 1 this is
    z < 3.0."""
    from scipy import stats
    alpha = 2.0 * stats.norm.sf(3.0)
    ps = sorted(2.0 * stats.norm.sf(np.asarray(zs, dtype=float)))
    for rank, pv in enumerate(ps):
        assert pv > alpha / (len(ps) - rank), (rank, pv, sorted(zs, reverse=True)[:3])


def test_cfg1_ensemble_statistics(rt):
    """BASELINE config 1 in full: 1000 birth-death trajectories to t_end = 1000 (~2e4 firings each,
    far past the bit-exact horizon).  Same Philox seed: rows identical to the oracle's.  A different
    seed on the GPU side (so the test is not vacuous): mean and variance of X within 3 standard
    errors of the stationary Poisson(100) law and of the oracle's sample, KS p > 0.01."""
    from scipy import stats
    net, x0, par = W.make_config("cfg1")
    n = 1000
    o = _oracle().ensemble(net, x0, par["seed"], 0, n, par["max_firings"], 1000.0, n_threads=8)
    with rt.Model(net) as m:
        same = m.ensemble(x0, par["seed"], 0, n, par["max_firings"], 1000.0)
        other = m.ensemble(x0, par["seed"] + 12345, 0, n, par["max_firings"], 1000.0)
    np.testing.assert_array_equal(same["x"], o["x"])
    np.testing.assert_array_equal(same["firings"], o["firings"])
    assert (other["stop"] == rt.RT_STOP_T_END).all() and (other["t"] == 1000.0).all()
    xg, xo = other["x"][:, 0].astype(float), o["x"][:, 0].astype(float)
    assert abs(xg.mean() - 100.0) < 3 * math.sqrt(100.0 / n)
    assert abs(xg.var(ddof=1) - 100.0) < 3 * 100.0 * math.sqrt(2.0 / (n - 1)) + 3 * math.sqrt(100.0 / n)
    p, z, zv = _ks_and_moments(xg, xo)
    assert p > 0.01 and z < 3.0 and zv < 3.0              # (one species: plain 3 SE each)
    # exact law: KS against the Poisson(100) CDF is conservative for a discrete law
    assert stats.kstest(xg, stats.poisson(100).cdf).pvalue > 0.01


def test_cfg2_ensemble_statistics(rt):
    """BASELINE config 2 shape (Lotka-Volterra, one thread per trajectory), t_end = 1 (~3e4 firings
    per trajectory): same seed -> identical rows; different seed -> both species' marginals agree
    with the oracle's (means and variances within 3 SE, KS p > 0.01, Holm over the two species).
    The config's own size (1e5 trajectories to t_end = 10, 3e10 steps) is bench.py's cfg2 run, far
    beyond what the oracle can follow; this is the same path at a size it can."""
    net, x0, par = W.make_config("cfg2")
    n = 2000
    o = _oracle().ensemble(net, x0, par["seed"], 0, n, par["max_firings"], 1.0, n_threads=os.cpu_count() or 8)
    with rt.Model(net) as m:
        same = m.ensemble(x0, par["seed"], 0, n, par["max_firings"], 1.0)
        other = m.ensemble(x0, par["seed"] + 777, 0, n, par["max_firings"], 1.0)
        assert m.info("ensemble_path") == 1
    np.testing.assert_array_equal(same["x"], o["x"])
    np.testing.assert_array_equal(same["firings"], o["firings"])
    ps, zs = [], []
    for j in range(2):
        p, z, zv = _ks_and_moments(other["x"][:, j].astype(float), o["x"][:, j].astype(float))
        ps.append(p)
        zs += [z, zv]
    ps.sort()
    assert ps[0] > 0.01 / 2 and ps[1] > 0.01      # Holm-corrected
    _, fz, fzv = _ks_and_moments(other["firings"].astype(float), o["firings"].astype(float))
    _assert_within_3se(zs + [fz, fzv])


# ------------------------------------------------------------------ residual (Table 3) formulation
def _check_residual(rt, net, x0, seed, traj, max_firings, t_end, trace_cap, options=()):
    o = _oracle().run_residual(net, x0, seed, traj, max_firings, t_end, trace_cap)
    with rt.Model(net) as m:
        m.set_option("formulation", 1)
        for name, val in options:
            m.set_option(name, val)
        g = m.run(x0, seed, traj, max_firings, t_end, trace_cap, want_state=True)
    assert g["firings"] == o["firings"] and g["stop"] == o["stop"]
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)
    # T_out holds -R_k, P_out zeros
    np.testing.assert_allclose(-g["T"], o["R"], rtol=1e-10, atol=1e-12)
    assert not g["P"].any()
    return g, o


@pytest.mark.parametrize("ctas,state_mode", [(0, 0), (3, 0), (0, 1), (1, 1)])
def test_residual_form_matches_its_oracle(rt, ctas, state_mode):
    """PAPER.md Table 3 in residual form (formulation = 1) against oracle_run_residual: fired
    sequence and counts bit-exact, times to 1e-12 -- with the state in shared memory and streamed
    from global memory (where P is not read at all: 24 instead of 32 bytes per reaction)."""
    net, x0, par = W.make_config("cfg3", scale=0.03)
    _check_residual(rt, net, x0, par["seed"], 1, 1500, math.inf, 1500,
                    options=[("bundle_ctas", ctas), ("state_mode", state_mode)])
    net, x0 = _hub_network()
    _check_residual(rt, net, x0, 21, 0, 400, math.inf, 400,
                    options=[("bundle_ctas", ctas), ("state_mode", state_mode)])


def test_residual_form_stops_and_full_recompute(rt):
    net, x0, par = W.make_config("cfg3", scale=0.01)
    g, o = _check_residual(rt, net, x0, 11, 0, 0, 0.002, 4096)
    assert g["stop"] == rt.RT_STOP_T_END and g["t"] == 0.002
    _check_residual(rt, net, x0, 11, 0, 700, math.inf, 700, options=[("refresh_mode", 1)])
    net, x0 = W.lotka_volterra()
    _check_residual(rt, net, x0, 5, 9, 2000, math.inf, 2000)


def test_residual_form_cfg4_prefix_and_differs_from_default(rt):
    """Bench shape (M = 1e6): 1500 firings against the residual oracle.  The two formulations
    are the same process but round differently, so their paths eventually part."""
    net, x0, par = W.make_config("cfg4")
    g, o = _check_residual(rt, net, x0, par["seed"], 0, 1500, math.inf, 1500)
    with rt.Model(net) as m:
        d = m.run(x0, par["seed"], 0, 1500, trace_cap=1500)
    assert d["trace_mu"][0] == g["trace_mu"][0]          # same first draws -> same first firing


# ------------------------------------------------------------------ time-dependent rates (Eq.28)
def _check_sched(rt, net, x0, seed, traj, max_firings, t_end, trace_cap, t_break, factor, mask,
                 options=()):
    o = _oracle().run_sched(net, x0, seed, traj, max_firings, t_end, trace_cap,
                            t_break=t_break, factor=factor, mask=mask)
    with rt.Model(net) as m:
        for name, val in options:
            m.set_option(name, val)
        m.set_rate_schedule(t_break, factor, mask)
        g = m.run(x0, seed, traj, max_firings, t_end, trace_cap, want_state=True)
    assert g["firings"] == o["firings"] and g["stop"] == o["stop"]
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)
    assert math.isclose(g["t"], o["t"], rel_tol=RTOL_T, abs_tol=0)
    np.testing.assert_allclose(g["T"], o["T"], rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(g["P"], o["P"], rtol=1e-12, atol=0)
    return g, o


@pytest.mark.parametrize("ctas,state_mode", [(0, 0), (3, 0), (1, 1), (0, 1)])
def test_time_dependent_rates_match_oracle(rt, ctas, state_mode):
    """PAPER.md Eq.28 with piecewise-constant c_k(t): several breakpoints inside the run (the
    network fires ~2e5 times per unit time, so they fall between firings), a zero-rate window
    for a masked half of the reactions, with the state in shared and in global memory."""
    net, x0, par = W.make_config("cfg3", scale=0.03)
    M = int(net["n_reactions"])
    mask = (np.arange(M) % 2).astype(np.uint8)
    o0 = _oracle().run(net, x0, par["seed"], 1, 1200, math.inf, 1200)
    tt = o0["trace_t"]
    t_break = [float(tt[150]) * 1.0000001, float(tt[400]), float(tt[800]) * 0.9999999]
    factor = [3.0, 0.0, 0.5]
    opts = [("bundle_ctas", ctas), ("state_mode", state_mode)]
    _check_sched(rt, net, x0, par["seed"], 1, 1500, math.inf, 1500, t_break, factor, mask, opts)
    _check_sched(rt, net, x0, par["seed"], 1, 1500, math.inf, 1500, t_break, factor, None, opts)
    # a t_end between two breakpoints: later breakpoints must not act
    g, o = _check_sched(rt, net, x0, par["seed"], 1, 0, float(tt[600]), 4096, t_break, factor, mask, opts)
    assert g["stop"] == rt.RT_STOP_T_END


def test_time_dependent_rates_revive_an_absorbed_state(rt):
    """All rates 0 until the first breakpoint: nothing can fire, the run must jump to the
    breakpoint instead of reporting ABSORBED, then proceed; hub network (pre-walk, staging rounds)."""
    net, x0 = _hub_network()
    o0 = _oracle().run(net, x0, 21, 0, 300, math.inf, 300)
    b1 = float(o0["trace_t"][100])
    _check_sched(rt, net, x0, 21, 0, 500, math.inf, 500, [0.0, b1, 2 * b1], [0.0, 1.0, 2.5], None)


@pytest.mark.parametrize("pipeline,exchange", [(1, 0), (1, 1), (0, 0)])
def test_ensemble_to_t_end_on_the_bundle_path(rt, pipeline, exchange):
    """Trajectories of a mid-size network that stop at t_end after DIFFERENT numbers of firings,
    more trajectories than bundles (the bundles pick up their next trajectory at different times):
    every row against the oracle, stop reason and clock included."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    o1 = _oracle().run(net, x0, 11, 0, 600, math.inf, 600)
    t_end = float(o1["trace_t"][450])
    n = 23
    o = _oracle().ensemble(net, x0, 11, 0, n, 0, t_end)
    assert len(set(o["firings"].tolist())) > 5
    with rt.Model(net) as m:
        m.set_option("ensemble_path", 2)
        m.set_option("pipeline", pipeline)
        m.set_option("exchange", exchange)
        m.set_option("bundle_ctas", 4)
        g = m.ensemble(x0, 11, 0, n, 0, t_end)
        assert m.info("pipeline") == pipeline and m.info("bundles") >= 2
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["firings"], o["firings"])
    np.testing.assert_array_equal(g["stop"], o["stop"])
    assert (g["stop"] == rt.RT_STOP_T_END).all() and (g["t"] == t_end).all()


def test_kernels_agree_bit_for_bit_far_beyond_the_horizon(rt):
    """1.5e5 firings of a cfg3-like network -- fifteen times the bit-exact horizon north_star sets
    for GPU vs oracle.  Between host and device a one-ulp difference of a log grows tenfold every
    ~1e4 firings until two events swap (reading G9; pinned on the oracle alone by
    test_one_ulp_in_one_draw_bounds_the_bit_exact_horizon), so against the oracle only the first
    5e4 firings are compared, with the drift of the event times inside that envelope.  But every
    GPU path performs the SAME rounded operations in the same order, so all of them -- candidate-
    first and pass-then-reduce kernel, cluster and L2 exchange, 1 to 16 CTAs, state on chip or in
    global memory -- must agree with one another to the last bit over the whole run."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    nf = 150_000
    o = _oracle().run(net, x0, par["seed"], 0, 50_000, math.inf, 50_000)
    runs = []
    for opts in ((), (("pipeline", 0),), (("exchange", 1),), (("bundle_ctas", 1),), (("bundle_ctas", 16),),
                 (("state_mode", 1),), (("pipeline", 0), ("exchange", 1), ("bundle_ctas", 7))):
        with rt.Model(net) as m:
            for k, v in opts:
                m.set_option(k, v)
            runs.append(m.run(x0, par["seed"], 0, nf, math.inf, nf, want_state=True))
    g = runs[0]
    np.testing.assert_array_equal(g["trace_mu"][:50_000], o["trace_mu"])
    rel = np.abs(g["trace_t"][:50_000] - o["trace_t"]) / o["trace_t"]
    assert rel[:10_000].max() < RTOL_T and rel.max() < 1e-8
    for h in runs[1:]:
        np.testing.assert_array_equal(h["trace_mu"], g["trace_mu"])
        np.testing.assert_array_equal(h["trace_t"], g["trace_t"])
        np.testing.assert_array_equal(h["x"], g["x"])
        np.testing.assert_array_equal(h["T"], g["T"])
        np.testing.assert_array_equal(h["P"], g["P"])
        np.testing.assert_array_equal(h["fire_count"], g["fire_count"])


def test_options_are_validated_and_reported(rt):
    """Every tuning knob of rt.h: out-of-range values and unknown names are refused, accepted values
    show up in rt_get_info after a launch, and none of them changes a result."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    ranges = {"refresh_mode": (0, 1), "bundle_ctas": (0, 1024), "ensemble_path": (0, 2), "formulation": (0, 1),
              "prefetch": (0, 7), "x_replicas": (0, 64), "state_mode": (0, 1), "exchange": (0, 1),
              "pipeline": (0, 1), "l2_persist": (0, 2), "tiny_kernel": (0, 1)}
    with rt.Model(net) as m:
        for name, (lo, hi) in ranges.items():
            for bad in (lo - 1, hi + 1):
                assert rt.rt_set_option(m.handle, name, bad) == rt.RT_ERR_BAD_ARG, (name, bad)
            assert rt.rt_set_option(m.handle, name, lo) == rt.RT_OK
        assert rt.rt_set_option(m.handle, "no_such_option", 0) == rt.RT_ERR_BAD_ARG
        with pytest.raises(rt.RtError):
            m.info("no_such_info")
        base = m.run(x0, 3, 0, 400, math.inf, 400)
        assert m.info("pipeline") == 0 and m.info("cluster_exchange") == 1 and m.info("state_in_smem") == 1
        for name, val in (("pipeline", 1), ("exchange", 1), ("prefetch", 0), ("prefetch", 7), ("x_replicas", 2),
                          ("state_mode", 1), ("l2_persist", 0), ("l2_persist", 1), ("bundle_ctas", 3)):
            m.set_option(name, val)
            g = m.run(x0, 3, 0, 400, math.inf, 400)
            np.testing.assert_array_equal(g["trace_mu"], base["trace_mu"])
            np.testing.assert_array_equal(g["trace_t"], base["trace_t"])
            np.testing.assert_array_equal(g["x"], base["x"])
        assert m.info("state_in_smem") == 0 and m.info("bundle_ctas") == 3 and m.info("l2_persist") in (0, 1)


def test_rate_schedule_validation_and_unsupported_combinations(rt):
    net, x0 = W.lotka_volterra()
    with rt.Model(net) as m:
        assert rt.rt_set_rate_schedule(m.handle, [1.0, 0.5], [1.0, 1.0]) == rt.RT_ERR_BAD_ARG   # not increasing
        assert rt.rt_set_rate_schedule(m.handle, [-1.0], [1.0]) == rt.RT_ERR_BAD_ARG
        assert rt.rt_set_rate_schedule(m.handle, [1.0], [-2.0]) == rt.RT_ERR_BAD_ARG
        assert rt.rt_set_rate_schedule(m.handle, [1.0], [math.inf]) == rt.RT_ERR_BAD_ARG
        m.set_rate_schedule([0.01], [2.0])
        m.set_option("refresh_mode", 1)
        assert m.run(x0, 1, 0, 10, check=False)["code"] == rt.RT_ERR_UNSUPPORTED
        m.set_option("refresh_mode", 0)
        ens = m.ensemble(x0, 2, 0, 5, 300, math.inf)          # tiny network, schedule -> bundle path
        assert m.info("ensemble_path") == 2
        o = [_oracle().run_sched(net, x0, 2, i, 300, math.inf, 0, t_break=[0.01], factor=[2.0])["x"] for i in range(5)]
        np.testing.assert_array_equal(ens["x"], np.array(o))
        m.set_rate_schedule([], [])                            # removed again
        a = m.run(x0, 2, 0, 300)
        np.testing.assert_array_equal(a["x"], _oracle().run(net, x0, 2, 0, 300)["x"])


# ------------------------------------------------- smooth time-dependent rates (Eq.28, exponential)
def _check_rate_exp(rt, net, x0, lam, seed, traj, max_firings, t_end, trace_cap, options=()):
    """GPU vs oracle_run_rate_exp.  exp / log1p / expm1 are glibc's on the host and CUDA's on the
    device (<= 2 ulp apart), so the bar is DESIGN.md's for this mode: fired sequence, counts and
    stop reason exact over the tested horizon, times to 1e-12, clocks to 1e-10."""
    o = _oracle().run_rate_exp(net, x0, lam, seed, traj, max_firings, t_end, trace_cap)
    with rt.Model(net) as m:
        for name, val in options:
            m.set_option(name, val)
        m.set_rate_exponent(lam)
        g = m.run(x0, seed, traj, max_firings, t_end, trace_cap, want_state=True)
    assert g["firings"] == o["firings"] and g["stop"] == o["stop"]
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["fire_count"], o["fire_count"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)
    assert math.isclose(g["t"], o["t"], rel_tol=RTOL_T, abs_tol=0)
    np.testing.assert_allclose(g["T"], o["T"], rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(g["P"], o["P"], rtol=1e-12, atol=0)
    return g, o


@pytest.mark.parametrize("ctas,state_mode", [(0, 0), (3, 0), (1, 1), (0, 1)])
def test_exponential_rates_match_oracle(rt, ctas, state_mode):
    """PAPER.md Eq.28 with c_k(t) = c_k exp(lambda_k t), per-channel lambda_k (growth, decay strong
    enough that channels go silent, and 0 = constant): every channel solves its own equation in
    closed form.  lambda is scaled by the duration of the constant-rate run so that lambda t = O(1)."""
    net, x0, par = W.make_config("cfg3", scale=0.03)
    M = int(net["n_reactions"])
    plain = _oracle().run(net, x0, par["seed"], 1, 2500, math.inf, 2500)
    lam = np.random.default_rng(17).choice([0.0, 0.6, -1.5, 0.15, -8.0], size=M) / float(plain["trace_t"][-1])
    opts = [("bundle_ctas", ctas), ("state_mode", state_mode)]
    g, o = _check_rate_exp(rt, net, x0, lam, par["seed"], 1, 2500, math.inf, 2500, opts)
    assert not np.array_equal(plain["trace_mu"], o["trace_mu"])       # (the exponents do act)
    # a time limit inside the run: closing pass advances every clock with expm1
    g, o = _check_rate_exp(rt, net, x0, lam, par["seed"], 1, 0, float(o["trace_t"][1400]) * 1.0000001, 4096, opts)
    assert g["stop"] == rt.RT_STOP_T_END and g["firings"] == 1401


def test_exponential_rates_decay_to_silence_hub_network_and_ensemble(rt):
    """Every channel decays: the run ends ABSORBED once no channel's remaining integral covers its
    residual.  Hub network (staging rounds, general rows); then an ensemble row by row."""
    net, x0 = _hub_network()
    M = int(net["n_reactions"])
    o0 = _oracle().run(net, x0, 21, 0, 300, math.inf, 300)
    # One common lambda < 0 is a time change of the constant-rate run: internal time saturates at
    # 1/|lambda|, so the decaying run fires exactly the constant-rate firings before that instant.
    # Put it BETWEEN two firings (on a firing time the last channel's argument is -1 +- rounding).
    lam = np.full(M, -2.0 / float(o0["trace_t"][200] + o0["trace_t"][201]))
    g, o = _check_rate_exp(rt, net, x0, lam, 21, 0, 100000, math.inf, 4096)
    assert g["stop"] == rt.RT_STOP_ABSORBED and g["firings"] == 201
    np.testing.assert_array_equal(g["trace_mu"][:201], o0["trace_mu"][:201])
    net, x0 = W.lotka_volterra(y1=60, y2=40, c1=2.0, c2=0.02, c3=1.5)
    lam3 = [0.4, -0.3, 0.0]
    with rt.Model(net) as m:
        m.set_rate_exponent(lam3)
        ens = m.ensemble(x0, 5, 10, 6, 0, 1.5)
        assert m.info("ensemble_path") == 2                    # (the thread kernel has constant rates only)
        m.set_option("ensemble_path", 1)
        assert m.ensemble(x0, 5, 10, 6, 0, 1.5, check=False)["code"] == rt.RT_ERR_UNSUPPORTED
        m.set_option("ensemble_path", 0)
        m.set_option("formulation", 1)
        assert m.run(x0, 5, 0, 10, check=False)["code"] == rt.RT_ERR_UNSUPPORTED
        m.set_option("formulation", 0)
        assert rt.rt_set_rate_exponent(m.handle, [0.1, math.nan, 0.0], 3) == rt.RT_ERR_BAD_ARG
        m.set_rate_exponent(None)                              # removed again: constant rates
        a = m.run(x0, 5, 0, 300)
        np.testing.assert_array_equal(a["x"], _oracle().run(net, x0, 5, 0, 300)["x"])
    rows = [_oracle().run_rate_exp(net, x0, lam3, 5, 10 + i, 0, 1.5) for i in range(6)]
    np.testing.assert_array_equal(ens["x"], np.array([r["x"] for r in rows]))
    np.testing.assert_array_equal(ens["firings"], np.array([r["firings"] for r in rows]))


def test_global_state_odd_M_and_ensembles(rt):
    """State in global memory with an odd number of reactions (one padding slot in the last
    16-byte pair), for single runs in both formulations and for a multi-bundle ensemble."""
    net, x0 = _hub_network(n_species=30, n_reactions=4999, seed=9)
    assert net["n_reactions"] % 2 == 1
    for ctas in (1, 4):
        _check_run(rt, net, x0, 13, 0, 400, math.inf, 400,
                   options=[("state_mode", 1), ("bundle_ctas", ctas)])
        _check_residual(rt, net, x0, 13, 0, 400, math.inf, 400,
                        options=[("state_mode", 1), ("bundle_ctas", ctas)])
    n = 7
    o = _oracle().ensemble(net, x0, 13, 3, n, 300, math.inf)
    with rt.Model(net) as m:
        m.set_option("state_mode", 1)
        m.set_option("bundle_ctas", 2)
        g = m.ensemble(x0, 13, 3, n, 300, math.inf)
        assert m.info("ensemble_path") == 2 and m.info("state_in_smem") == 0 and m.info("bundles") >= 2
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_array_equal(g["firings"], o["firings"])
    np.testing.assert_allclose(g["t"], o["t"], rtol=RTOL_T)


def test_cfg3_scaled_ensemble_beyond_the_bit_exact_horizon(rt):
    """Past the first 1e4 firings north_star asks for statistical agreement: 96 trajectories of a
    cfg3-like network run to 3e4 firings each.  Same seed: still identical to the oracle (the only
    host/device difference is the last bit of a log now and then).  Different seed on the GPU side:
    means within 3 standard errors and KS p > 0.01 (Holm) on 8 pre-registered species marginals and
    on the elapsed time."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    n, firings = 96, 30_000
    species = [0, 1, 2, 3, 5, 8, 13, 21]
    o = _oracle().ensemble(net, x0, par["seed"], 0, n, firings, math.inf, n_threads=os.cpu_count() or 8)
    with rt.Model(net) as m:
        same = m.ensemble(x0, par["seed"], 0, n, firings, math.inf)
        other = m.ensemble(x0, par["seed"] + 99, 0, n, firings, math.inf)
        assert m.info("ensemble_path") == 2
    np.testing.assert_array_equal(same["x"], o["x"])
    np.testing.assert_allclose(same["t"], o["t"], rtol=1e-11)
    ps, zs = [], []
    for j in species:
        p, z, zv = _ks_and_moments(other["x"][:, j].astype(float), o["x"][:, j].astype(float))
        ps.append(p)
        zs += [z, zv]
    p, z, zv = _ks_and_moments(other["t"], o["t"])
    ps.append(p)
    _assert_within_3se(zs + [z, zv])
    for rank, p in enumerate(sorted(ps)):
        assert p > 0.01 / (len(ps) - rank), (rank, p)      # Holm step-down


def test_frozen_channels_boundary_condition(rt):
    """PAPER.md Table 2, note (:260): "the boundary conditions can be achieved by restrict the
    firing channels.  Those channels that are forbidden for firing is assigned a frozen internal
    time."  A factor-0 schedule from t = 0 on a mask does exactly that: the masked channels never
    fire and their internal time T_k stays frozen at 0, the others run as in the oracle."""
    net, x0, par = W.make_config("cfg3", scale=0.02)
    M = int(net["n_reactions"])
    mask = (np.arange(M) % 3 == 0).astype(np.uint8)
    g, o = _check_sched(rt, net, x0, par["seed"], 0, 1500, math.inf, 1500, [0.0], [0.0], mask)
    frozen = mask.astype(bool)
    assert not g["fire_count"][frozen].any() and not g["T"][frozen].any()
    assert g["fire_count"][~frozen].sum() == 1500 and g["T"][~frozen].any()


def test_shared_memory_capacity_edge(rt):
    """The largest network whose state still fits in shared memory on 148 SMs (M = 1.3e6:
    8 960 slots = 210 KB per CTA) and the first size that does not (M = 1.4e6 -> global memory)."""
    for scale, smem in ((1.3, 1), (1.4, 0)):
        net, x0, par = W.make_config("cfg4", scale=scale)
        o = _oracle().run(net, x0, par["seed"], 0, 60, math.inf, 60)
        with rt.Model(net) as m:
            g = m.run(x0, par["seed"], 0, 60, math.inf, 60)
            assert m.info("state_in_smem") == smem, (scale, m.info("state_in_smem"))
        np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
        np.testing.assert_array_equal(g["x"], o["x"])
        np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)


# ------------------------------------------------------------------ multi-GPU sharding on the CUDA path
def test_ensemble_sharded_over_the_cuda_path(rt):
    """SURVEY 8(f)-3 on the CUDA path: dist.ensemble_sharded over Model.ensemble in a world_size-1
    process group gives, row by row, what one Model.ensemble call gives (and what every rank of a
    larger group would hold, by the determinism contract: row i = rt_run(trajectory = first + i));
    shard_range blocks run as separate launches reproduce the same rows."""
    import torch.distributed as dist
    net, x0, par = W.make_config("cfg3", scale=0.02)
    n, firings, first = 11, 400, 5
    own = not dist.is_initialized()
    if own:
        dist.init_process_group("gloo", init_method="tcp://127.0.0.1:29617", rank=0, world_size=1)
    try:
        with rt.Model(net) as m:
            whole = m.ensemble(x0, par["seed"], first, n, firings, math.inf)
            sharded = rt.ensemble_sharded(lambda f, c: m.ensemble(x0, par["seed"], f, c, firings, math.inf),
                                          int(net["n_species"]), first, n)
            parts = []
            for rank in range(3):                       # what ranks 0..2 of a 3-GPU job would run
                f, c = rt.shard_range(n, rank, 3)
                parts.append(m.ensemble(x0, par["seed"], first + f, c, firings, math.inf))
    finally:
        if own:
            dist.destroy_process_group()
    for key in ("x", "t", "firings", "stop"):
        np.testing.assert_array_equal(sharded[key], whole[key])
        np.testing.assert_array_equal(np.concatenate([p[key] for p in parts], axis=0), whole[key])
    o = _oracle().ensemble(net, x0, par["seed"], first, n, firings, math.inf)
    np.testing.assert_array_equal(whole["x"], o["x"])


def test_bench_line_on_the_gpu(rt):
    """bench.py's own arm end to end (small step counts): one JSON line with the contract keys,
    the roofline / e2e / clocks objects and the secondary workloads."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--steps", "1", "--warmup", "3",
                        "--no-cpu-baseline"], cwd=root, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["config"]["workload"] == "cfg4" and line["config"]["n_reactions"] == 1_000_000
    assert line["unit"] == "firings/s" and line["value"] > 1e5 and line["gpu_launches"] >= 1
    assert line["e2e"]["value"] > 0 and line["e2e"]["h2d_bytes_per_step"] > 0
    assert line["roofline"]["bound"] == "hbm" and 0 < line["roofline"]["smem_frac"] < 1
    sec = line["secondary"]
    assert set(sec) == {"cfg5a", "cfg5b", "cfg3", "cfg2"}
    assert sec["cfg5a"]["config"]["state_in_shared_memory"] is False
    assert 0.3 < sec["cfg5a"]["roofline"]["frac"] < 1.2
    assert sec["cfg5b"]["unit"] == "trajectory-steps/s" and sec["cfg2"]["roofline"]["bound"] == "alu"
