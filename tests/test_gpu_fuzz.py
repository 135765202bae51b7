"""Randomised parity: seeded random networks, counts and library options (tests/helpers/fuzz_cases.py),
the CUDA path against (1) its own simplest variant, bit for bit, and (2) the oracle.

(2) needs care.  Host `log` (glibc) and device `log` differ by one ulp in about 0.3 % of the draws
(reading G9).  On the fixed configs that difference stays far below the 1e-12 bar over
the tested horizon, but small tightly coupled networks (a handful of species shared by hundreds of
reactions) amplify it by orders of magnitude within a thousand firings -- the oracle perturbed by
one ulp in one draw drifts from ITSELF just as fast.  So the oracle here starts from the device's
own initial draws (read back with t_end = 0), and wherever GPU and oracle still part, the first
bitwise difference of their states must be exactly this: after some firing n, P of the reaction
that fired differs by ONE ulp (its redraw) and nothing else differs.  The oracle then continues
from the GPU's state at n.  Every firing of every case is thereby checked against the oracle's
arithmetic; the only thing taken from the GPU is the last bit of a logarithm."""
import math

import numpy as np
import pytest

from helpers.fuzz_cases import make_case, REFERENCE_OPTIONS, INF

pytestmark = pytest.mark.gpu

RTOL_T = 1e-12
N_CHUNKS, PER_CHUNK = 16, 25          # seeds 1..400, about a minute on one B200


@pytest.fixture(scope="module")
def rt():
    import paper_2103_00405_b200 as rt
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    rt.lib()
    return rt


def _bits(a):
    return np.ascontiguousarray(a, dtype=np.float64).view(np.int64)


def _assert_bitwise(g, h, what):
    for k in ("firings", "stop", "code"):
        assert g[k] == h[k], f"{what}: {k}"
    for k in ("x", "trace_mu", "fire_count"):
        np.testing.assert_array_equal(g[k], h[k], err_msg=f"{what}: {k}")
    for k in ("trace_t", "T", "P"):
        np.testing.assert_array_equal(_bits(g[k]), _bits(h[k]), err_msg=f"{what}: {k}")
    assert _bits([g["t"]])[0] == _bits([h["t"]])[0], f"{what}: t"


def _state_equal(g, o, pos):
    """GPU state after g["firings"] firings from scratch against the oracle segment started at firing pos."""
    return (np.array_equal(_bits(g["T"]), _bits(o["T"])) and np.array_equal(_bits(g["P"]), _bits(o["P"]))
            and np.array_equal(g["x"], o["x"]) and np.array_equal(g["fire_count"], o["fire_count"])
            and g["t"] == o["t"] and g["firings"] == pos + o["firings"])


def _within_bar(o, g, pos):
    """Oracle segment o (started at firing `pos` of the GPU run g) against the rest of g."""
    n = len(o["trace_mu"])
    if pos + o["firings"] != g["firings"] or o["stop"] != g["stop"] or o["code"] != g["code"]:
        return False
    return (np.array_equal(o["trace_mu"], g["trace_mu"][pos:pos + n])
            and np.array_equal(o["x"], g["x"]) and np.array_equal(o["fire_count"], g["fire_count"])
            and np.allclose(g["trace_t"][pos:pos + n], o["trace_t"], rtol=RTOL_T, atol=0)
            and math.isclose(g["t"], o["t"], rel_tol=RTOL_T, abs_tol=0)
            and np.allclose(g["T"], o["T"], rtol=1e-10, atol=1e-12)
            and np.allclose(g["P"], o["P"], rtol=RTOL_T, atol=0))


def _fuzz_one(rt, seed):
    import oracle
    net, x0, opts, firings, traj = make_case(seed)
    assert rt.rt_validate_network(net) == rt.RT_OK
    M = int(net["n_reactions"])
    with rt.Model(net) as m:
        for k, v in opts:
            m.set_option(k, v)
        g = m.run(x0, seed, traj, firings, INF, firings, want_state=True, check=False)
    with rt.Model(net) as ref:
        for k, v in REFERENCE_OPTIONS:
            ref.set_option(k, v)
        h = ref.run(x0, seed, traj, firings, INF, firings, want_state=True, check=False)
        _assert_bitwise(g, h, f"seed {seed} {opts} vs the reference variant")          # (1)

        def gpu_state(c):                  # state after c >= 1 firings, from scratch (deterministic)
            return ref.run(x0, seed, traj, c, INF, 0, want_state=True, check=False)

        # (2) the device's initial draws: one ulp from the oracle's at most
        g0 = ref.run(x0, seed, traj, 0, 0.0, 0, want_state=True, check=False)
        o0 = oracle.run(net, x0, seed, traj, 0, 0.0, 0, check=False)
        assert g0["firings"] == 0 and np.array_equal(g0["T"], o0["T"])
        assert np.abs(_bits(g0["P"]) - _bits(o0["P"])).max() <= 1
        state = dict(x=x0, t=0.0, T=np.zeros(M), P=g0["P"], fire_count=np.zeros(M, dtype=np.uint64))
        pos, resyncs, total = 0, 0, g["firings"]
        while True:
            left = firings - pos
            o = oracle.run_from(net, state["x"], state["t"], state["T"], state["P"], state["fire_count"],
                                seed, traj, left, INF, left, check=False)
            if _within_bar(o, g, pos):
                break
            # first firing count c in (pos, total] after which the states differ
            lo, hi = pos, total
            assert not _state_equal(gpu_state(hi), oracle.run_from(
                net, state["x"], state["t"], state["T"], state["P"], state["fire_count"], seed, traj,
                hi - pos, INF, 0, check=False), pos), f"seed {seed}: outside the bar but states agree at the end"
            while hi - lo > 1:
                mid = (lo + hi) // 2
                om = oracle.run_from(net, state["x"], state["t"], state["T"], state["P"], state["fire_count"],
                                     seed, traj, mid - pos, INF, 0, check=False)
                if _state_equal(gpu_state(mid), om, pos):
                    lo = mid
                else:
                    hi = mid
            gc = gpu_state(hi)
            oc = oracle.run_from(net, state["x"], state["t"], state["T"], state["P"], state["fire_count"],
                                 seed, traj, hi - pos, INF, hi - pos, check=False)
            mu = int(oc["trace_mu"][-1])
            assert mu == int(g["trace_mu"][hi - 1]), f"seed {seed}: different reaction at firing {hi}"
            assert gc["t"] == oc["t"] and np.array_equal(gc["x"], oc["x"])
            assert np.array_equal(gc["fire_count"], oc["fire_count"])
            assert np.array_equal(_bits(gc["T"]), _bits(oc["T"])), f"seed {seed}: T differs after firing {hi}"
            dP = np.nonzero(_bits(gc["P"]) != _bits(oc["P"]))[0]
            assert list(dP) == [mu] and abs(int(_bits(gc["P"])[mu]) - int(_bits(oc["P"])[mu])) == 1, \
                f"seed {seed}: after firing {hi} (mu {mu}) P differs at {dP[:8]}"
            state = dict(x=gc["x"], t=gc["t"], T=gc["T"], P=gc["P"], fire_count=gc["fire_count"])
            pos = hi
            resyncs += 1
            assert resyncs <= 64, f"seed {seed}: {resyncs} resyncs, at firing {pos} of {total}"
            if pos == firings:             # the last redraw of the run: nothing left to compare
                break
    return resyncs


@pytest.mark.parametrize("chunk", range(N_CHUNKS))
def test_random_networks_and_options_against_reference_variant_and_oracle(rt, chunk):
    resyncs = [_fuzz_one(rt, seed) for seed in range(1 + chunk * PER_CHUNK, 1 + (chunk + 1) * PER_CHUNK)]
    assert len(resyncs) == PER_CHUNK


def test_a_known_sensitive_case_is_checked_through_its_resyncs(rt):
    """Seed 136 (296 reactions over 8 species, counts below 30, 2052 firings): one of the cases where a
    one-ulp redraw is amplified past the 1e-12 bar, so that the check above has to follow the GPU
    run through resyncs instead of passing on the first comparison."""
    assert _fuzz_one(rt, 136) >= 1


# ---- the other entry points and modes ----------------------------------------------------------
def _bitwise_common(g, h, what):
    for k in ("firings", "stop", "x", "trace_mu", "fire_count"):
        if k in g and g[k] is not None and k in h and h[k] is not None:
            np.testing.assert_array_equal(np.asarray(g[k]), np.asarray(h[k]), err_msg=f"{what}: {k}")
    for k in ("t", "trace_t"):
        if k in g and g[k] is not None and k in h and h[k] is not None:
            np.testing.assert_array_equal(_bits(g[k]), _bits(h[k]), err_msg=f"{what}: {k}")


def _at_the_bar(g, o):
    ok = (np.array_equal(np.asarray(g["firings"]), np.asarray(o["firings"]))
          and np.array_equal(np.asarray(g["stop"]), np.asarray(o["stop"]))
          and np.array_equal(g["x"], o["x"])
          and np.allclose(np.asarray(g["t"]), np.asarray(o["t"]), rtol=RTOL_T, atol=0))
    if ok and g.get("trace_mu") is not None:
        n = len(o["trace_mu"])
        ok = (len(g["trace_mu"]) == n and np.array_equal(g["trace_mu"], o["trace_mu"])
              and np.allclose(g["trace_t"], o["trace_t"], rtol=RTOL_T, atol=0)
              and np.array_equal(g["fire_count"], o["fire_count"]))
    return ok


def _mode_one(rt, seed):
    """Returns True if the case also meets the oracle at the bar (it always must match the simplest
    GPU variant bit for bit), None if the generated case is degenerate (nothing happens in it)."""
    import oracle
    from helpers.fuzz_cases import make_mode_case, SIMPLE_OPTIONS
    c = make_mode_case(seed)
    net, x0, opts, firings, mode = c["net"], c["x0"], c["options"], c["firings"], c["mode"]
    what = f"seed {seed} {mode} {opts}"
    if mode == "ensemble":
        t_end = INF
        if c["t_end_fraction"] is not None:
            t1 = oracle.run(net, x0, seed, 0, firings, INF, 0, check=False)["t"]
            t_end = t1 * c["t_end_fraction"] if t1 > 0 else 1.0
            if c["drop_firing_limit"]:
                firings = 0
        try:
            o = oracle.ensemble(net, x0, seed, c["traj_first"], c["n_traj"], firings, t_end, n_threads=4)
        except RuntimeError:
            return None                     # (a count overflow: covered by its own parity test)
        with rt.Model(net) as m:
            for k, v in opts:
                m.set_option(k, v)
            g = m.ensemble(x0, seed, c["traj_first"], c["n_traj"], firings, t_end, check=False)
        with rt.Model(net) as m:
            for k, v in (("ensemble_path", 2), ("pipeline", 0), ("bundle_ctas", 1)):
                m.set_option(k, v)
            h = m.ensemble(x0, seed, c["traj_first"], c["n_traj"], firings, t_end, check=False)
        _bitwise_common(g, h, what)
        return _at_the_bar(g, o)
    traj = c["trajectory"]
    plain = oracle.run(net, x0, seed, traj, firings, INF, 0, check=False)
    if plain["code"] != 0 or plain["t"] <= 0.0:
        return None
    duration = plain["t"]

    def configure(m, options):
        for k, v in options:
            m.set_option(k, v)
        if mode == "residual":
            m.set_option("formulation", 1)
        elif mode == "schedule":
            m.set_rate_schedule(tb, c["factor"], c["mask"])
        elif mode == "exponential":
            m.set_rate_exponent(lam)

    if mode == "schedule":
        tb = c["break_fractions"] * duration
        if len(np.unique(tb)) != len(tb):
            return None
        o = oracle.run_sched(net, x0, seed, traj, firings, INF, firings, t_break=tb, factor=c["factor"],
                             mask=c["mask"])
    elif mode == "exponential":
        lam = c["lambda_times_duration"] / duration
        o = oracle.run_rate_exp(net, x0, lam, seed, traj, firings, INF, firings)
    elif mode == "residual":
        o = oracle.run_residual(net, x0, seed, traj, firings, INF, firings)
    else:
        o = oracle.run(net, x0, seed, traj, firings, INF, firings, check=False)
    with rt.Model(net) as m:
        configure(m, opts)
        if mode in ("resume", "residual"):
            n1 = max(1, min(firings - 1, int(firings * c["split"])))
            a = m.run(x0, seed, traj, n1, INF, n1, want_state=True, check=False)
            b = m.run_resume(a["x"], a["t"], a["T"], a["P"], a["fire_count"], seed, traj, firings - n1, INF,
                             firings - n1, want_state=True, check=False)
            g = dict(x=b["x"], t=b["t"], firings=a["firings"] + b["firings"], stop=b["stop"],
                     trace_mu=np.concatenate([a["trace_mu"], b["trace_mu"]]),
                     trace_t=np.concatenate([a["trace_t"], b["trace_t"]]), fire_count=b["fire_count"])
        else:
            g = m.run(x0, seed, traj, firings, INF, firings, want_state=True, check=False)
    with rt.Model(net) as m:
        configure(m, SIMPLE_OPTIONS)
        h = m.run(x0, seed, traj, firings, INF, firings, want_state=True, check=False)     # (in one piece)
    _bitwise_common(g, h, what)
    return _at_the_bar(g, o)


@pytest.mark.parametrize("chunk", range(8))
def test_random_cases_of_the_other_modes(rt, chunk):
    """Ensembles (register, shared-memory and bundle kernels; firing and time limits), checkpoint /
    resume in both formulations, rate schedules and exponential rates on random networks and
    options: each case bit for bit against the simplest variant of the library run in one piece,
    and against the oracle at the bar.  The one-ulp differences between host and device log
    (module docstring) are not followed through resyncs here; during development 2 % of 10 000
    such cases left the bar because of them (each one bit-identical to the simplest variant),
    none for any other reason; of the 240 cases here one does.  A chunk of 30 may miss the bar in at
    most two cases."""
    results = [_mode_one(rt, seed) for seed in range(1 + chunk * 30, 1 + (chunk + 1) * 30)]
    ran = [x for x in results if x is not None]
    assert len(ran) >= 20
    assert sum(1 for x in ran if not x) <= 2, results
