"""rt_run_dev_noalloc (include/rt.h): the bundle launch with its scratch -- T, P, a, n, X and the
argmin exchange slots -- in the library's static __device__ array instead of cudaMalloc'ed
buffers.  Checked against the existing path (rt_run_dev) on two calls in a row; integer outputs
bit for bit, times at the tolerance of tests/test_gpu_parity.py.  Collected last on purpose."""
import math

import numpy as np
import pytest

import rt_workloads as W

pytestmark = pytest.mark.gpu

RTOL_T = 1e-12


@pytest.fixture(scope="module")
def rt():
    import paper_2103_00405_b200 as rt
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    rt.lib()   # fails loudly if librt_b200.so is missing
    return rt


class _Bufs:
    def __init__(self, x0, cap):
        import torch
        dev = torch.device("cuda:0")
        self.x0 = torch.from_numpy(np.ascontiguousarray(x0, dtype=np.int64)).to(dev)
        self.x_out = torch.full((len(x0),), -1, dtype=torch.int64, device=dev)
        self.res = torch.zeros(3, dtype=torch.int64, device=dev)        # one rt_result
        self.mu = torch.full((cap,), -1, dtype=torch.int32, device=dev)
        self.t = torch.full((cap,), -1.0, dtype=torch.float64, device=dev)

    def host(self, rt):
        res = self.res.cpu().numpy().view(rt.RESULT_DTYPE)[0]
        return dict(x=self.x_out.cpu().numpy(), mu=self.mu.cpu().numpy(), tt=self.t.cpu().numpy(),
                    t=float(res["t"]), firings=int(res["firings"]), stop=int(res["stop"]),
                    status=int(res["status"]))


def _run(rt, m, fn, x0, seed, traj, firings):
    b = _Bufs(x0, firings)
    rc = fn(m.handle, b.x0, seed, traj, firings, math.inf, b.x_out, b.res, b.mu, b.t, firings)
    assert rc == rt.RT_OK, rt.rt_strerror(rc)
    assert rt.rt_sync(m.handle) == rt.RT_OK
    return b.host(rt)


def _same(got, want):
    assert got["firings"] == want["firings"] and got["stop"] == want["stop"]
    assert got["status"] == want["status"] == 0
    np.testing.assert_array_equal(got["mu"], want["mu"])
    np.testing.assert_array_equal(got["x"], want["x"])
    np.testing.assert_allclose(got["tt"], want["tt"], rtol=RTOL_T, atol=0)
    assert math.isclose(got["t"], want["t"], rel_tol=RTOL_T, abs_tol=0)


CASES = [
    ("cfg3", 1.0, 2000, ()),                        # config 3 at full size: candidate-first kernel
    ("cfg3", 0.0517, 1500, (("pipeline", 0),)),     # plain bundle kernel, ragged M
    ("cfg3", 0.0517, 1500, (("state_mode", 1),)),   # (T, P, a) LIVE in the scratch, streamed every firing
    ("cfg3", 0.02, 1500, (("exchange", 1), ("bundle_ctas", 7))),   # exchange through the slots in L2
    ("cfg1", 1.0, 500, ()),                         # M = 2: one CTA
]


@pytest.mark.parametrize("name,scale,firings,options", CASES)
def test_noalloc_matches_the_existing_path_on_two_calls_in_a_row(rt, name, scale, firings, options):
    import torch
    net, x0, par = W.make_config(name, scale=scale)
    seed = par["seed"]
    # existing path: scratch in buffers the model allocates
    with rt.Model(net) as m:
        for k, v in options:
            m.set_option(k, v)
        want = [_run(rt, m, rt.rt_run_dev, x0, seed, traj, firings) for traj in (0, 1)]
        shape = [m.info(k) for k in ("bundle_ctas", "state_in_smem", "cluster_exchange", "pipeline")]
    assert want[0]["firings"] == firings
    assert not np.array_equal(want[0]["mu"], want[1]["mu"])      # (the two calls differ)
    # new entry point: a fresh model that never allocated that scratch
    with rt.Model(net) as m:
        for k, v in options:
            m.set_option(k, v)
        rc, need = rt.rt_noalloc_prepare(m.handle)
        assert rc == rt.RT_OK and 0 < need <= rt.RT_NOALLOC_SCRATCH_BYTES
        _same(_run(rt, m, rt.rt_run_dev_noalloc, x0, seed, 0, firings), want[0])   # (also loads everything)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        bufs = [_Bufs(x0, firings) for _ in (0, 1)]          # the caller's inputs and outputs
        free1 = torch.cuda.mem_get_info()[0]
        # two calls in a row, different trajectories, stream order, no sync in between: the second
        # starts from whatever the first left in the shared array
        for traj, b in zip((0, 1), bufs):
            rc = rt.rt_run_dev_noalloc(m.handle, b.x0, seed, traj, firings, math.inf, b.x_out, b.res,
                                       b.mu, b.t, firings)
            assert rc == rt.RT_OK, rt.rt_strerror(rc)
        assert rt.rt_sync(m.handle) == rt.RT_OK
        free2 = torch.cuda.mem_get_info()[0]
        for b, w in zip(bufs, want):
            _same(b.host(rt), w)
        assert [m.info(k) for k in ("bundle_ctas", "state_in_smem", "cluster_exchange", "pipeline")] == shape
        assert free2 == free1, f"device memory changed across the calls: {free1 - free2} bytes ({free0})"


def test_noalloc_rejects_what_does_not_fit_and_unprepared_models(rt):
    net, x0, par = W.make_config("cfg3", scale=2.0)        # 2e5 reactions: 5.6 MB of (T, P, a, n)
    with rt.Model(net) as m:
        b = _Bufs(x0, 4)
        args = (m.handle, b.x0, par["seed"], 0, 4, math.inf, b.x_out, b.res, b.mu, b.t, 4)
        assert rt.rt_run_dev_noalloc(*args) == rt.RT_ERR_SCRATCH           # not prepared
        rc, need = rt.rt_noalloc_prepare(m.handle)
        assert rc == rt.RT_ERR_SCRATCH and need > rt.RT_NOALLOC_SCRATCH_BYTES
        assert need >= 28 * net["n_reactions"] + 8 * net["n_species"]
        assert rt.rt_run_dev_noalloc(*args) == rt.RT_ERR_SCRATCH           # too large
        assert "RT_NOALLOC_SCRATCH_BYTES" in rt.rt_strerror(rt.RT_ERR_SCRATCH)
        assert m.info("kernel_launches") == 0
        assert rt.rt_sync(m.handle) == rt.RT_OK
        assert int(b.res.cpu().numpy().view(rt.RESULT_DTYPE)[0]["firings"]) == 0     # nothing ran
        # the existing path is unaffected
        assert rt.rt_run_dev(*args) == rt.RT_OK and rt.rt_sync(m.handle) == rt.RT_OK
        assert int(b.res.cpu().numpy().view(rt.RESULT_DTYPE)[0]["firings"]) == 4
