"""ctypes binding of include/rt.h -- argument marshalling only.

Function names and argument order follow the C header.  Host-pointer entry points take numpy
arrays; the *_dev entry points take torch CUDA tensors (PyTorch is used for device memory and
streams only) and enqueue on torch's current stream.
"""
import ctypes as C
import math
import os

import numpy as np

RT_OK = 0
RT_ERR_NULL, RT_ERR_BAD_NETWORK, RT_ERR_BAD_ARG, RT_ERR_UNSUPPORTED = -1, -2, -3, -4
RT_ERR_OVERFLOW, RT_ERR_CUDA, RT_ERR_OOM = -5, -6, -7
RT_ERR_SCRATCH = -8
RT_NOALLOC_SCRATCH_BYTES = 4 << 20
RT_STOP_T_END, RT_STOP_MAX_FIRINGS, RT_STOP_ABSORBED = 1, 2, 3

# rt_result: (f64 t, u64 firings, i32 stop, i32 status), 24 bytes
RESULT_DTYPE = np.dtype([("t", "<f8"), ("firings", "<u8"), ("stop", "<i4"), ("status", "<i4")])

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "librt_b200.so")
_lib = None


class RtError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {rt_strerror(code)} ({code})")


class _Network(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32),
                ("react_ptr", C.c_void_p), ("react_species", C.c_void_p), ("react_sigma", C.c_void_p),
                ("stoich_ptr", C.c_void_p), ("stoich_species", C.c_void_p), ("stoich_v", C.c_void_p),
                ("rate", C.c_void_p)]


def library_path():
    return _LIB_PATH


def lib():
    """Load librt_b200.so (built by `python -m paper_2103_00405_b200.build`); no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build the CUDA extension with "
            "`python -m paper_2103_00405_b200.build` (there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp, u64, i64, f64, i32 = C.c_void_p, C.c_uint64, C.c_int64, C.c_double, C.c_int
    L.rt_validate_network.argtypes = [C.POINTER(_Network)]
    L.rt_create.argtypes = [C.POINTER(_Network), i32, C.POINTER(vp)]
    L.rt_run.argtypes = [vp, vp, u64, u64, u64, f64, vp, vp, vp, vp, vp, vp, vp, u64]
    L.rt_run_resume.argtypes = [vp, vp, f64, vp, vp, vp, u64, u64, u64, f64, vp, vp, vp, vp, vp, vp, vp, u64]
    L.rt_run_dev.argtypes = [vp, vp, u64, u64, u64, f64, vp, vp, vp, vp, u64, vp]
    L.rt_run_dev_noalloc.argtypes = [vp, vp, u64, u64, u64, f64, vp, vp, vp, vp, u64, vp]
    L.rt_noalloc_prepare.argtypes = [vp, C.POINTER(u64)]
    L.rt_ensemble.argtypes = [vp, vp, u64, u64, u64, u64, f64, vp, vp]
    L.rt_ensemble_dev.argtypes = [vp, vp, u64, u64, u64, u64, f64, vp, vp, vp]
    L.rt_sync.argtypes = [vp, vp]
    L.rt_set_rate_schedule.argtypes = [vp, C.c_int32, vp, vp, vp]
    L.rt_set_rate_exponent.argtypes = [vp, vp]
    L.rt_set_option.argtypes = [vp, C.c_char_p, i64]
    L.rt_get_info.argtypes = [vp, C.c_char_p, C.POINTER(i64)]
    L.rt_destroy.argtypes = [vp]
    L.rt_destroy.restype = None
    L.rt_strerror.argtypes = [i32]
    L.rt_strerror.restype = C.c_char_p
    for name in ("rt_validate_network", "rt_create", "rt_run", "rt_run_resume", "rt_run_dev", "rt_ensemble", "rt_set_rate_schedule",
                 "rt_set_rate_exponent", "rt_run_dev_noalloc", "rt_noalloc_prepare",
                 "rt_ensemble_dev", "rt_sync", "rt_set_option", "rt_get_info"):
        getattr(L, name).restype = i32
    _lib = L
    return L


def _np(arr, dtype):
    return np.ascontiguousarray(arr, dtype=dtype)


def _ptr(arr):
    return None if arr is None else C.c_void_p(arr.ctypes.data)


def _pack_network(net):
    keep = [_np(net["react_ptr"], np.int64), _np(net["react_species"], np.int32),
            _np(net["react_sigma"], np.int32), _np(net["stoich_ptr"], np.int64),
            _np(net["stoich_species"], np.int32), _np(net["stoich_v"], np.int32),
            _np(net["rate"], np.float64)]
    s = _Network(int(net["n_species"]), int(net["n_reactions"]), *[a.ctypes.data for a in keep])
    return s, keep


def rt_strerror(code):
    return lib().rt_strerror(int(code)).decode()


def rt_validate_network(net):
    s, keep = _pack_network(net)
    return lib().rt_validate_network(C.byref(s))


def rt_create(net, device=0):
    """Returns (code, handle).  handle is an opaque pointer (int) or None."""
    s, keep = _pack_network(net)
    h = C.c_void_p()
    rc = lib().rt_create(C.byref(s), int(device), C.byref(h))
    return rc, (h.value if rc == RT_OK else None)


def rt_destroy(handle):
    if handle:
        lib().rt_destroy(C.c_void_p(handle))


def rt_set_rate_schedule(handle, t_break, factor, mask=None):
    """Piecewise-constant rate modulation (include/rt.h); empty t_break removes it."""
    tb = _np(t_break, np.float64)
    fa = _np(factor, np.float64)
    if tb.shape != fa.shape or tb.ndim != 1:
        return RT_ERR_BAD_ARG
    mk = None if mask is None else _np(mask, np.uint8)
    return lib().rt_set_rate_schedule(C.c_void_p(handle), int(tb.size), _ptr(tb) if tb.size else None,
                                      _ptr(fa) if fa.size else None, _ptr(mk))


def rt_set_rate_exponent(handle, lam, n_reactions):
    """c_k(t) = c_k exp(lam[k] t) (include/rt.h); lam = None removes it."""
    if lam is None:
        return lib().rt_set_rate_exponent(C.c_void_p(handle), None)
    lam = _np(lam, np.float64)
    if lam.shape != (n_reactions,):
        return RT_ERR_BAD_ARG
    return lib().rt_set_rate_exponent(C.c_void_p(handle), _ptr(lam))


def rt_set_option(handle, name, value):
    return lib().rt_set_option(C.c_void_p(handle), name.encode(), int(value))


def rt_get_info(handle, name):
    v = C.c_int64(0)
    rc = lib().rt_get_info(C.c_void_p(handle), name.encode(), C.byref(v))
    if rc != RT_OK:
        raise RtError(rc, f"rt_get_info({name})")
    return v.value


def rt_run(handle, x0, seed, trajectory, max_firings, t_end, n_species, n_reactions,
           trace_cap=0, want_state=False):
    """Host-pointer rt_run.  Returns (code, dict).  The dict mirrors the C outputs."""
    x0 = _np(x0, np.int64)
    x_out = np.zeros(n_species, dtype=np.int64)
    res = np.zeros(1, dtype=RESULT_DTYPE)
    fc = np.zeros(n_reactions, dtype=np.uint64) if want_state else None
    T = np.zeros(n_reactions, dtype=np.float64) if want_state else None
    P = np.zeros(n_reactions, dtype=np.float64) if want_state else None
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().rt_run(C.c_void_p(handle), _ptr(x0), int(seed), int(trajectory), int(max_firings),
                      float(t_end), _ptr(x_out), _ptr(res), _ptr(fc), _ptr(T), _ptr(P),
                      _ptr(tmu), _ptr(tt), int(trace_cap))
    nrec = min(int(res["firings"][0]), trace_cap)
    out = dict(x=x_out, t=float(res["t"][0]), firings=int(res["firings"][0]),
               stop=int(res["stop"][0]), status=int(res["status"][0]), fire_count=fc, T=T, P=P,
               trace_mu=None if tmu is None else tmu[:nrec],
               trace_t=None if tt is None else tt[:nrec])
    return rc, out


def rt_run_resume(handle, x0, t0, T0, P0, fire_count0, seed, trajectory, max_firings, t_end,
                  n_species, n_reactions, trace_cap=0, want_state=False):
    """Host-pointer rt_run_resume.  Returns (code, dict) like rt_run."""
    x0 = _np(x0, np.int64)
    T0 = None if T0 is None else _np(T0, np.float64)
    P0 = None if P0 is None else _np(P0, np.float64)
    n0 = None if fire_count0 is None else _np(fire_count0, np.uint64)
    x_out = np.zeros(n_species, dtype=np.int64)
    res = np.zeros(1, dtype=RESULT_DTYPE)
    fc = np.zeros(n_reactions, dtype=np.uint64) if want_state else None
    T = np.zeros(n_reactions, dtype=np.float64) if want_state else None
    P = np.zeros(n_reactions, dtype=np.float64) if want_state else None
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().rt_run_resume(C.c_void_p(handle), _ptr(x0), float(t0), _ptr(T0), _ptr(P0), _ptr(n0),
                             int(seed), int(trajectory), int(max_firings), float(t_end),
                             _ptr(x_out), _ptr(res), _ptr(fc), _ptr(T), _ptr(P), _ptr(tmu), _ptr(tt),
                             int(trace_cap))
    nrec = min(int(res["firings"][0]), trace_cap)
    out = dict(x=x_out, t=float(res["t"][0]), firings=int(res["firings"][0]),
               stop=int(res["stop"][0]), status=int(res["status"][0]), fire_count=fc, T=T, P=P,
               trace_mu=None if tmu is None else tmu[:nrec],
               trace_t=None if tt is None else tt[:nrec])
    return rc, out


def rt_ensemble(handle, x0, seed, traj_first, n_traj, max_firings, t_end, n_species, want_x=True):
    """Host-pointer rt_ensemble.  Returns (code, dict(x[n_traj,N], t, firings, stop, status))."""
    x0 = _np(x0, np.int64)
    x_out = np.zeros((n_traj, n_species), dtype=np.int64) if want_x else None
    res = np.zeros(n_traj, dtype=RESULT_DTYPE)
    rc = lib().rt_ensemble(C.c_void_p(handle), _ptr(x0), int(seed), int(traj_first), int(n_traj),
                           int(max_firings), float(t_end), _ptr(x_out), _ptr(res))
    return rc, dict(x=x_out, t=res["t"].copy(), firings=res["firings"].copy(),
                    stop=res["stop"].copy(), status=res["status"].copy())


def _dev_ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def rt_run_dev(handle, x0_dev, seed, trajectory, max_firings, t_end, x_out_dev, res_dev,
               trace_mu_dev=None, trace_t_dev=None, trace_cap=0):
    """Device-pointer rt_run on torch's current stream; tensors are torch CUDA tensors
    (x0/x_out int64 [N], res uint8 [24] or int64 [3], trace_mu int32, trace_t float64)."""
    return lib().rt_run_dev(C.c_void_p(handle), _dev_ptr(x0_dev), int(seed), int(trajectory),
                            int(max_firings), float(t_end), _dev_ptr(x_out_dev), _dev_ptr(res_dev),
                            _dev_ptr(trace_mu_dev), _dev_ptr(trace_t_dev), int(trace_cap),
                            _stream_ptr())


def rt_noalloc_prepare(handle):
    """Set-up for rt_run_dev_noalloc (may allocate).  Returns (rc, scratch bytes the options need)."""
    need = C.c_uint64(0)
    rc = lib().rt_noalloc_prepare(C.c_void_p(handle), C.byref(need))
    return rc, int(need.value)


def rt_run_dev_noalloc(handle, x0_dev, seed, trajectory, max_firings, t_end, x_out_dev, res_dev,
                       trace_mu_dev=None, trace_t_dev=None, trace_cap=0):
    """rt_run_dev with its scratch in the library's static device array: no allocation in the call."""
    return lib().rt_run_dev_noalloc(C.c_void_p(handle), _dev_ptr(x0_dev), int(seed), int(trajectory),
                                    int(max_firings), float(t_end), _dev_ptr(x_out_dev), _dev_ptr(res_dev),
                                    _dev_ptr(trace_mu_dev), _dev_ptr(trace_t_dev), int(trace_cap),
                                    _stream_ptr())


def rt_ensemble_dev(handle, x0_dev, seed, traj_first, n_traj, max_firings, t_end, x_out_dev, res_dev):
    return lib().rt_ensemble_dev(C.c_void_p(handle), _dev_ptr(x0_dev), int(seed), int(traj_first),
                                 int(n_traj), int(max_firings), float(t_end), _dev_ptr(x_out_dev),
                                 _dev_ptr(res_dev), _stream_ptr())


def rt_sync(handle):
    return lib().rt_sync(C.c_void_p(handle), _stream_ptr())


class Model:
    """Small convenience wrapper: owns the handle, raises RtError on failure."""

    def __init__(self, net, device=0):
        self.n_species = int(net["n_species"])
        self.n_reactions = int(net["n_reactions"])
        rc, self.handle = rt_create(net, device)
        if rc != RT_OK:
            raise RtError(rc, "rt_create")

    def close(self):
        if self.handle:
            rt_destroy(self.handle)
            self.handle = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_option(self, name, value):
        rc = rt_set_option(self.handle, name, value)
        if rc != RT_OK:
            raise RtError(rc, f"rt_set_option({name})")

    def set_rate_schedule(self, t_break, factor, mask=None):
        rc = rt_set_rate_schedule(self.handle, t_break, factor, mask)
        if rc != RT_OK:
            raise RtError(rc, "rt_set_rate_schedule")

    def set_rate_exponent(self, lam):
        rc = rt_set_rate_exponent(self.handle, lam, self.n_reactions)
        if rc != RT_OK:
            raise RtError(rc, "rt_set_rate_exponent")

    def info(self, name):
        return rt_get_info(self.handle, name)

    def run(self, x0, seed, trajectory=0, max_firings=0, t_end=math.inf, trace_cap=0,
            want_state=False, check=True):
        rc, out = rt_run(self.handle, x0, seed, trajectory, max_firings, t_end, self.n_species,
                         self.n_reactions, trace_cap, want_state)
        if check and rc != RT_OK:
            raise RtError(rc, "rt_run")
        out["code"] = rc
        return out

    def run_resume(self, x0, t0, T0, P0, fire_count0, seed, trajectory=0, max_firings=0,
                   t_end=math.inf, trace_cap=0, want_state=False, check=True):
        rc, out = rt_run_resume(self.handle, x0, t0, T0, P0, fire_count0, seed, trajectory,
                                max_firings, t_end, self.n_species, self.n_reactions, trace_cap,
                                want_state)
        if check and rc != RT_OK:
            raise RtError(rc, "rt_run_resume")
        out["code"] = rc
        return out

    def ensemble(self, x0, seed, traj_first, n_traj, max_firings=0, t_end=math.inf, want_x=True,
                 check=True):
        rc, out = rt_ensemble(self.handle, x0, seed, traj_first, n_traj, max_firings, t_end,
                              self.n_species, want_x)
        if check and rc != RT_OK:
            raise RtError(rc, "rt_ensemble")
        out["code"] = rc
        return out
