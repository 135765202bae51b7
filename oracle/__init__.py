"""ctypes wrapper of the CPU oracle (TEST INFRASTRUCTURE, not product code).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2103_00405_b200 and shares nothing with it.
A network is passed as a plain dict of numpy arrays (the layout rt_workloads produces):
    n_species, n_reactions, react_ptr[i8, M+1], react_species[i4], react_sigma[i4],
    stoich_ptr[i8, M+1], stoich_species[i4], stoich_v[i4], rate[f8, M]
"""
import ctypes as C
import math

import numpy as np

from .build import build as _build

STOP_T_END, STOP_MAX_FIRINGS, STOP_ABSORBED = 1, 2, 3

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_exp_draw.restype = C.c_double
        _lib.oracle_exp_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
        _lib.oracle_binom.restype = C.c_int64
        _lib.oracle_binom.argtypes = [C.c_int64, C.c_int32]
        _lib.oracle_run.restype = C.c_int
        _lib.oracle_run_from.restype = C.c_int
        _lib.oracle_run_rate_exp.restype = C.c_int
        _lib.oracle_run_residual.restype = C.c_int
        _lib.oracle_run_sched.restype = C.c_int
        _lib.oracle_ensemble.restype = C.c_int
    return _lib


def _p(arr, ctype):
    return None if arr is None else arr.ctypes.data_as(C.POINTER(ctype))


def _net_args(net):
    keep = dict(
        react_ptr=np.ascontiguousarray(net["react_ptr"], dtype=np.int64),
        react_species=np.ascontiguousarray(net["react_species"], dtype=np.int32),
        react_sigma=np.ascontiguousarray(net["react_sigma"], dtype=np.int32),
        stoich_ptr=np.ascontiguousarray(net["stoich_ptr"], dtype=np.int64),
        stoich_species=np.ascontiguousarray(net["stoich_species"], dtype=np.int32),
        stoich_v=np.ascontiguousarray(net["stoich_v"], dtype=np.int32),
        rate=np.ascontiguousarray(net["rate"], dtype=np.float64),
    )
    args = [C.c_int32(int(net["n_species"])), C.c_int32(int(net["n_reactions"])),
            _p(keep["react_ptr"], C.c_int64), _p(keep["react_species"], C.c_int32),
            _p(keep["react_sigma"], C.c_int32), _p(keep["stoich_ptr"], C.c_int64),
            _p(keep["stoich_species"], C.c_int32), _p(keep["stoich_v"], C.c_int32),
            _p(keep["rate"], C.c_double)]
    return args, keep


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def exp_draw(seed, traj, k, n):
    return lib().oracle_exp_draw(seed, traj, k, n)


def binom(x, sigma):
    return lib().oracle_binom(x, sigma)


def propensities(net, X):
    args, keep = _net_args(net)
    X = np.ascontiguousarray(X, dtype=np.int64)
    a = np.zeros(int(net["n_reactions"]), dtype=np.float64)
    lib().oracle_propensities(args[0], args[1], args[2], args[3], args[4], args[8],
                              _p(X, C.c_int64), _p(a, C.c_double))
    return a


def run(net, x0, seed, trajectory=0, max_firings=0, t_end=math.inf, trace_cap=0,
        want_state=True, check=True):
    """One trajectory.  Returns a dict: x, t, firings, stop, fire_count, T, P, trace_mu, trace_t."""
    args, keep = _net_args(net)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    x0 = np.ascontiguousarray(x0, dtype=np.int64)
    assert x0.shape == (N,)
    x = np.zeros(N, dtype=np.int64)
    t = C.c_double(0.0)
    firings = C.c_uint64(0)
    stop = C.c_int32(0)
    fc = np.zeros(M, dtype=np.uint64) if want_state else None
    T = np.zeros(M, dtype=np.float64) if want_state else None
    P = np.zeros(M, dtype=np.float64) if want_state else None
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().oracle_run(*args, _p(x0, C.c_int64), C.c_uint64(seed), C.c_uint64(trajectory),
                          C.c_uint64(max_firings), C.c_double(t_end), _p(x, C.c_int64),
                          C.byref(t), C.byref(firings), C.byref(stop), _p(fc, C.c_uint64),
                          _p(T, C.c_double), _p(P, C.c_double), _p(tmu, C.c_int32),
                          _p(tt, C.c_double), C.c_uint64(trace_cap))
    if rc != 0 and check:
        raise RuntimeError(f"oracle_run failed with code {rc}")
    nrec = min(int(firings.value), trace_cap)
    return dict(x=x, t=t.value, firings=int(firings.value), stop=int(stop.value), code=rc,
                fire_count=fc, T=T, P=P,
                trace_mu=None if tmu is None else tmu[:nrec],
                trace_t=None if tt is None else tt[:nrec])


def run_from(net, x0, t0, T0, P0, n0, seed, trajectory=0, max_firings=0, t_end=math.inf,
             trace_cap=0, residual=False, check=True):
    """One trajectory resumed from a checkpoint: real time t0, internal times T0, next internal
    firing times P0, firings so far n0 (each array may be None = fresh).  residual=True: the
    residual (Table 3) form; P0 then holds the residuals R_k and the result's "P" returns them."""
    args, keep = _net_args(net)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    x0 = np.ascontiguousarray(x0, dtype=np.int64)
    T0 = None if T0 is None else np.ascontiguousarray(T0, dtype=np.float64)
    P0 = None if P0 is None else np.ascontiguousarray(P0, dtype=np.float64)
    n0 = None if n0 is None else np.ascontiguousarray(n0, dtype=np.uint64)
    x = np.zeros(N, dtype=np.int64)
    t = C.c_double(0.0)
    firings = C.c_uint64(0)
    stop = C.c_int32(0)
    fc = np.zeros(M, dtype=np.uint64)
    T = np.zeros(M, dtype=np.float64)
    P = np.zeros(M, dtype=np.float64)
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().oracle_run_from(*args, _p(x0, C.c_int64), C.c_double(t0), _p(T0, C.c_double),
                               _p(P0, C.c_double), _p(n0, C.c_uint64), C.c_int32(1 if residual else 0),
                               C.c_uint64(seed), C.c_uint64(trajectory), C.c_uint64(max_firings),
                               C.c_double(t_end), _p(x, C.c_int64), C.byref(t), C.byref(firings),
                               C.byref(stop), _p(fc, C.c_uint64), _p(T, C.c_double), _p(P, C.c_double),
                               _p(tmu, C.c_int32), _p(tt, C.c_double), C.c_uint64(trace_cap))
    if rc != 0 and check:
        raise RuntimeError(f"oracle_run_from failed with code {rc}")
    nrec = min(int(firings.value), trace_cap)
    return dict(x=x, t=t.value, firings=int(firings.value), stop=int(stop.value), code=rc,
                fire_count=fc, T=T, P=P, R=P if residual else None,
                trace_mu=None if tmu is None else tmu[:nrec],
                trace_t=None if tt is None else tt[:nrec])


def run_sched(net, x0, seed, trajectory=0, max_firings=0, t_end=math.inf, trace_cap=0,
              t_break=(), factor=(), mask=None):
    """One trajectory with piecewise-constant rate modulation (Eq.28): c_k(t) = c_k *
    factor[i] for t in [t_break[i], t_break[i+1]) for the channels with mask[k] != 0 (all if None)."""
    args, keep = _net_args(net)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    x0 = np.ascontiguousarray(x0, dtype=np.int64)
    tb = np.ascontiguousarray(t_break, dtype=np.float64)
    fa = np.ascontiguousarray(factor, dtype=np.float64)
    assert tb.shape == fa.shape
    mk = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    x = np.zeros(N, dtype=np.int64)
    t = C.c_double(0.0)
    firings = C.c_uint64(0)
    stop = C.c_int32(0)
    fc = np.zeros(M, dtype=np.uint64)
    T = np.zeros(M, dtype=np.float64)
    P = np.zeros(M, dtype=np.float64)
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().oracle_run_sched(*args, _p(x0, C.c_int64), C.c_uint64(seed), C.c_uint64(trajectory),
                                C.c_uint64(max_firings), C.c_double(t_end), C.c_int32(len(tb)),
                                _p(tb, C.c_double), _p(fa, C.c_double), _p(mk, C.c_uint8),
                                _p(x, C.c_int64), C.byref(t), C.byref(firings), C.byref(stop),
                                _p(fc, C.c_uint64), _p(T, C.c_double), _p(P, C.c_double),
                                _p(tmu, C.c_int32), _p(tt, C.c_double), C.c_uint64(trace_cap))
    if rc != 0:
        raise RuntimeError(f"oracle_run_sched failed with code {rc}")
    nrec = min(int(firings.value), trace_cap)
    return dict(x=x, t=t.value, firings=int(firings.value), stop=int(stop.value), fire_count=fc, T=T, P=P,
                trace_mu=None if tmu is None else tmu[:nrec],
                trace_t=None if tt is None else tt[:nrec])


def run_rate_exp(net, x0, lam, seed, trajectory=0, max_firings=0, t_end=math.inf, trace_cap=0):
    """One trajectory with smoothly time-dependent rates c_k(t) = c_k exp(lam[k] t) (PAPER.md
    Eq.28 solved per channel in closed form)."""
    args, keep = _net_args(net)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    x0 = np.ascontiguousarray(x0, dtype=np.int64)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    assert lam.shape == (M,)
    x = np.zeros(N, dtype=np.int64)
    t = C.c_double(0.0)
    firings = C.c_uint64(0)
    stop = C.c_int32(0)
    fc = np.zeros(M, dtype=np.uint64)
    T = np.zeros(M, dtype=np.float64)
    P = np.zeros(M, dtype=np.float64)
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().oracle_run_rate_exp(*args, _p(x0, C.c_int64), _p(lam, C.c_double), C.c_uint64(seed),
                                   C.c_uint64(trajectory), C.c_uint64(max_firings), C.c_double(t_end),
                                   _p(x, C.c_int64), C.byref(t), C.byref(firings), C.byref(stop),
                                   _p(fc, C.c_uint64), _p(T, C.c_double), _p(P, C.c_double),
                                   _p(tmu, C.c_int32), _p(tt, C.c_double), C.c_uint64(trace_cap))
    if rc != 0:
        raise RuntimeError(f"oracle_run_rate_exp failed with code {rc}")
    nrec = min(int(firings.value), trace_cap)
    return dict(x=x, t=t.value, firings=int(firings.value), stop=int(stop.value), fire_count=fc, T=T, P=P,
                trace_mu=None if tmu is None else tmu[:nrec],
                trace_t=None if tt is None else tt[:nrec])


def run_residual(net, x0, seed, trajectory=0, max_firings=0, t_end=math.inf, trace_cap=0):
    """One trajectory of the residual (Table 3) form.  Returns x, t, firings, stop, fire_count, R,
    trace_mu, trace_t."""
    args, keep = _net_args(net)
    N, M = int(net["n_species"]), int(net["n_reactions"])
    x0 = np.ascontiguousarray(x0, dtype=np.int64)
    x = np.zeros(N, dtype=np.int64)
    t = C.c_double(0.0)
    firings = C.c_uint64(0)
    stop = C.c_int32(0)
    fc = np.zeros(M, dtype=np.uint64)
    R = np.zeros(M, dtype=np.float64)
    tmu = np.zeros(trace_cap, dtype=np.int32) if trace_cap else None
    tt = np.zeros(trace_cap, dtype=np.float64) if trace_cap else None
    rc = lib().oracle_run_residual(*args, _p(x0, C.c_int64), C.c_uint64(seed), C.c_uint64(trajectory),
                                   C.c_uint64(max_firings), C.c_double(t_end), _p(x, C.c_int64),
                                   C.byref(t), C.byref(firings), C.byref(stop), _p(fc, C.c_uint64),
                                   _p(R, C.c_double), _p(tmu, C.c_int32), _p(tt, C.c_double),
                                   C.c_uint64(trace_cap))
    if rc != 0:
        raise RuntimeError(f"oracle_run_residual failed with code {rc}")
    nrec = min(int(firings.value), trace_cap)
    return dict(x=x, t=t.value, firings=int(firings.value), stop=int(stop.value), fire_count=fc, R=R,
                trace_mu=None if tmu is None else tmu[:nrec],
                trace_t=None if tt is None else tt[:nrec])


def ensemble(net, x0, seed, traj_first, n_traj, max_firings=0, t_end=math.inf, n_threads=1):
    """Independent trajectories traj_first..traj_first+n_traj-1.  Returns dict of arrays."""
    args, keep = _net_args(net)
    N = int(net["n_species"])
    x0 = np.ascontiguousarray(x0, dtype=np.int64)
    x = np.zeros((n_traj, N), dtype=np.int64)
    t = np.zeros(n_traj, dtype=np.float64)
    firings = np.zeros(n_traj, dtype=np.uint64)
    stop = np.zeros(n_traj, dtype=np.int32)
    rc = lib().oracle_ensemble(*args, _p(x0, C.c_int64), C.c_uint64(seed), C.c_uint64(traj_first),
                               C.c_uint64(n_traj), C.c_uint64(max_firings), C.c_double(t_end),
                               _p(x, C.c_int64), _p(t, C.c_double), _p(firings, C.c_uint64),
                               _p(stop, C.c_int32), C.c_int32(n_threads))
    if rc != 0:
        raise RuntimeError(f"oracle_ensemble failed with code {rc}")
    return dict(x=x, t=t, firings=firings, stop=stop)
