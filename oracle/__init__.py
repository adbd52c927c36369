"""ctypes loader for the serial fp64 CPU oracle (oracle/imrt_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package paper_0908_4421_b200 never imports
this module, and this module never imports the product package.

Every function here only marshals numpy arrays into the C functions; the arithmetic, with its
citations of PAPER.md, lives in imrt_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "imrt_oracle.c")
_LIB = os.path.join(_HERE, "libimrt_oracle.so")

STOP_MAX_ITERS, STOP_TOLERANCE, STOP_STATIONARY, STOP_LS_STALLED = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc.  -O2 without -ffast-math: summation order stays as written."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_P = ctypes.c_void_p


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_eval.argtypes = [ctypes.c_int64] + [_P] * 12
        lib.oracle_eval.restype = None
        lib.oracle_eval_v.argtypes = [ctypes.c_int64] + [_P] * 14
        lib.oracle_eval_v.restype = None
        lib.oracle_grad.argtypes = [ctypes.c_int64, ctypes.c_int64] + [_P] * 5
        lib.oracle_grad.restype = None
        lib.oracle_trial_point.argtypes = [ctypes.c_int64, _P, _P, ctypes.c_double, _P, _P]
        lib.oracle_trial_point.restype = None
        lib.oracle_run.argtypes = ([ctypes.c_int64, ctypes.c_int64] + [_P] * 8 +
                                   [ctypes.c_double] * 4 + [ctypes.c_int, ctypes.c_int] +
                                   [_P, ctypes.c_double] + [_P] * 11)
        lib.oracle_run.restype = ctypes.c_int
        lib.oracle_run_v.argtypes = ([ctypes.c_int64, ctypes.c_int64] + [_P] * 10 +
                                     [ctypes.c_double] * 4 + [ctypes.c_int, ctypes.c_int] +
                                     [_P, ctypes.c_double] + [_P] * 11)
        lib.oracle_run_v.restype = ctypes.c_int
        lib.oracle_dvh.argtypes = [ctypes.c_int64, _P, _P, ctypes.c_int, _P, ctypes.c_int, _P, _P]
        lib.oracle_dvh.restype = None
        lib.oracle_merge_rows_count.argtypes = [ctypes.c_int64, ctypes.c_int64, _P, _P, _P, ctypes.c_int64, _P]
        lib.oracle_merge_rows_count.restype = None
        lib.oracle_merge_rows_fill.argtypes = [ctypes.c_int64, ctypes.c_int64, _P, _P, _P, _P, ctypes.c_int64, _P, _P, _P]
        lib.oracle_merge_rows_fill.restype = None
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_P)


def _c(a, dt):
    a = np.ascontiguousarray(a, dtype=dt)
    return a


def _csr(prob):
    return (_c(prob.row_ptr, np.int32), _c(prob.col, np.int32), _c(prob.val, np.float32), _c(prob.sid, np.uint8),
            _c(prob.t_under, np.float32), _c(prob.t_over, np.float32), _c(prob.w_under, np.float32),
            _c(prob.w_over, np.float32))


def _voxel_limits(prob):
    """Optional per-voxel limits of a problem (attributes tv_under / tv_over, float32 [n_v]) or (None, None)."""
    tvu, tvo = getattr(prob, "tv_under", None), getattr(prob, "tv_over", None)
    return (None if tvu is None else _c(tvu, np.float32)), (None if tvo is None else _c(tvo, np.float32))


def eval_objective(prob, x):
    """(d, r, G) at x.  imrt_oracle.c: oracle_eval."""
    lib = _load()
    rp, col, val, sid, tu, to, wu, wo = _csr(prob)
    x = _c(x, np.float64)
    d = np.empty(prob.n_v, np.float64)
    r = np.empty(prob.n_v, np.float64)
    G = ctypes.c_double(0.0)
    tvu, tvo = _voxel_limits(prob)
    lib.oracle_eval_v(prob.n_v, _p(rp), _p(col), _p(val), _p(sid), _p(tu), _p(to), _p(wu), _p(wo), _p(tvu), _p(tvo),
                      _p(x), _p(d), _p(r), ctypes.addressof(G))
    return d, r, G.value


def gradient(prob, r):
    """g = D^T r by scatter.  imrt_oracle.c: oracle_grad."""
    lib = _load()
    rp, col, val = _c(prob.row_ptr, np.int32), _c(prob.col, np.int32), _c(prob.val, np.float32)
    r = _c(r, np.float64)
    g = np.empty(prob.n_b, np.float64)
    lib.oracle_grad(prob.n_v, prob.n_b, _p(rp), _p(col), _p(val), _p(r), _p(g))
    return g


def trial_point(x, g, lam):
    """(x+, Delta) with x+ = max(0, x - lam g).  imrt_oracle.c: oracle_trial_point."""
    lib = _load()
    x = _c(x, np.float64)
    g = _c(g, np.float64)
    xn = np.empty_like(x)
    delta = ctypes.c_double(0.0)
    lib.oracle_trial_point(x.shape[0], _p(x), _p(g), float(lam), _p(xn), ctypes.addressof(delta))
    return xn, delta.value


@dataclass
class RunResult:
    n_iters: int
    stop_reason: int
    x: np.ndarray          # float64 [n_b]
    obj: np.ndarray        # float64 [n_iters+1]
    lam: np.ndarray        # float64 [n_iters]
    n_trials: np.ndarray   # int32 [n_iters]
    step_sq: np.ndarray    # float64 [n_iters]
    margin: np.ndarray     # float64 [n_iters]  (C - G+)/G_k of the accepted trial
    n_follow_violations: int
    first_violation: int
    fwd_passes: int
    tr_passes: int


def run(prob, x0=None, n_iters=None, delta=None, follow_trials=None, tau_rel=1e-6,
        eps=None, alpha=None, lambda0=None, max_ls=None) -> RunResult:
    """The Main Iterative Loop.  delta <= 0 or None-with-prob.delta==0 => fixed count."""
    lib = _load()
    rp, col, val, sid, tu, to, wu, wo = _csr(prob)
    n = int(prob.n_iters if n_iters is None else n_iters)
    dl = float(prob.delta if delta is None else delta)
    x = _c(prob.x0 if x0 is None else x0, np.float64).copy()
    obj = np.zeros(n + 1, np.float64)
    lam = np.zeros(max(n, 1), np.float64)
    ntr = np.zeros(max(n, 1), np.int32)
    ssq = np.zeros(max(n, 1), np.float64)
    mar = np.zeros(max(n, 1), np.float64)
    ft = None
    if follow_trials is not None:
        ft = _c(follow_trials, np.int32)
        assert ft.shape[0] >= n
    stop = ctypes.c_int(0)
    viol = ctypes.c_int(0)
    first = ctypes.c_int(-1)
    fwd = ctypes.c_int64(0)
    tr = ctypes.c_int64(0)
    tvu, tvo = _voxel_limits(prob)
    k = lib.oracle_run_v(prob.n_v, prob.n_b, _p(rp), _p(col), _p(val), _p(sid), _p(tu), _p(to), _p(wu), _p(wo), _p(tvu), _p(tvo),
                       float(prob.eps if eps is None else eps), float(prob.alpha if alpha is None else alpha),
                       float(prob.lambda0 if lambda0 is None else lambda0), dl,
                       int(prob.max_ls if max_ls is None else max_ls), n,
                       _p(ft), float(tau_rel),
                       _p(x), _p(obj), _p(lam), _p(ntr), _p(ssq), _p(mar),
                       ctypes.addressof(stop), ctypes.addressof(viol), ctypes.addressof(first),
                       ctypes.addressof(fwd), ctypes.addressof(tr))
    return RunResult(k, stop.value, x, obj[:k + 1].copy(), lam[:k].copy(), ntr[:k].copy(), ssq[:k].copy(),
                     mar[:k].copy(), viol.value, first.value, fwd.value, tr.value)


DVH_PCTS = (2.0, 5.0, 50.0, 95.0, 98.0)


def dvh_points(sid, d, n_structures, pcts=DVH_PCTS):
    """(D_p [n_s, n_p], mean [n_s]).  imrt_oracle.c: oracle_dvh."""
    lib = _load()
    sid = _c(sid, np.uint8)
    d = _c(d, np.float64)
    pc = _c(pcts, np.float64)
    out = np.empty((n_structures, pc.shape[0]), np.float64)
    mean = np.empty(n_structures, np.float64)
    lib.oracle_dvh(sid.shape[0], _p(sid), _p(d), n_structures, _p(pc), pc.shape[0], _p(out), _p(mean))
    return out, mean


def merge_rows(n_b, row_ptr, col, val, group, n_groups):
    """Rows with the same group id replaced by their mean (reading R17): (row_ptr, col, val) of the merged
    matrix, one row per group.  imrt_oracle.c: oracle_merge_rows_count / oracle_merge_rows_fill."""
    lib = _load()
    rp, c, v, g = _c(row_ptr, np.int32), _c(col, np.int32), _c(val, np.float32), _c(group, np.int32)
    n_v = rp.shape[0] - 1
    out_rp = np.zeros(n_groups + 1, np.int32)
    lib.oracle_merge_rows_count(n_v, n_b, _p(rp), _p(c), _p(g), n_groups, _p(out_rp))
    out_c = np.zeros(max(int(out_rp[-1]), 1), np.int32)
    out_v = np.zeros(max(int(out_rp[-1]), 1), np.float32)
    lib.oracle_merge_rows_fill(n_v, n_b, _p(rp), _p(c), _p(v), _p(g), n_groups, _p(out_rp), _p(out_c), _p(out_v))
    return out_rp, out_c[:out_rp[-1]], out_v[:out_rp[-1]]
