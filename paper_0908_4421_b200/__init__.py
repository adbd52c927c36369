"""paper_0908_4421_b200 -- Python binding of libimrtgp (include/imrtgp.h).

Argument marshalling only: every step of the optimiser (dose SpMV, penalty / residual / objective reduction,
transpose SpMV, projection, Armijo line search, stop test -- PAPER.md:51-114) runs in the CUDA kernels of
csrc/.  PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: if the shared
library cannot be loaded, importing the binding's functions raises.

Module-level functions carry the C names (imrt_plan_create, imrt_plan_run_iters, ...) and take torch CUDA
tensors where the C-ABI takes device pointers; `Plan` is a small convenience wrapper around them.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build
from . import sharded  # noqa: E402,F401  (row-sharded set-up: slab selection, inboxes)

__all__ = ["Plan", "ImrtError", "lib", "Params", "Options", "STATUS_NAMES", "STOP_NAMES", "EXPORTS"]

STATUS_NAMES = ("OK", "INVALID_ARG", "BAD_CSR", "BAD_STRUCTURE", "WORKSPACE_TOO_SMALL", "CUDA_ERROR",
                "UNSUPPORTED_DEVICE", "UNSUPPORTED", "BAD_X", "NOT_READY")
STOP_NAMES = ("MAX_ITERS", "TOLERANCE", "STATIONARY", "LINESEARCH_STALLED", "TRACE_FULL", "PEER_TIMEOUT")
DRIVER_GRAPH, DRIVER_HOST, DRIVER_PERSISTENT = 0, 1, 2

# every symbol include/imrtgp.h declares
EXPORTS = ("imrt_workspace_bytes", "imrt_plan_create", "imrt_plan_set_x", "imrt_plan_set_voxel_limits", "imrt_plan_run_iters", "imrt_plan_run_to_tol",
           "imrt_plan_eval", "imrt_plan_eval_batch", "imrt_plan_gradient", "imrt_trial_point", "imrt_armijo_accepts", "imrt_stop_test", "imrt_plan_get_x", "imrt_plan_get_dose", "imrt_plan_dvh", "imrt_plan_get_trace",
           "imrt_plan_get_counters", "imrt_plan_get_info", "imrt_plan_launch_pass", "imrt_plan_get_pass_timing", "imrt_plan_get_tuning", "imrt_plan_get_create_times",
           "imrt_shard_inbox_bytes", "imrt_plan_set_shard", "imrt_plan_run_ranks",
           "imrt_merge_rows_workspace_bytes", "imrt_merge_rows_count", "imrt_merge_rows_fill", "imrt_dvh_static", "imrt_last_error", "imrt_plan_destroy",
           "imrt_version")


class ImrtError(RuntimeError):
    def __init__(self, status: int, message: str):
        self.status = status
        self.status_name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        super().__init__("libimrtgp: %s: %s" % (self.status_name, message))


class Params(ctypes.Structure):
    """imrt_params."""
    _fields_ = [("eps", ctypes.c_double), ("alpha", ctypes.c_double), ("lambda0", ctypes.c_double),
                ("max_ls", ctypes.c_int32), ("max_iters", ctypes.c_int32), ("driver", ctypes.c_int32),
                ("ls_batch", ctypes.c_int32)]


class Options(ctypes.Structure):
    """imrt_options: layout / tuning switches of imrt_plan_create (all 0 = defaults)."""
    _fields_ = [("tune_level", ctypes.c_int32), ("dose_format", ctypes.c_int32), ("col_bits", ctypes.c_int32),
                ("transpose_format", ctypes.c_int32), ("quad_cap", ctypes.c_int32), ("n_ctas", ctypes.c_int32),
                ("profile_create", ctypes.c_int32), ("spin_timeout_ms", ctypes.c_int32),
                ("host_tuning", ctypes.c_void_p), ("host_tuning_bytes", ctypes.c_size_t)]


CREATE_PHASES = ("validate", "quad_unions", "record_layout", "pack_records", "transpose_sort", "pack_transpose", "state",
                 "tune_dose", "tune_transpose", "graph")

_lib = None
_P = ctypes.c_void_p


def lib() -> ctypes.CDLL:
    """Load libimrtgp.so (building it in-tree first if it is missing or older than its sources)."""
    global _lib
    if _lib is None:
        try:
            path = _build.build()
        except Exception as exc:  # no nvcc and no prebuilt library: there is nothing to fall back to
            if not os.path.exists(_build.LIB):
                raise ImportError("libimrtgp.so is not built and could not be built (%s); run "
                                  "`python -m paper_0908_4421_b200.build` where nvcc is available" % exc) from exc
            path = _build.LIB
        L = ctypes.CDLL(path)
        i64, i32, dbl = ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        L.imrt_workspace_bytes.argtypes = [i64, i64, i64, i32, i32, ctypes.POINTER(ctypes.c_size_t)]
        L.imrt_plan_create.argtypes = [ctypes.POINTER(_P), i64, i64, i64, _P, _P, _P, _P, i32, _P, _P, _P, _P,
                                       ctypes.POINTER(Params), ctypes.POINTER(Options), _P, ctypes.c_size_t, _P]
        L.imrt_plan_set_x.argtypes = [_P, _P]
        L.imrt_plan_set_voxel_limits.argtypes = [_P, _P, _P]
        L.imrt_plan_run_iters.argtypes = [_P, i32]
        L.imrt_plan_run_to_tol.argtypes = [_P, dbl, i32]
        L.imrt_plan_eval.argtypes = [_P, _P, _P, _P, _P, ctypes.POINTER(dbl)]
        L.imrt_plan_eval_batch.argtypes = [_P, i32, _P, _P, _P]
        L.imrt_plan_gradient.argtypes = [_P, _P, _P]
        L.imrt_plan_get_tuning.argtypes = [_P, _P, ctypes.c_size_t, ctypes.POINTER(ctypes.c_size_t)]
        L.imrt_plan_get_create_times.argtypes = [_P, _P, i32, ctypes.POINTER(i32)]
        L.imrt_shard_inbox_bytes.argtypes = [i64, i32, ctypes.POINTER(ctypes.c_size_t)]
        L.imrt_plan_set_shard.argtypes = [_P, i32, i32, ctypes.POINTER(_P)]
        L.imrt_plan_run_ranks.argtypes = [ctypes.POINTER(_P), i32, i32, dbl]
        L.imrt_merge_rows_workspace_bytes.argtypes = [i64, i64, ctypes.POINTER(ctypes.c_size_t)]
        L.imrt_merge_rows_count.argtypes = [i64, i64, _P, _P, _P, i64, _P, ctypes.POINTER(i64), _P, ctypes.c_size_t, _P]
        L.imrt_merge_rows_fill.argtypes = [i64, i64, _P, _P, _P, i64, _P, _P, _P, _P, ctypes.c_size_t, _P]
        L.imrt_trial_point.argtypes = [_P, _P, dbl, i64, _P, _P, _P]
        L.imrt_armijo_accepts.argtypes = [dbl] * 5
        L.imrt_stop_test.argtypes = [dbl] * 3
        L.imrt_plan_get_x.argtypes = [_P, _P]
        L.imrt_plan_get_dose.argtypes = [_P, _P]
        L.imrt_plan_dvh.argtypes = [_P, _P, i32, _P, _P]
        L.imrt_dvh_static.argtypes = [_P, _P, i64, i32, _P, i32, _P, _P, _P]
        L.imrt_plan_get_trace.argtypes = [_P, ctypes.POINTER(i32), ctypes.POINTER(i32), _P, _P, _P, _P, i32]
        L.imrt_plan_get_counters.argtypes = [_P, ctypes.POINTER(i64), ctypes.POINTER(i64)]
        L.imrt_plan_get_info.argtypes = [_P, _P, i32, _P, _P, _P]
        L.imrt_plan_launch_pass.argtypes = [_P, i32, i32]
        L.imrt_plan_get_pass_timing.argtypes = [_P, i32, _P, _P, i32, ctypes.POINTER(i32)]
        L.imrt_plan_destroy.argtypes = [_P]
        L.imrt_last_error.argtypes = [_P]
        L.imrt_last_error.restype = ctypes.c_char_p
        L.imrt_version.argtypes = []
        L.imrt_version.restype = ctypes.c_char_p
        for name in EXPORTS:
            if name in ("imrt_armijo_accepts", "imrt_stop_test"):
                getattr(L, name).restype = ctypes.c_int32
            elif name not in ("imrt_last_error", "imrt_version"):
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def _check(status: int, plan=None):
    if status != 0:
        msg = lib().imrt_last_error(plan)
        raise ImrtError(status, msg.decode() if msg else "")


def _dptr(t, dtype=None, n=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError("expected dtype %s, got %s" % (dtype, t.dtype))
    if n is not None and t.numel() < n:
        raise ValueError("tensor too small: %d < %d" % (t.numel(), n))
    return ctypes.c_void_p(t.data_ptr())


def _hptr(a):
    return a.ctypes.data_as(_P)


# ------------------------------------------------------------------------------------------------ C names
def imrt_version() -> str:
    return lib().imrt_version().decode()


def imrt_workspace_bytes(n_v: int, n_b: int, nnz: int, n_structures: int, max_iters: int) -> int:
    out = ctypes.c_size_t(0)
    _check(lib().imrt_workspace_bytes(n_v, n_b, nnz, n_structures, max_iters, ctypes.byref(out)))
    return out.value


def imrt_plan_create(n_v, n_b, nnz, row_ptr, col_idx, val, structure_id, t_under, t_over, w_under, w_over, params: Params,
                     workspace, stream_ptr: int = 0, options: Options = None):
    """Returns the opaque plan handle (a ctypes.c_void_p).  Tensors are borrowed: keep them alive."""
    import torch
    tabs = [np.ascontiguousarray(a, dtype=np.float32) for a in (t_under, t_over, w_under, w_over)]
    n_s = tabs[0].shape[0]
    handle = _P()
    st = lib().imrt_plan_create(ctypes.byref(handle), n_v, n_b, nnz, _dptr(row_ptr, torch.int32, n_v + 1),
                                _dptr(col_idx, torch.int32, nnz), _dptr(val, torch.float32, nnz),
                                _dptr(structure_id, torch.uint8, n_v), n_s, _hptr(tabs[0]), _hptr(tabs[1]), _hptr(tabs[2]),
                                _hptr(tabs[3]), ctypes.byref(params), ctypes.byref(options) if options is not None else None,
                                _dptr(workspace), workspace.numel() * workspace.element_size(),
                                ctypes.c_void_p(stream_ptr))
    _check(st, None)
    return handle


def imrt_plan_set_x(plan, x0):
    import torch
    _check(lib().imrt_plan_set_x(plan, _dptr(x0, torch.float32)), plan)


def imrt_plan_set_voxel_limits(plan, t_under_v=None, t_over_v=None):
    """Per-voxel limits (fp32 CUDA tensors [n_v], borrowed: keep them alive) or None for the structure's limit."""
    import torch
    _check(lib().imrt_plan_set_voxel_limits(plan, _dptr(t_under_v, torch.float32), _dptr(t_over_v, torch.float32)), plan)


def imrt_plan_run_iters(plan, n_iters: int):
    _check(lib().imrt_plan_run_iters(plan, n_iters), plan)


def imrt_plan_run_to_tol(plan, delta: float, max_iters: int):
    _check(lib().imrt_plan_run_to_tol(plan, delta, max_iters), plan)


def imrt_plan_eval(plan, x, d=None, r=None, g=None) -> float:
    import torch
    obj = ctypes.c_double(0.0)
    _check(lib().imrt_plan_eval(plan, _dptr(x, torch.float32), _dptr(d, torch.float32), _dptr(r, torch.float32),
                                _dptr(g, torch.float32), ctypes.byref(obj)), plan)
    return obj.value


def imrt_plan_eval_batch(plan, x, r=None):
    """x: fp32 CUDA tensor [n_points, n_b] (n_points = 1, 2 or 4); r: optional fp32 [n_points, n_v].  Returns G [n_points]."""
    import torch
    n = int(x.shape[0])
    obj = np.zeros(n, np.float64)
    _check(lib().imrt_plan_eval_batch(plan, n, _dptr(x, torch.float32), _dptr(r, torch.float32), _hptr(obj)), plan)
    return obj


def imrt_plan_get_tuning(plan) -> bytes:
    n = ctypes.c_size_t(0)
    _check(lib().imrt_plan_get_tuning(plan, None, 0, ctypes.byref(n)), plan)
    buf = ctypes.create_string_buffer(n.value)
    _check(lib().imrt_plan_get_tuning(plan, buf, n.value, ctypes.byref(n)), plan)
    return buf.raw


def imrt_plan_get_create_times(plan) -> dict:
    ms = np.zeros(16, np.float64)
    n = ctypes.c_int32(0)
    _check(lib().imrt_plan_get_create_times(plan, _hptr(ms), 16, ctypes.byref(n)), plan)
    return dict(zip(CREATE_PHASES, (float(v) for v in ms[:n.value])))


def imrt_shard_inbox_bytes(n_b: int, world: int) -> int:
    nb = ctypes.c_size_t(0)
    _check(lib().imrt_shard_inbox_bytes(n_b, world, ctypes.byref(nb)))
    return nb.value


def imrt_plan_set_shard(plan, rank: int, world: int, inbox_ptrs):
    """inbox_ptrs: device addresses (ints) of every rank's inbox as this rank's device addresses them."""
    arr = (_P * max(world, 1))(*[ctypes.c_void_p(int(p)) for p in inbox_ptrs]) if world > 1 else None
    _check(lib().imrt_plan_set_shard(plan, rank, world, arr), plan)


def imrt_plan_run_ranks(plans, n_iters: int, delta: float = 0.0):
    """Run the co-resident ranks `plans` (handles, in rank order) in one cooperative launch."""
    arr = (_P * len(plans))(*plans)
    _check(lib().imrt_plan_run_ranks(arr, len(plans), int(n_iters), float(delta)), plans[0])


def imrt_merge_rows_workspace_bytes(n_v: int, n_groups: int) -> int:
    nb = ctypes.c_size_t(0)
    _check(lib().imrt_merge_rows_workspace_bytes(n_v, n_groups, ctypes.byref(nb)))
    return nb.value


def imrt_merge_rows_count(n_v, n_b, row_ptr, col_idx, group_id, n_groups, out_row_ptr, workspace, stream_ptr: int = 0) -> int:
    """Fills out_row_ptr (int32 CUDA tensor [n_groups + 1]); returns the non-zeros of the merged matrix."""
    import torch
    nnz = ctypes.c_int64(0)
    _check(lib().imrt_merge_rows_count(n_v, n_b, _dptr(row_ptr, torch.int32, n_v + 1), _dptr(col_idx, torch.int32), _dptr(group_id, torch.int32, n_v),
                                       n_groups, _dptr(out_row_ptr, torch.int32, n_groups + 1), ctypes.byref(nnz), _dptr(workspace),
                                       workspace.numel() * workspace.element_size(), ctypes.c_void_p(stream_ptr)))
    return nnz.value


def imrt_merge_rows_fill(n_v, n_b, row_ptr, col_idx, val, n_groups, out_row_ptr, out_col, out_val, workspace, stream_ptr: int = 0):
    import torch
    _check(lib().imrt_merge_rows_fill(n_v, n_b, _dptr(row_ptr, torch.int32, n_v + 1), _dptr(col_idx, torch.int32), _dptr(val, torch.float32), n_groups,
                                      _dptr(out_row_ptr, torch.int32), _dptr(out_col, torch.int32), _dptr(out_val, torch.float32), _dptr(workspace),
                                      workspace.numel() * workspace.element_size(), ctypes.c_void_p(stream_ptr)))


def imrt_merge_rows(n_b: int, row_ptr, col_idx, val, group_id, n_groups: int, stream_ptr: int = 0):
    """Mixed-resolution row merging: (row_ptr, col, val) CUDA tensors of the matrix whose row g is the mean
    of the rows of D with group_id == g.  Allocation + the two C calls (imrt_merge_rows_count / imrt_merge_rows_fill)."""
    import torch
    n_v = row_ptr.numel() - 1
    ws = torch.empty(imrt_merge_rows_workspace_bytes(n_v, n_groups), dtype=torch.uint8, device=row_ptr.device)
    out_rp = torch.empty(n_groups + 1, dtype=torch.int32, device=row_ptr.device)
    nnz = imrt_merge_rows_count(n_v, n_b, row_ptr, col_idx, group_id, n_groups, out_rp, ws, stream_ptr)
    out_c = torch.empty(max(nnz, 4), dtype=torch.int32, device=row_ptr.device)
    out_v = torch.empty(max(nnz, 4), dtype=torch.float32, device=row_ptr.device)
    imrt_merge_rows_fill(n_v, n_b, row_ptr, col_idx, val, n_groups, out_rp, out_c, out_v, ws, stream_ptr)
    torch.cuda.current_stream(row_ptr.device).synchronize()      # ws goes out of scope
    return out_rp, out_c[:nnz], out_v[:nnz]


def imrt_plan_gradient(plan, r, g):
    import torch
    _check(lib().imrt_plan_gradient(plan, _dptr(r, torch.float32), _dptr(g, torch.float32)), plan)


def imrt_trial_point(x, g, lam: float, x_out, step_sq, stream_ptr: int = 0):
    """x_out = max(0, x - lam g); step_sq: float64 CUDA tensor of one element receiving ||x_out - x||^2."""
    import torch
    _check(lib().imrt_trial_point(_dptr(x, torch.float32), _dptr(g, torch.float32), float(lam), x.numel(),
                                  _dptr(x_out, torch.float32), _dptr(step_sq, torch.float64), ctypes.c_void_p(stream_ptr)))


def imrt_armijo_accepts(G_k: float, G_new: float, step_sq: float, eps: float, lam: float) -> bool:
    return bool(lib().imrt_armijo_accepts(G_k, G_new, step_sq, eps, lam))


def imrt_stop_test(G_old: float, G_new: float, delta: float) -> bool:
    return bool(lib().imrt_stop_test(G_old, G_new, delta))


def imrt_plan_get_x(plan, x):
    import torch
    _check(lib().imrt_plan_get_x(plan, _dptr(x, torch.float32)), plan)


def imrt_plan_get_dose(plan, d):
    import torch
    _check(lib().imrt_plan_get_dose(plan, _dptr(d, torch.float32)), plan)


def imrt_plan_dvh(plan, pcts, n_structures: int):
    pc = np.ascontiguousarray(pcts, dtype=np.float64)
    dp = np.empty((n_structures, pc.shape[0]), np.float64)
    mean = np.empty(n_structures, np.float64)
    _check(lib().imrt_plan_dvh(plan, _hptr(pc), pc.shape[0], _hptr(dp), _hptr(mean)), plan)
    return dp, mean


def imrt_dvh_static(dose, structure_id, n_structures: int, pcts, stream_ptr: int = 0):
    """DVH points and mean dose of an fp32 CUDA dose tensor without a plan or a workspace: the scratch is an array built
    into libimrtgp.so, so nothing is allocated on the device (for processes whose memory pool already owns the GPU).
    At most 16 structures and 128 structure x percentage pairs; one call at a time per process (the call synchronises)."""
    import torch
    pc = np.ascontiguousarray(pcts, dtype=np.float64)
    dp = np.empty((n_structures, pc.shape[0]), np.float64)
    mean = np.empty(n_structures, np.float64)
    n_v = dose.numel()
    _check(lib().imrt_dvh_static(_dptr(dose, torch.float32), _dptr(structure_id, torch.uint8, n_v), n_v, n_structures, _hptr(pc),
                                 pc.shape[0], _hptr(dp), _hptr(mean), ctypes.c_void_p(stream_ptr)))
    return dp, mean


@dataclass
class Trace:
    n_iters: int
    stop_reason: int
    obj: np.ndarray        # float64 [n+1]
    lam: np.ndarray        # float64 [n]
    n_trials: np.ndarray   # int32 [n]
    step_sq: np.ndarray    # float64 [n]


def imrt_plan_get_trace(plan, capacity: int) -> Trace:
    n = ctypes.c_int32(0)
    reason = ctypes.c_int32(0)
    obj = np.zeros(capacity + 1, np.float64)
    lam = np.zeros(max(capacity, 1), np.float64)
    ntr = np.zeros(max(capacity, 1), np.int32)
    ssq = np.zeros(max(capacity, 1), np.float64)
    _check(lib().imrt_plan_get_trace(plan, ctypes.byref(n), ctypes.byref(reason), _hptr(obj), _hptr(lam), _hptr(ntr),
                                     _hptr(ssq), capacity), plan)
    k = min(n.value, capacity)
    return Trace(n.value, reason.value, obj[:k + 1].copy(), lam[:k].copy(), ntr[:k].copy(), ssq[:k].copy())


def imrt_plan_get_counters(plan):
    f, t = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(lib().imrt_plan_get_counters(plan, ctypes.byref(f), ctypes.byref(t)), plan)
    return f.value, t.value


INFO_KEYS = ("nnzT", "fwd_blocks", "fwd_grid", "tr_grid", "smem_bytes", "pack_bytes", "g_slots", "nonempty_rows", "n_sm", "col16",
             "ls_batch", "fwd_ring_bytes", "tr_stages", "quad_rows", "tr_format", "tr_stream_bytes")


def imrt_plan_get_info(plan, rowT_ptr=None, colT=None, valT=None) -> dict:
    import torch
    info = np.zeros(len(INFO_KEYS), np.int64)
    _check(lib().imrt_plan_get_info(plan, _hptr(info), len(INFO_KEYS), _dptr(rowT_ptr, torch.int32), _dptr(colT, torch.int32),
                                    _dptr(valT, torch.float32)), plan)
    return dict(zip(INFO_KEYS, (int(v) for v in info)))


def imrt_plan_launch_pass(plan, kind: int, n_repeat: int):
    _check(lib().imrt_plan_launch_pass(plan, kind, n_repeat), plan)


def imrt_plan_get_pass_timing(plan, kind: int):
    """(start_ns, end_ns) int64 arrays, one entry per CTA of the last dose (0) / transpose (1) pass."""
    s = np.zeros(1024, np.int64)
    e = np.zeros(1024, np.int64)
    n = ctypes.c_int32(0)
    _check(lib().imrt_plan_get_pass_timing(plan, kind, _hptr(s), _hptr(e), 1024, ctypes.byref(n)), plan)
    return s[:n.value].copy(), e[:n.value].copy()


def imrt_plan_destroy(plan):
    _check(lib().imrt_plan_destroy(plan))


# ------------------------------------------------------------------------------------------------ convenience
class Plan:
    """Owns the device copies of a problem, the workspace and the plan handle.

    `prob` is any object with the fields n_v, n_b, row_ptr, col, val, sid, t_under, t_over, w_under, w_over,
    eps, alpha, lambda0, max_ls (numpy arrays / scalars); arrays may also already be torch CUDA tensors.
    """

    def __init__(self, prob, max_iters: int = 1000, driver: int = DRIVER_PERSISTENT, device="cuda:0", stream=None,
                 ls_batch: int = 0, tuning: bytes = None, **options):
        """options: fields of imrt_options (tune_level, dose_format, col_bits, transpose_format, quad_cap, n_ctas, profile_create, spin_timeout_ms); tuning: a blob from Plan.tuning() of an earlier plan of the same problem."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_0908_4421_b200 needs a CUDA device (sm_100a); there is no CPU path")
        lib()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)

        def dev(a, dt):
            if isinstance(a, torch.Tensor):
                return a.to(device=self.device, dtype=dt).contiguous()
            return torch.from_numpy(np.ascontiguousarray(a)).to(device=self.device, dtype=dt)

        self.n_v, self.n_b = int(prob.n_v), int(prob.n_b)
        self.row_ptr = dev(prob.row_ptr, torch.int32)
        self.nnz = int(self.row_ptr[-1].item()) if self.n_v > 0 else 0
        self.col = dev(prob.col, torch.int32) if self.nnz else torch.zeros(4, dtype=torch.int32, device=self.device)
        self.val = dev(prob.val, torch.float32) if self.nnz else torch.zeros(4, dtype=torch.float32, device=self.device)
        self.sid = dev(prob.sid, torch.uint8)
        self.n_structures = int(len(prob.t_under))
        self.max_iters = int(max_iters)
        self.params = Params(float(prob.eps), float(prob.alpha), float(prob.lambda0), int(prob.max_ls), self.max_iters,
                             int(driver), int(ls_batch))
        nbytes = imrt_workspace_bytes(self.n_v, self.n_b, self.nnz, self.n_structures, self.max_iters)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.options = Options(**{k: int(v) for k, v in options.items()})
        self._tuning = tuning
        if tuning is not None:
            self._tuning_buf = ctypes.create_string_buffer(tuning, len(tuning))
            self.options.host_tuning = ctypes.cast(self._tuning_buf, ctypes.c_void_p)
            self.options.host_tuning_bytes = len(tuning)
        self.handle = imrt_plan_create(self.n_v, self.n_b, self.nnz, self.row_ptr, self.col, self.val, self.sid,
                                       prob.t_under, prob.t_over, prob.w_under, prob.w_over, self.params, self.workspace,
                                       self.stream.cuda_stream, self.options)
        self._tvu = self._tvo = None
        if getattr(prob, "tv_under", None) is not None or getattr(prob, "tv_over", None) is not None:
            self.set_voxel_limits(getattr(prob, "tv_under", None), getattr(prob, "tv_over", None))

    # -- the calls of the C-ABI
    def set_x(self, x0):
        import torch
        if not isinstance(x0, torch.Tensor):
            x0 = torch.from_numpy(np.ascontiguousarray(x0, dtype=np.float32))
        self._x0 = x0.to(device=self.device, dtype=torch.float32).contiguous()
        imrt_plan_set_x(self.handle, self._x0)

    def set_voxel_limits(self, t_under_v=None, t_over_v=None):
        import torch

        def dev(a):
            if a is None:
                return None
            if not isinstance(a, torch.Tensor):
                a = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
            return a.to(device=self.device, dtype=torch.float32).contiguous()

        self._tvu, self._tvo = dev(t_under_v), dev(t_over_v)      # borrowed by the plan: keep them alive
        imrt_plan_set_voxel_limits(self.handle, self._tvu, self._tvo)

    def run_iters(self, n: int):
        imrt_plan_run_iters(self.handle, int(n))

    def run_to_tol(self, delta: float, max_iters: int):
        imrt_plan_run_to_tol(self.handle, float(delta), int(max_iters))

    def eval(self, x, want_d=True, want_r=True, want_g=True):
        """(d, r, g, G) at x -- tensors on the device (None where not wanted)."""
        import torch
        if not isinstance(x, torch.Tensor):
            x = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32))
        x = x.to(device=self.device, dtype=torch.float32).contiguous()
        d = torch.empty(self.n_v, dtype=torch.float32, device=self.device) if want_d else None
        r = torch.empty(self.n_v, dtype=torch.float32, device=self.device) if want_r else None
        g = torch.empty(self.n_b, dtype=torch.float32, device=self.device) if want_g else None
        G = imrt_plan_eval(self.handle, x, d, r, g)
        return d, r, g, G

    def eval_batch(self, xs, want_r=True):
        """(r [n, n_v] or None, G [n]) of n = 1, 2 or 4 points evaluated in one pass over D (the line search's batched pass)."""
        import torch
        x = torch.from_numpy(np.ascontiguousarray(xs, dtype=np.float32)).to(self.device) if not isinstance(xs, torch.Tensor) else xs
        x = x.to(device=self.device, dtype=torch.float32).contiguous()
        r = torch.empty((x.shape[0], self.n_v), dtype=torch.float32, device=self.device) if want_r else None
        return r, imrt_plan_eval_batch(self.handle, x, r)

    def gradient(self, r):
        """g = D^T r for an arbitrary residual (one transpose pass)."""
        import torch
        if not isinstance(r, torch.Tensor):
            r = torch.from_numpy(np.ascontiguousarray(r, dtype=np.float32))
        r = r.to(device=self.device, dtype=torch.float32).contiguous()
        g = torch.empty(self.n_b, dtype=torch.float32, device=self.device)
        imrt_plan_gradient(self.handle, r, g)
        return g

    def tuning(self) -> bytes:
        return imrt_plan_get_tuning(self.handle)

    def create_times(self) -> dict:
        return imrt_plan_get_create_times(self.handle)

    def get_x(self):
        import torch
        x = torch.empty(self.n_b, dtype=torch.float32, device=self.device)
        imrt_plan_get_x(self.handle, x)
        return x

    def get_dose(self):
        import torch
        d = torch.empty(self.n_v, dtype=torch.float32, device=self.device)
        imrt_plan_get_dose(self.handle, d)
        return d

    def dvh(self, pcts):
        return imrt_plan_dvh(self.handle, pcts, self.n_structures)

    def trace(self) -> Trace:
        return imrt_plan_get_trace(self.handle, self.max_iters)

    def counters(self):
        return imrt_plan_get_counters(self.handle)

    def info(self) -> dict:
        return imrt_plan_get_info(self.handle)

    def transpose_csr(self):
        """(rowT_ptr, colT, valT) copies of the library-built D^T."""
        import torch
        rp = torch.empty(self.n_b + 1, dtype=torch.int32, device=self.device)
        c = torch.empty(max(self.nnz, 1), dtype=torch.int32, device=self.device)
        v = torch.empty(max(self.nnz, 1), dtype=torch.float32, device=self.device)
        imrt_plan_get_info(self.handle, rp, c, v)
        return rp, c[:self.nnz], v[:self.nnz]

    def pass_timing(self, kind: int):
        return imrt_plan_get_pass_timing(self.handle, int(kind))

    def launch_pass(self, kind: int, n_repeat: int = 1):
        imrt_plan_launch_pass(self.handle, int(kind), int(n_repeat))

    def close(self):
        if getattr(self, "handle", None):
            imrt_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
