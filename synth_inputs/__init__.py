"""Seeded synthetic inputs shared by the oracle tests and the CUDA library tests.

This module is HARNESS code: it produces arrays (CSR dose-deposition matrix,
structure ids, penalty table, x0, line-search parameters) and holds none of
the optimiser's arithmetic.  It imports neither ``oracle`` nor
``paper_0908_4421_b200``; both are handed the very same arrays.

The five phantoms follow BASELINE.json ``configs`` under the geometry reading of
SURVEY.md section 8(d); they stand in for the clinical prostate case of
PAPER.md:150 (section 3.1), which is not in this repository.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "phantom_gen.c")
_LIB = os.path.join(_HERE, "libphantom_gen.so")


def build(force: bool = False) -> str:
    """Compile the generator with gcc (idempotent)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Cfg(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("h", ctypes.c_double), ("geom", ctypes.c_int32), ("n_beams", ctypes.c_int32),
                ("beamlet", ctypes.c_double), ("half_field", ctypes.c_double),
                ("sigma", ctypes.c_double), ("tau", ctypes.c_double), ("mu", ctypes.c_double)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P = ctypes.c_void_p
        lib.phantom_structures.argtypes = [ctypes.POINTER(_Cfg), P]
        lib.phantom_structures.restype = None
        lib.phantom_dose_max.argtypes = [ctypes.POINTER(_Cfg), ctypes.c_int64, P]
        lib.phantom_dose_max.restype = ctypes.c_double
        lib.phantom_dose_count.argtypes = [ctypes.POINTER(_Cfg), ctypes.c_int64, P, ctypes.c_double, P]
        lib.phantom_dose_count.restype = None
        lib.phantom_dose_fill.argtypes = [ctypes.POINTER(_Cfg), ctypes.c_int64, P, ctypes.c_double, P, P, P]
        lib.phantom_dose_fill.restype = None
        lib.phantom_power_iter.argtypes = [ctypes.c_int64, ctypes.c_int64, P, P, P, P, ctypes.c_int]
        lib.phantom_power_iter.restype = ctypes.c_double
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


# ----------------------------------------------------------------------------------------------
# Configurations (BASELINE.json `configs`)
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class PhantomConfig:
    name: str
    grid: tuple            # (nx, ny, nz)
    h: float               # mm
    geom: int              # 0 box phantom, 1 elliptic phantom
    n_beams: int
    beamlet: float         # mm
    sigma: float           # mm
    tau: float
    seed: int
    x0_uniform_one: bool   # config 0: x0 = 1.0
    n_iters: int           # iteration cap / fixed count
    delta: float           # 0 => fixed-count run
    mu: float = 0.005

    @property
    def half_field(self) -> float:
        h_max = 20.0 if self.geom == 0 else 30.0
        return 10.0 * math.ceil((h_max + 5.0) / 10.0)

    @property
    def n_beamlets(self) -> int:
        m = int(round(2 * self.half_field / self.beamlet))
        return self.n_beams * m * m


CONFIGS = {
    0: PhantomConfig("cfg0-tiny-5field", (40, 40, 24), 5.0, 0, 5, 10.0, 6.0, 1e-3, 0, True, 50, 0.0),
    1: PhantomConfig("cfg1-9field-10mm-5mm", (64, 96, 48), 5.0, 1, 9, 10.0, 6.0, 1e-3, 1, False, 200, 0.0),
    2: PhantomConfig("cfg2-9field-5mm-5mm", (64, 96, 48), 5.0, 1, 9, 5.0, 4.0, 1e-3, 2, False, 500, 1e-6),
    3: PhantomConfig("cfg3-9field-5mm-2.5mm", (128, 192, 96), 2.5, 1, 9, 5.0, 6.0, 1e-3, 3, False, 500, 1e-6),
    4: PhantomConfig("cfg4-15field-5mm-2mm", (200, 240, 120), 2.0, 1, 15, 5.0, 5.0, 5e-4, 3, False, 300, 0.0),
}

# (T_under, T_over, w_under, w_over) per structure: PTV, rectum, bladder, body   [BASELINE.json, SURVEY 8(d)]
PENALTY_TABLE = np.array([[70.0, 70.0, 100.0, 100.0],
                          [0.0, 50.0, 0.0, 10.0],
                          [0.0, 50.0, 0.0, 10.0],
                          [0.0, 60.0, 0.0, 1.0]], dtype=np.float32)
STRUCTURE_NAMES = ("PTV", "rectum", "bladder", "body")


@dataclass
class Problem:
    """Everything both sides need; arrays are C-contiguous numpy."""
    name: str
    n_v: int
    n_b: int
    row_ptr: np.ndarray      # int32 [n_v+1]
    col: np.ndarray          # int32 [nnz], ascending within a row
    val: np.ndarray          # float32 [nnz]
    sid: np.ndarray          # uint8 [n_v]
    t_under: np.ndarray      # float32 [n_s]
    t_over: np.ndarray
    w_under: np.ndarray
    w_over: np.ndarray
    x0: np.ndarray           # float32 [n_b], >= 0
    eps: float = 0.2
    alpha: float = 2.0
    lambda0: float = 1.0
    delta: float = 0.0
    max_ls: int = 40
    n_iters: int = 50
    voxel_ids: np.ndarray | None = None   # row -> linear grid id (phantoms only)
    tv_under: np.ndarray | None = None    # optional per-voxel limits, float32 [n_v] (PAPER.md:58 T_j); None = per structure
    tv_over: np.ndarray | None = None
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    @property
    def n_structures(self) -> int:
        return int(self.t_under.shape[0])


def pick_lambda0(row_ptr, col, val, sid, w_under, w_over, n_iter: int = 30) -> tuple:
    """lambda0 = 2^ceil(log2(8 / L)), L = 2 lambda_max(D^T diag(max(w-, w+)) D)   [SURVEY 8(c.2) #4]."""
    lib = _load()
    w_row = np.maximum(w_under.astype(np.float64), w_over.astype(np.float64))[sid]
    w_row = np.ascontiguousarray(w_row)
    n_v = sid.shape[0]
    n_b = int(col.max()) + 1 if col.size else 1
    lam = lib.phantom_power_iter(n_v, n_b, _p(row_ptr), _p(col), _p(val), _p(w_row), n_iter)
    L = 2.0 * lam
    if not (L > 0.0) or not math.isfinite(L):
        return 1.0, L
    return 2.0 ** math.ceil(math.log2(8.0 / L)), L


def make_phantom(cfg_id: int) -> Problem:
    """Build config `cfg_id` (0..4).  cfg3 takes a few seconds and ~1 GB, cfg4 ~3 GB of host memory."""
    cfg = CONFIGS[cfg_id]
    lib = _load()
    nx, ny, nz = cfg.grid
    c = _Cfg(nx, ny, nz, cfg.h, cfg.geom, cfg.n_beams, cfg.beamlet, cfg.half_field, cfg.sigma, cfg.tau, cfg.mu)
    sid_grid = np.empty(nx * ny * nz, dtype=np.uint8)
    lib.phantom_structures(ctypes.byref(c), _p(sid_grid))
    vox = np.ascontiguousarray(np.flatnonzero(sid_grid != 255).astype(np.int64))
    sid = np.ascontiguousarray(sid_grid[vox])
    n_v = int(vox.shape[0])
    gmax = lib.phantom_dose_max(ctypes.byref(c), n_v, _p(vox))
    row_nnz = np.zeros(n_v, dtype=np.int64)
    lib.phantom_dose_count(ctypes.byref(c), n_v, _p(vox), gmax, _p(row_nnz))
    row_ptr64 = np.zeros(n_v + 1, dtype=np.int64)
    np.cumsum(row_nnz, out=row_ptr64[1:])
    nnz = int(row_ptr64[-1])
    assert nnz < 2 ** 31
    col = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float32)
    lib.phantom_dose_fill(ctypes.byref(c), n_v, _p(vox), gmax, _p(row_ptr64), _p(col), _p(val))
    row_ptr = row_ptr64.astype(np.int32)
    n_b = cfg.n_beamlets
    tab = PENALTY_TABLE
    if cfg.x0_uniform_one:
        x0 = np.ones(n_b, dtype=np.float32)
    else:
        x0 = np.random.default_rng(cfg.seed).uniform(0.5, 1.5, size=n_b).astype(np.float32)
    t_u, t_o, w_u, w_o = (np.ascontiguousarray(tab[:, i]) for i in range(4))
    lam0, L = pick_lambda0(row_ptr, col, val, sid, w_u, w_o)
    return Problem(cfg.name, n_v, n_b, row_ptr, col, val, sid, t_u, t_o, w_u, w_o, x0,
                   eps=0.2, alpha=2.0, lambda0=lam0, delta=cfg.delta, max_ls=40, n_iters=cfg.n_iters,
                   voxel_ids=vox, meta={"cfg_id": cfg_id, "gmax": gmax, "L_hat": L, "grid": cfg.grid, "h": cfg.h,
                                        "nonempty_rows": int((row_nnz > 0).sum())})


def make_random(seed: int, n_v: int, n_b: int, density: float = 0.3, n_structures: int = 3,
                empty_row_frac: float = 0.1, full_rows: int = 0, target_frac: float = 0.4) -> Problem:
    """Small random CSR problems with empty rows, single-entry rows and optional full rows (edge cases)."""
    rng = np.random.default_rng(seed)
    rows = []
    for j in range(n_v):
        r = rng.random()
        if j < full_rows:
            cols = np.arange(n_b)
        elif r < empty_row_frac:
            cols = np.empty(0, dtype=np.int64)
        elif r < empty_row_frac + 0.05:
            cols = rng.integers(0, n_b, size=1)
        else:
            k = max(1, int(rng.binomial(n_b, density)))
            cols = np.sort(rng.choice(n_b, size=min(k, n_b), replace=False))
        rows.append(cols)
    row_ptr = np.zeros(n_v + 1, dtype=np.int32)
    row_ptr[1:] = np.cumsum([len(r) for r in rows])
    col = np.concatenate(rows).astype(np.int32) if rows else np.empty(0, np.int32)
    val = rng.uniform(0.05, 1.0, size=col.shape[0]).astype(np.float32)
    sid = rng.integers(0, n_structures, size=n_v).astype(np.uint8)
    # structure 0 is a target (two-sided), the others are one-sided limits
    t_u = np.zeros(n_structures, np.float32)
    t_o = rng.uniform(20.0, 60.0, size=n_structures).astype(np.float32)
    w_u = np.zeros(n_structures, np.float32)
    w_o = rng.uniform(0.5, 10.0, size=n_structures).astype(np.float32)
    t_u[0] = t_o[0] = 70.0
    w_u[0] = w_o[0] = 100.0
    x0 = rng.uniform(0.5, 1.5, size=n_b).astype(np.float32)
    sid[: max(1, int(target_frac * n_v))] = 0
    prob = Problem("random-%d" % seed, n_v, n_b, row_ptr, np.ascontiguousarray(col), val, sid,
                   t_u, t_o, w_u, w_o, x0, n_iters=30)
    if col.size:
        prob.lambda0, _ = pick_lambda0(row_ptr, prob.col, val, sid, w_u, w_o)
    return prob


def mixed_resolution_groups(prob: Problem, body_sid: int = 3):
    """Group id per row for the paper's mixed-resolution problem: every target / OAR voxel is a group of
    its own (ids 0 .. n_fine-1, in row order), the body voxels of one 2x2x2 block share a group (ids n_fine ..., in
    ascending block key).  Returns (group int32 [n_v], n_groups, structure id per group uint8 [n_groups]).  Index
    arithmetic only: the merging itself is imrt_merge_rows (library) / oracle.merge_rows (oracle)."""
    nx, ny, nz = prob.meta["grid"]
    vid = prob.voxel_ids
    ix, iy, iz = vid % nx, (vid // nx) % ny, vid // (nx * ny)
    body = prob.sid == body_sid
    key = (ix // 2) + ((nx + 1) // 2) * ((iy // 2) + ((ny + 1) // 2) * (iz // 2))
    n_fine = int((~body).sum())
    uniq, inv = np.unique(key[body], return_inverse=True)
    group = np.empty(prob.n_v, np.int32)
    group[~body] = np.arange(n_fine, dtype=np.int32)
    group[body] = n_fine + inv.astype(np.int32)
    n_groups = n_fine + int(uniq.shape[0])
    sid_g = np.concatenate([prob.sid[~body], np.full(uniq.shape[0], body_sid, np.uint8)])
    return group, n_groups, sid_g


def mixed_resolution(prob: Problem, body_sid: int = 3) -> Problem:
    """The paper's mixed-resolution problem: voxels of unspecified tissue (structure `body_sid`) are
    doubled in each dimension, targets and OARs keep the full resolution.  A coarse voxel's row of D is the mean of
    the rows of the fine body voxels it contains (its dose is their mean dose); it counts as ONE voxel in Eq. (1),
    as every voxel does in the paper (reading R17).  Harness code: sparse row averaging with scipy, no
    optimiser arithmetic.  Rows: the full-resolution voxels in their order, then the coarse voxels."""
    import scipy.sparse as sp
    nx, ny, nz = prob.meta["grid"]
    vid = prob.voxel_ids
    ix, iy, iz = vid % nx, (vid // nx) % ny, vid // (nx * ny)
    body = prob.sid == body_sid
    key = (ix // 2) + ((nx + 1) // 2) * ((iy // 2) + ((ny + 1) // 2) * (iz // 2))
    fine_rows = np.flatnonzero(~body)
    body_rows = np.flatnonzero(body)
    uniq, inv = np.unique(key[body_rows], return_inverse=True)
    counts = np.bincount(inv).astype(np.float64)
    D = sp.csr_matrix((prob.val.astype(np.float64), prob.col, prob.row_ptr), shape=(prob.n_v, prob.n_b))
    S = sp.csr_matrix((1.0 / counts[inv], (inv, np.arange(body_rows.shape[0]))), shape=(uniq.shape[0], body_rows.shape[0]))
    Dm = sp.vstack([D[fine_rows], S @ D[body_rows]]).tocsr()
    Dm.sort_indices()
    Dm.eliminate_zeros()
    out = Problem(prob.name + "-mixed", Dm.shape[0], prob.n_b, Dm.indptr.astype(np.int32), Dm.indices.astype(np.int32),
                  Dm.data.astype(np.float32),
                  np.concatenate([prob.sid[fine_rows], np.full(uniq.shape[0], body_sid, np.uint8)]),
                  prob.t_under, prob.t_over, prob.w_under, prob.w_over, prob.x0, eps=prob.eps, alpha=prob.alpha,
                  delta=prob.delta, max_ls=prob.max_ls, n_iters=prob.n_iters,
                  meta={**prob.meta, "fine_rows": int(fine_rows.shape[0]), "coarse_rows": int(uniq.shape[0]),
                        "body_rows_merged": int(body_rows.shape[0])})
    out.lambda0, _ = pick_lambda0(out.row_ptr, out.col, out.val, out.sid, out.w_under, out.w_over)
    return out


def make_banded(seed: int, n_v: int, n_b: int, width: int, jitter: float, empty_frac: float, n_structures: int = 3) -> Problem:
    """Rows whose column sets drift slowly from row to row (neighbouring rows overlap, as neighbouring voxels do), with
    holes, empty rows and rows of very different lengths: the shapes that make a plan mix its record formats."""
    rng = np.random.default_rng(seed)
    rows, c0 = [], 0.0
    for _ in range(n_v):
        if rng.random() < empty_frac:
            rows.append(np.empty(0, np.int64))
            continue
        c0 = (c0 + rng.uniform(0, jitter)) % max(1, n_b - width)
        w = max(1, int(width * rng.uniform(0.5, 1.0)))
        cols = np.arange(int(c0), min(n_b, int(c0) + w))
        if rng.random() < 0.3 and cols.size > 3:
            cols = np.unique(np.delete(cols, rng.integers(0, cols.size, size=max(1, cols.size // 6))))
        rows.append(cols)
    row_ptr = np.zeros(n_v + 1, np.int32)
    row_ptr[1:] = np.cumsum([len(r) for r in rows])
    col = np.concatenate(rows).astype(np.int32) if row_ptr[-1] else np.empty(0, np.int32)
    val = rng.uniform(0.05, 1.0, col.shape[0]).astype(np.float32)
    sid = rng.integers(0, n_structures, n_v).astype(np.uint8)
    sid[: max(1, n_v // 3)] = 0
    t_u = np.zeros(n_structures, np.float32)
    t_o = rng.uniform(20.0, 60.0, n_structures).astype(np.float32)
    w_u = np.zeros(n_structures, np.float32)
    w_o = rng.uniform(0.5, 10.0, n_structures).astype(np.float32)
    t_u[0] = t_o[0] = 70.0
    w_u[0] = w_o[0] = 100.0
    x0 = rng.uniform(0.5, 1.5, n_b).astype(np.float32)
    prob = Problem("banded-%d" % seed, n_v, n_b, row_ptr, col, val, sid, t_u, t_o, w_u, w_o, x0, n_iters=10)
    if col.size:
        prob.lambda0, _ = pick_lambda0(row_ptr, col, val, sid, w_u, w_o)
    return prob


def make_quad_blocks(seed: int, n_quads: int, n_b: int, tail_rows: int, lengths=(0, 1, 3, 17, 40, 300),
                     n_structures: int = 3) -> Problem:
    """Groups of 4 consecutive rows that share one column window (so that a plan picks its quad-row records), the
    window length drawn per group from `lengths` -- neighbouring groups differ wildly, some are empty, rows inside a
    group drop a few columns -- followed by `tail_rows` (0..3) rows of a last, incomplete group.  No arithmetic of the
    method here: only the sparsity pattern and random values."""
    rng = np.random.default_rng(seed)
    rows = []
    n_groups = n_quads + (1 if tail_rows else 0)
    for q in range(n_groups):
        L = min(int(rng.choice(lengths)), n_b)
        c0 = int(rng.integers(0, n_b - L + 1))
        window = np.arange(c0, c0 + L)
        for i in range(4 if q < n_quads else tail_rows):
            if L == 0 or rng.random() < 0.1:
                rows.append(np.empty(0, np.int64))            # a row without entries inside a group
            else:
                keep = rng.random(L) < rng.uniform(0.6, 1.0)
                keep[rng.integers(0, L)] = True
                rows.append(window[keep])
    n_v = len(rows)
    row_ptr = np.zeros(n_v + 1, np.int32)
    row_ptr[1:] = np.cumsum([len(r) for r in rows])
    col = np.concatenate(rows).astype(np.int32) if row_ptr[-1] else np.empty(0, np.int32)
    val = rng.uniform(0.05, 1.0, col.shape[0]).astype(np.float32)
    sid = rng.integers(0, n_structures, n_v).astype(np.uint8)
    sid[: max(1, n_v // 3)] = 0
    t_u = np.zeros(n_structures, np.float32)
    t_o = rng.uniform(20.0, 60.0, n_structures).astype(np.float32)
    w_u = np.zeros(n_structures, np.float32)
    w_o = rng.uniform(0.5, 10.0, n_structures).astype(np.float32)
    t_u[0] = t_o[0] = 70.0
    w_u[0] = w_o[0] = 100.0
    x0 = rng.uniform(0.5, 1.5, n_b).astype(np.float32)
    prob = Problem("quadblocks-%d" % seed, n_v, n_b, row_ptr, col, val, sid, t_u, t_o, w_u, w_o, x0, n_iters=10)
    if col.size:
        prob.lambda0, _ = pick_lambda0(row_ptr, col, val, sid, w_u, w_o)
    return prob
