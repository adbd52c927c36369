"""Row-sharded gradient projection: slab selection and the set-up of the device-resident sharded loop.

Rank q holds a contiguous slab of rows of D (voxels) -- and with it the matching columns of D^T --, the full x,
and computes local dose, residual, a partial objective and a partial gradient over ALL beamlets.  The exchange
steps of the method are

    g     = sum over ranks of D_q^T r_q         n_b fp32 (9-15 KB) per iteration
    G(x+) = sum over ranks of G_q(x+)           R scalars per batch of line-search trial points

and every rank takes the same Armijo decisions from the same sums (readings R4-R7 of DESIGN.md),
so the iterates stay replicated without ever being broadcast.

BOTH exchange steps run INSIDE the library's persistent kernel (csrc/kernels.cuh: shard_sum_gradient /
shard_sum_objective): a rank pushes its partial into every rank's inbox with peer-memory stores, raises a sequence
flag, and adds its own inbox's entries in rank order.  This module only marshals: it cuts the slabs, allocates the
inboxes, hands every plan the inbox addresses (imrt_plan_set_shard) and calls the run functions.  None of the
method's arithmetic or control flow lives here.

  CoResidentRanks   all ranks on ONE device, each on its share of the SMs, one cooperative launch
                    (imrt_plan_run_ranks) -- how the sharded loop is exercised where a single GPU is available
  PeerRank          one rank per process / GPU (torchrun): the inboxes live in torch symmetric memory, whose rendezvous
                    returns every peer's buffer address as this device maps it (NVLink peer access)
"""
from __future__ import annotations

import copy

import numpy as np


def slab_bounds(row_ptr: np.ndarray, world: int) -> np.ndarray:
    """Row boundaries [world + 1] of contiguous slabs with (nearly) equal numbers of non-zeros; every slab gets at least
    one row as long as there are at least `world` rows (a plan cannot be created from zero rows)."""
    row_ptr = np.asarray(row_ptr, dtype=np.int64)
    n_v, nnz = row_ptr.shape[0] - 1, int(row_ptr[-1])
    b = np.zeros(world + 1, dtype=np.int64)
    for q in range(1, world):
        b[q] = int(np.searchsorted(row_ptr, nnz * q // world, side="left"))
    b[world] = n_v
    b = np.maximum.accumulate(np.minimum(b, n_v))
    if n_v >= world:
        for q in range(1, world):                    # push boundaries apart where a slab came out empty
            b[q] = max(b[q], b[q - 1] + 1)
        for q in range(world - 1, 0, -1):
            b[q] = min(b[q], b[q + 1] - 1)
    return b


def shard_rows(prob, world: int, rank: int):
    """The sub-problem of `rank`: rows [r0, r1) of D with their structure ids (and per-voxel limits, if any)."""
    if prob.n_v < world:             # the same refusal on every rank, before any collective
        raise ValueError("%d ranks for a %d-row matrix: some rank would hold no rows; use fewer ranks" % (world, prob.n_v))
    b = slab_bounds(prob.row_ptr, world)
    r0, r1 = int(b[rank]), int(b[rank + 1])
    p0, p1 = int(prob.row_ptr[r0]), int(prob.row_ptr[r1])
    sub = copy.copy(prob)
    sub.name = "%s[rows %d:%d]" % (prob.name, r0, r1)
    sub.n_v = r1 - r0
    sub.row_ptr = np.ascontiguousarray(prob.row_ptr[r0:r1 + 1] - prob.row_ptr[r0]).astype(np.int32)
    sub.col = np.ascontiguousarray(prob.col[p0:p1])
    sub.val = np.ascontiguousarray(prob.val[p0:p1])
    sub.sid = np.ascontiguousarray(prob.sid[r0:r1])
    for name in ("tv_under", "tv_over", "voxel_ids"):
        a = getattr(prob, name, None)
        setattr(sub, name, None if a is None else np.ascontiguousarray(a[r0:r1]))
    return sub, (r0, r1)


class CoResidentRanks:
    """`world` ranks of one problem on ONE device: plan q gets slab q and SMs / world CTAs; all of them run in one
    cooperative launch and exchange through inboxes in that device's memory, exactly as ranks on different GPUs do."""

    def __init__(self, prob, world: int, max_iters: int = 1000, device="cuda:0", **options):
        import torch
        from . import Plan, imrt_plan_set_shard, imrt_shard_inbox_bytes
        self.device = torch.device(device)
        self.world = int(world)
        n_sm = torch.cuda.get_device_properties(self.device).multi_processor_count
        self.rows = []
        self.plans = []
        for q in range(self.world):
            sub, rows = shard_rows(prob, self.world, q)
            self.rows.append(rows)
            self.plans.append(Plan(sub, max_iters=max_iters, device=self.device, n_ctas=n_sm // self.world, **options))
        nbytes = imrt_shard_inbox_bytes(int(prob.n_b), self.world)
        self.inboxes = [torch.zeros(nbytes, dtype=torch.uint8, device=self.device) for _ in range(self.world)]
        ptrs = [t.data_ptr() for t in self.inboxes]
        for q, p in enumerate(self.plans):
            imrt_plan_set_shard(p.handle, q, self.world, ptrs)

    def set_x(self, x0):
        for p in self.plans:
            p.set_x(x0)

    def run_iters(self, n: int):
        from . import imrt_plan_run_ranks
        imrt_plan_run_ranks([p.handle for p in self.plans], int(n), 0.0)

    def run_to_tol(self, delta: float, max_iters: int):
        from . import imrt_plan_run_ranks
        imrt_plan_run_ranks([p.handle for p in self.plans], int(max_iters), float(delta))

    def trace(self, rank: int = 0):
        return self.plans[rank].trace()

    def get_x(self, rank: int = 0):
        return self.plans[rank].get_x()

    def get_dose(self):
        """Dose of the whole problem: the slabs' doses in row order."""
        import torch
        return torch.cat([p.get_dose() for p in self.plans])

    def close(self):
        for p in self.plans:
            p.close()


class PeerRank:
    """This process's rank of a row-sharded problem, one GPU per process (torch.distributed initialised, NCCL).  The inbox
    is allocated in torch symmetric memory; its rendezvous maps every peer's inbox into this device's address space."""

    def __init__(self, prob, max_iters: int = 1000, device=None, group=None, **options):
        import torch
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm_mem
        from . import Plan, imrt_plan_set_shard, imrt_shard_inbox_bytes
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.device = torch.device(device if device is not None else "cuda:%d" % torch.cuda.current_device())
        sub, self.rows = shard_rows(prob, self.world, self.rank)
        self.plan = Plan(sub, max_iters=max_iters, device=self.device, **options)
        nbytes = imrt_shard_inbox_bytes(int(prob.n_b), self.world)
        self.inbox = symm_mem.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.inbox.zero_()
        self.handle = symm_mem.rendezvous(self.inbox, group if group is not None else dist.group.WORLD)
        torch.cuda.synchronize(self.device)
        dist.barrier(group)                          # every inbox is zero before anybody pushes
        imrt_plan_set_shard(self.plan.handle, self.rank, self.world, [int(p) for p in self.handle.buffer_ptrs])

    def set_x(self, x0):
        self.plan.set_x(x0)

    def run_iters(self, n: int):
        self.plan.run_iters(n)

    def run_to_tol(self, delta: float, max_iters: int):
        self.plan.run_to_tol(delta, max_iters)

    def trace(self):
        return self.plan.trace()

    def close(self):
        self.plan.close()
