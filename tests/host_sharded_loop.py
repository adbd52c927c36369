"""Host-driven reference of the row-sharded loop -- TEST INFRASTRUCTURE (tests/ only).

The product's sharded loop runs inside the library's persistent kernel (paper_0908_4421_b200/sharded.py sets it up).  This
module spells the same protocol out on the host -- the Main Iterative Loop of PAPER.md:99-114 over row slabs with the two
exchange steps as torch.distributed all-reduces -- so that it can run under the gloo backend on CPU with oracle-backed
shards (world_size 2), and, on a GPU, over the library's per-slab calls (imrt_plan_eval / imrt_plan_gradient /
imrt_trial_point) as an independent check of the device-resident loop.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

STOP_MAX_ITERS, STOP_TOLERANCE, STOP_STATIONARY, STOP_LS_STALLED = 0, 1, 2, 3


@dataclass
class ShardedTrace:
    n_iters: int
    stop_reason: int
    obj: np.ndarray        # float64 [n+1]
    lam: np.ndarray        # float64 [n]
    n_trials: np.ndarray   # int32 [n]
    step_sq: np.ndarray    # float64 [n]


class GpuShard:
    """One slab on one GPU: a Plan of the sub-problem; every method is one C-ABI call (argument marshalling only)."""

    def __init__(self, sub_prob, device):
        import torch
        from paper_0908_4421_b200 import Plan, imrt_plan_eval, imrt_plan_gradient, imrt_trial_point
        self._eval, self._grad, self._trial = imrt_plan_eval, imrt_plan_gradient, imrt_trial_point
        self.device = torch.device(device)
        self.n_b = int(sub_prob.n_b)
        self.plan = Plan(sub_prob, max_iters=1, device=self.device)
        self.r = torch.empty(max(int(sub_prob.n_v), 1), dtype=torch.float32, device=self.device)
        self.step = torch.zeros(1, dtype=torch.float64, device=self.device)

    def vector(self, x0):
        import torch
        return torch.from_numpy(np.ascontiguousarray(x0, dtype=np.float32)).to(self.device)

    def eval_partial(self, x) -> float:
        """G_q(x); leaves r_q(x) in self.r."""
        return self._eval(self.plan.handle, x, None, self.r, None)

    def grad_partial(self):
        """D_q^T r_q for the residual of the last eval_partial (fp32 [n_b])."""
        import torch
        g = torch.empty(self.n_b, dtype=torch.float32, device=self.device)
        self._grad(self.plan.handle, self.r, g)
        return g

    def trial_point(self, x, g, lam: float):
        import torch
        x_new = torch.empty_like(x)
        self._trial(x, g, lam, x_new, self.step, self.plan.stream.cuda_stream)
        return x_new, float(self.step.item())

    def to_numpy(self, x):
        return x.detach().cpu().numpy()


class ShardedOptimizer:
    """The Main Iterative Loop of PAPER.md:99-114 over row slabs; `shard` is this rank's local shard."""

    def __init__(self, prob, shard, group=None, accepts=None, stop_test=None):
        import torch.distributed as dist
        self.dist, self.group, self.shard = dist, group, shard
        if accepts is None or stop_test is None:      # the library's own scalar decisions (pure host C functions)
            from paper_0908_4421_b200 import imrt_armijo_accepts, imrt_stop_test
            accepts, stop_test = accepts or imrt_armijo_accepts, stop_test or imrt_stop_test
        self.accepts, self.stop_test = accepts, stop_test
        self.eps, self.alpha, self.lambda0, self.max_ls = float(prob.eps), float(prob.alpha), float(prob.lambda0), int(prob.max_ls)

    # -- the two exchange steps
    def _sum_scalar(self, v: float) -> float:
        import torch
        t = torch.tensor([v], dtype=torch.float64, device=getattr(self.shard, "device", "cpu"))
        if self.dist.is_initialized() and self.dist.get_world_size(self.group) > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return float(t.item())

    def _sum_vector(self, g):
        if self.dist.is_initialized() and self.dist.get_world_size(self.group) > 1:
            self.dist.all_reduce(g, op=self.dist.ReduceOp.SUM, group=self.group)
        return g

    def run(self, x0, n_iters: int, delta: float = 0.0):
        sh = self.shard
        x = sh.vector(x0)
        G_k = self._sum_scalar(sh.eval_partial(x))
        obj, lams, trials, steps = [G_k], [], [], []
        reason = STOP_MAX_ITERS
        while len(lams) < n_iters:
            g = self._sum_vector(sh.grad_partial())                     # step 1
            if G_k == 0.0:
                reason = STOP_STATIONARY
                break
            lam, m, accepted = self.lambda0, 0, False                   # step 2
            while True:
                x_new, step_sq = sh.trial_point(x, g, lam)
                if m == 0 and step_sq == 0.0:
                    reason = STOP_STATIONARY
                    break
                G_new = self._sum_scalar(sh.eval_partial(x_new))
                if self.accepts(G_k, G_new, step_sq, self.eps, lam):    # step 3, Eq. (5)
                    accepted = True
                    break
                m += 1                                                  # step 4
                if m > self.max_ls:
                    reason = STOP_LS_STALLED
                    break
                lam = lam / self.alpha
            if not accepted:
                if reason == STOP_LS_STALLED:
                    sh.eval_partial(x)                                  # restore r(x_k) (x_k is kept)
                break
            G_old, G_k, x = G_k, G_new, x_new
            obj.append(G_new); lams.append(lam); trials.append(m + 1); steps.append(step_sq)
            if self.stop_test(G_old, G_new, delta):                     # step 5
                reason = STOP_TOLERANCE
                break
        self.x = x
        return ShardedTrace(len(lams), reason, np.asarray(obj), np.asarray(lams), np.asarray(trials, np.int32), np.asarray(steps))
