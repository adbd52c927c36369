"""Row-sharded driver (paper_0908_4421_b200/sharded.py): slab selection, the loop and its two
collectives under the gloo backend with world_size 2 on CPU (the local shards are oracle-backed stand-ins: the
library has no CPU path), and -- on a GPU -- two slabs of the real kernels adding up to the single-plan result."""
import os
import socket

import numpy as np
import pytest

import oracle
import synth_inputs
from paper_0908_4421_b200 import sharded
import host_sharded_loop as host_loop


class OracleShard:
    """CPU stand-in for GpuShard: the same three operations on a row slab, computed by the fp64 oracle."""
    device = "cpu"

    def __init__(self, sub):
        self.sub, self.r = sub, None

    def vector(self, x0):
        import torch
        return torch.from_numpy(np.asarray(x0, np.float64).copy())

    def eval_partial(self, x):
        _, self.r, G = oracle.eval_objective(self.sub, x.numpy())
        return G

    def grad_partial(self):
        import torch
        return torch.from_numpy(oracle.gradient(self.sub, self.r))

    def trial_point(self, x, g, lam):
        import torch
        xn, step = oracle.trial_point(x.numpy(), g.numpy(), lam)
        return torch.from_numpy(xn), step


def test_slabs_cover_the_rows_and_balance_the_nonzeros():
    prob = synth_inputs.make_phantom(0)
    for world in (1, 2, 3, 8):
        b = sharded.slab_bounds(prob.row_ptr, world)
        assert b[0] == 0 and b[-1] == prob.n_v and (np.diff(b) >= 0).all()
        nnz = np.diff(prob.row_ptr[b].astype(np.int64))
        assert nnz.sum() == prob.nnz and nnz.max() - nnz.min() <= 2 * np.diff(prob.row_ptr).max()
        rows = 0
        for q in range(world):
            sub, (r0, r1) = sharded.shard_rows(prob, world, q)
            assert sub.n_v == r1 - r0 and sub.row_ptr[0] == 0 and sub.row_ptr[-1] == sub.col.shape[0] == sub.val.shape[0]
            np.testing.assert_array_equal(sub.sid, prob.sid[r0:r1])
            rows += sub.n_v
        assert rows == prob.n_v
    # an empty matrix and more ranks than rows
    empty = synth_inputs.Problem("e", 3, 2, np.zeros(4, np.int32), np.zeros(0, np.int32), np.zeros(0, np.float32), np.zeros(3, np.uint8),
                                 prob.t_under, prob.t_over, prob.w_under, prob.w_over, np.ones(2, np.float32))
    b = sharded.slab_bounds(empty.row_ptr, 5)
    assert b[0] == 0 and b[-1] == 3 and (np.diff(b) >= 0).all()


def _worker(rank, world, port, n_iters, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        prob = synth_inputs.make_phantom(0)
        sub, _ = sharded.shard_rows(prob, world, rank)
        opt = host_loop.ShardedOptimizer(prob, OracleShard(sub))
        tr = opt.run(prob.x0, n_iters)
        out[rank] = (tr.n_iters, tr.stop_reason, tr.obj.tolist(), tr.lam.tolist(), tr.n_trials.tolist(), opt.x.numpy().tolist())
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_reproduce_the_single_process_loop():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    n_iters, world = 12, 2
    out = mp.Manager().dict()
    mp.spawn(_worker, args=(world, port, n_iters, out), nprocs=world, join=True)
    prob = synth_inputs.make_phantom(0)
    ref = oracle.run(prob, n_iters=n_iters)
    assert set(out.keys()) == {0, 1}
    for rank in (0, 1):
        n, reason, obj, lam, trials, x = out[rank]
        assert n == ref.n_iters == n_iters and reason == ref.stop_reason
        assert trials == ref.n_trials.tolist() and lam == ref.lam.tolist()
        np.testing.assert_allclose(obj, ref.obj, rtol=1e-12)          # the partial sums are added in another order
        np.testing.assert_allclose(x, ref.x, rtol=1e-9, atol=1e-12)
    assert out[0] == out[1]                                           # the iterates stay replicated, bit for bit


def test_stationary_and_tolerance_exits_without_a_process_group():
    prob = synth_inputs.make_phantom(0)
    opt = host_loop.ShardedOptimizer(prob, OracleShard(prob))
    tr = opt.run(prob.x0, 400, delta=1e-3)
    ref = oracle.run(prob, n_iters=400, delta=1e-3)
    assert tr.stop_reason == host_loop.STOP_TOLERANCE == ref.stop_reason and tr.n_iters == ref.n_iters
    np.testing.assert_array_equal(tr.obj, ref.obj)                    # one slab: the very same arithmetic
    T = np.array([10.0, 20.0, 30.0], np.float32)
    ident = synth_inputs.Problem("ident", 3, 3, np.array([0, 1, 2, 3], np.int32), np.array([0, 1, 2], np.int32), np.ones(3, np.float32),
                                 np.array([0, 1, 2], np.uint8), T, T, np.ones(3, np.float32), np.ones(3, np.float32),
                                 np.array([12.0, 16.0, 30.0], np.float32), eps=0.2, alpha=2.0, lambda0=1.0)
    tr = host_loop.ShardedOptimizer(ident, OracleShard(ident)).run(ident.x0, 5)
    assert tr.n_iters == 1 and tr.stop_reason == host_loop.STOP_STATIONARY and tr.obj.tolist() == [20.0, 0.0] and tr.n_trials.tolist() == [2]


class _TwoSlabs:
    """Two GpuShards on one device whose partials are added here: what the all-reduce does across two GPUs."""

    def __init__(self, prob, device):
        self.a = host_loop.GpuShard(sharded.shard_rows(prob, 2, 0)[0], device)
        self.b = host_loop.GpuShard(sharded.shard_rows(prob, 2, 1)[0], device)
        self.device = self.a.device

    def vector(self, x0):
        return self.a.vector(x0)

    def eval_partial(self, x):
        return self.a.eval_partial(x) + self.b.eval_partial(x)

    def grad_partial(self):
        return self.a.grad_partial() + self.b.grad_partial()

    def trial_point(self, x, g, lam):
        return self.a.trial_point(x, g, lam)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [0, 2])
def test_two_slabs_of_the_cuda_path_add_up(cfg):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_0908_4421_b200 as m
    prob = synth_inputs.make_phantom(cfg)
    n = 15
    plan = m.Plan(prob, max_iters=n)
    plan.set_x(prob.x0)
    plan.run_iters(n)
    tr1 = plan.trace()
    one = host_loop.ShardedOptimizer(prob, host_loop.GpuShard(prob, "cuda:0")).run(prob.x0, n)
    two = host_loop.ShardedOptimizer(prob, _TwoSlabs(prob, "cuda:0")).run(prob.x0, n)
    for tr in (one, two):
        assert tr.n_iters == n
        np.testing.assert_array_equal(tr.n_trials, tr1.n_trials)
        np.testing.assert_array_equal(tr.lam, tr1.lam)
        np.testing.assert_allclose(tr.obj, tr1.obj, rtol=2e-5)     # other slabs, other summation order in fp32: the per-kernel tolerance
    fol = oracle.run(prob, n_iters=n, follow_trials=two.n_trials, tau_rel=1e-6)
    assert fol.n_follow_violations == 0 and abs(two.obj[-1] - fol.obj[-1]) <= 1e-4 * fol.obj[-1]
    plan.close()


def test_no_rank_is_left_without_rows():
    # a few rows hold most of the non-zeros: equal-nnz cuts would leave ranks empty; every rank still gets >= 1 row
    rp = np.array([0, 1000, 1000, 1001, 1002, 1003, 1004], np.int64)
    for world in (2, 3, 6):
        b = sharded.slab_bounds(rp, world)
        assert b[0] == 0 and b[-1] == 6 and (np.diff(b) >= 1).all(), b
    prob = synth_inputs.make_phantom(0)
    small = synth_inputs.Problem("two-rows", 2, 3, np.array([0, 1, 2], np.int32), np.array([0, 1], np.int32), np.ones(2, np.float32),
                                 np.zeros(2, np.uint8), prob.t_under, prob.t_over, prob.w_under, prob.w_over, np.ones(3, np.float32))
    with pytest.raises(ValueError):
        sharded.shard_rows(small, 3, 2)              # more ranks than rows: refused on every rank alike, before any collective


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,world,n", [(0, 2, 30), (2, 2, 60), (2, 4, 60), (1, 3, 40), (3, 2, 30)])      # (3, ...): the headline size
def test_device_resident_sharded_loop_co_resident_ranks(cfg, world, n):
    # The row-sharded loop INSIDE the persistent kernel (exchange of g per iteration and of the R objectives per batch through
    # the ranks' inboxes): `world` ranks co-resident on one device, one cooperative launch (imrt_plan_run_ranks).
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_0908_4421_b200 as m
    prob = synth_inputs.make_phantom(cfg)
    ranks = sharded.CoResidentRanks(prob, world, max_iters=n)
    ranks.set_x(prob.x0)
    ranks.run_iters(n // 2)
    ranks.run_iters(n - n // 2)                      # resumable: sequence numbers and inboxes carry over between launches
    traces = [ranks.trace(q) for q in range(world)]
    tr = traces[0]
    assert tr.n_iters == n and tr.stop_reason == oracle.STOP_MAX_ITERS
    for q in range(1, world):                        # the ranks hold the same bits: same sums, same order, same decisions
        np.testing.assert_array_equal(traces[q].obj, tr.obj)
        np.testing.assert_array_equal(traces[q].n_trials, tr.n_trials)
        np.testing.assert_array_equal(traces[q].step_sq, tr.step_sq)
        np.testing.assert_array_equal(ranks.get_x(q).cpu().numpy(), ranks.get_x(0).cpu().numpy())
    # against the oracle on the WHOLE problem, follow mode
    fol = oracle.run(prob, n_iters=n, follow_trials=tr.n_trials, tau_rel=1e-6)
    assert fol.n_follow_violations == 0
    np.testing.assert_array_equal(tr.lam, fol.lam)
    assert (np.abs(tr.obj - fol.obj) <= 1e-4 * fol.obj).all()      # every entry of the trace, relative to itself
    d = ranks.get_dose().cpu().numpy().astype(np.float64)
    d_o = oracle.eval_objective(prob, fol.x)[0]
    assert np.abs(d - d_o).max() <= 0.005 * 70.0
    # and against the single-plan loop of the same library: same trial counts
    plan = m.Plan(prob, max_iters=n)
    plan.set_x(prob.x0)
    plan.run_iters(n)
    np.testing.assert_array_equal(plan.trace().n_trials, tr.n_trials)
    np.testing.assert_allclose(plan.trace().obj, tr.obj, rtol=2e-5)
    plan.close()
    ranks.close()


@pytest.mark.gpu
def test_sharded_run_to_tolerance_and_refusals():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_0908_4421_b200 as m
    prob = synth_inputs.make_phantom(0)
    ranks = sharded.CoResidentRanks(prob, 2, max_iters=400)
    ranks.set_x(prob.x0)
    ranks.run_to_tol(1e-3, 400)
    tr = ranks.trace()
    ref = oracle.run(prob, n_iters=400, delta=1e-3)
    assert tr.stop_reason == oracle.STOP_TOLERANCE and abs(tr.n_iters - ref.n_iters) <= 1
    with pytest.raises(m.ImrtError):                 # a rank of a sharded problem cannot run alone on this device's stream
        m.imrt_plan_run_ranks([ranks.plans[0].handle], 1)
    ranks.close()
    solo = m.Plan(prob, max_iters=4, driver=m.DRIVER_GRAPH)
    with pytest.raises(m.ImrtError):
        m.imrt_plan_set_shard(solo.handle, 0, 2, [16, 32])           # persistent driver only
    solo.close()


@pytest.mark.gpu
def test_a_lost_peer_ends_the_run_with_a_status_instead_of_hanging_the_device():
    # SURVEY.md section 5 (failure detection): every wait inside the persistent kernel is bounded (imrt_options.spin_timeout_ms).
    # Rank 0 of a 2-rank group is launched ALONE (imrt_plan_run_iters on one plan of the pair): its peer never pushes a partial
    # sum, so rank 0 must give up after the bound, report IMRT_STOP_PEER_TIMEOUT and refuse to run on until it is set up again.
    import time
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_0908_4421_b200 as m
    prob = synth_inputs.make_phantom(0)
    ranks = sharded.CoResidentRanks(prob, 2, max_iters=20, spin_timeout_ms=300)
    ranks.set_x(prob.x0)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ranks.plans[0].run_iters(5)                          # the peer's CTAs are not in this launch
    tr = ranks.plans[0].trace()                          # synchronises
    waited = time.perf_counter() - t0
    assert m.STOP_NAMES[tr.stop_reason] == "PEER_TIMEOUT" and tr.n_iters == 0
    assert 0.25 <= waited < 5.0, waited
    ranks.plans[0].run_iters(5)                          # refused on the device, at once: the iterate is not valid any more
    t1 = time.perf_counter()
    tr = ranks.plans[0].trace()
    assert m.STOP_NAMES[tr.stop_reason] == "PEER_TIMEOUT" and tr.n_iters == 0 and time.perf_counter() - t1 < 0.2
    # the give-up was written into the peer's inbox as well: launched now, rank 1 stops at once rather than after its own bound
    t2 = time.perf_counter()
    ranks.plans[1].run_iters(5)
    tr1 = ranks.plans[1].trace()
    assert m.STOP_NAMES[tr1.stop_reason] == "PEER_TIMEOUT" and time.perf_counter() - t2 < 0.2
    # recovery: zero the inboxes, set the group up again, set x -- and the pair runs as if nothing had happened
    for box in ranks.inboxes:
        box.zero_()
    ptrs = [t.data_ptr() for t in ranks.inboxes]
    for q, p in enumerate(ranks.plans):
        m.imrt_plan_set_shard(p.handle, q, 2, ptrs)
    ranks.set_x(prob.x0)
    ranks.run_iters(20)
    tr = ranks.trace()
    fresh = sharded.CoResidentRanks(prob, 2, max_iters=20)
    fresh.set_x(prob.x0)
    fresh.run_iters(20)
    assert tr.n_iters == 20 and tr.stop_reason == oracle.STOP_MAX_ITERS
    np.testing.assert_array_equal(tr.obj, fresh.trace().obj)
    np.testing.assert_array_equal(ranks.get_x().cpu().numpy(), fresh.get_x().cpu().numpy())
    # a refused imrt_plan_set_shard (misaligned inbox) changes nothing: the group still runs
    with pytest.raises(m.ImrtError):
        m.imrt_plan_set_shard(ranks.plans[0].handle, 0, 2, [ptrs[0], ptrs[1] + 4])
    # ranks that disagree on the trace capacity are refused before anything is launched
    odd = sharded.CoResidentRanks(prob, 2, max_iters=21)
    odd.set_x(prob.x0)
    with pytest.raises(m.ImrtError):
        m.imrt_plan_run_ranks([fresh.plans[0].handle, odd.plans[1].handle], 1)
    for r in (ranks, fresh, odd):
        r.close()
