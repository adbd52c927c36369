"""GPU parity: libimrtgp (through its C-ABI binding) against the fp64 CPU oracle, element by element.

Tolerances (BASELINE.json north_star):
  per-kernel   d, r, g: ||a-b||_inf / ||b||_inf and ||a-b||_2 / ||b||_2 <= 1e-5;  G: |a-b|/|b| <= 1e-5
  trajectory   same accepted-iteration count, oracle in follow mode (slack 1e-6 G_k on the Armijo margin):
               final G within 1e-4 relative; DVH points within 0.5 % of the 70 Gy prescription (0.35 Gy)
"""
import numpy as np
import pytest

import oracle
import synth_inputs

pytestmark = pytest.mark.gpu

TOL_KERNEL = 1e-5
TOL_G_FINAL = 1e-4
TOL_DVH_GY = 0.005 * 70.0


@pytest.fixture(scope="module")
def m():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_0908_4421_b200 as mod
    mod.lib()
    return mod


_phantoms = {}


def phantom(i):
    if i not in _phantoms:
        _phantoms[i] = synth_inputs.make_phantom(i)
    return _phantoms[i]


def relerr(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    ninf = np.abs(b).max() if b.size else 0.0
    n2 = np.linalg.norm(b)
    einf = np.abs(a - b).max() / ninf if ninf > 0 else np.abs(a - b).max(initial=0.0)
    e2 = np.linalg.norm(a - b) / n2 if n2 > 0 else np.linalg.norm(a - b)
    return max(einf, e2)


def check_eval(m, plan, prob, x):
    d, r, g, G = plan.eval(x)
    x64 = np.asarray(x, np.float32).astype(np.float64)
    d_o, r_o, G_o = oracle.eval_objective(prob, x64)
    g_o = oracle.gradient(prob, r_o)
    dn = d.cpu().numpy().astype(np.float64)
    assert relerr(dn, d_o) <= TOL_KERNEL
    # d is a one-signed sum: also element by element, relative to the element itself (floor: 1e-3 of the largest dose), so
    # that a wrong short row at a field edge cannot hide behind the 70 Gy core
    floor = 1e-3 * np.abs(d_o).max() if d_o.size else 0.0
    assert (np.abs(dn - d_o) <= TOL_KERNEL * np.maximum(np.abs(d_o), floor)).all(), \
        "dose row %d off by %.3e" % (int(np.argmax(np.abs(dn - d_o) / np.maximum(np.abs(d_o), floor + 1e-300))), np.abs(dn - d_o).max())
    assert relerr(r.cpu().numpy(), r_o) <= TOL_KERNEL
    assert relerr(g.cpu().numpy(), g_o) <= TOL_KERNEL
    assert abs(G - G_o) <= TOL_KERNEL * abs(G_o) + 1e-300
    # the transpose kernel ALONE (a4 isolated from a2 / a3): it is fed the ORACLE's residual, rounded to fp32, and compared
    # with the oracle's gradient of that same rounded residual -- a compensating error in the penalty and the transpose
    # pass cannot pass this
    r32 = r_o.astype(np.float32)
    g_alone = plan.gradient(r32).cpu().numpy()
    assert relerr(g_alone, oracle.gradient(prob, r32.astype(np.float64))) <= TOL_KERNEL
    return d, r, g, G


def check_eval_batch(m, plan, prob, xs):
    """The line search's batched pass (the R = len(xs) kernels bench.py times) on given points: every residual vector
    and every objective against the oracle."""
    xs = np.ascontiguousarray(xs, np.float32)
    r, G = plan.eval_batch(xs)
    r = r.cpu().numpy()
    for j in range(xs.shape[0]):
        d_o, r_o, G_o = oracle.eval_objective(prob, xs[j].astype(np.float64))
        assert relerr(r[j], r_o) <= TOL_KERNEL, j
        assert abs(G[j] - G_o) <= TOL_KERNEL * abs(G_o) + 1e-300, j


def trial_points(prob, x, n):
    """The first n trial points of the line search at x, computed by the oracle."""
    x64 = np.asarray(x, np.float32).astype(np.float64)
    _, r_o, _ = oracle.eval_objective(prob, x64)
    g_o = oracle.gradient(prob, r_o)
    return np.stack([oracle.trial_point(x64, g_o, prob.lambda0 / prob.alpha ** j)[0] for j in range(n)]).astype(np.float32)


# ---------------------------------------------------------------------------------------------- D^T construction
@pytest.mark.parametrize("case", ["cfg0", "rand_a", "rand_b"])
def test_transpose_csr_is_exact(m, case):
    import scipy.sparse as sp
    prob = phantom(0) if case == "cfg0" else synth_inputs.make_random(7 if case == "rand_a" else 8, n_v=777, n_b=53,
                                                                      density=0.3, empty_row_frac=0.2, full_rows=3)
    plan = m.Plan(prob, max_iters=4)
    rpT, cT, vT = (t.cpu().numpy() for t in plan.transpose_csr())
    A = sp.csr_matrix((prob.val, prob.col, prob.row_ptr), shape=(prob.n_v, prob.n_b))
    T = A.T.tocsr()
    T.sort_indices()
    np.testing.assert_array_equal(rpT, T.indptr)
    np.testing.assert_array_equal(cT, T.indices)
    np.testing.assert_array_equal(vT, T.data)
    plan.close()


# ---------------------------------------------------------------------------------------------- per-kernel parity
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_eval_parity_phantoms(m, cfg):
    prob = phantom(cfg)
    plan = m.Plan(prob, max_iters=8)
    check_eval(m, plan, prob, prob.x0)
    # also at the oracle's iterate after 1 and 10 iterations (x rounded to fp32 is what both sides see)
    for n in (1, 10):
        xo = oracle.run(prob, n_iters=n).x.astype(np.float32)
        check_eval(m, plan, prob, xo)
    # the batched pass: the four trial points of the first line search, then two
    check_eval_batch(m, plan, prob, trial_points(prob, prob.x0, 4))
    check_eval_batch(m, plan, prob, trial_points(prob, xo, 2))
    plan.close()


def test_penalty_alone_on_identity_matrix(m):
    # a3 isolated from a2: with D = I the dose IS x (exactly, in fp32), so r and G test Eq. (1) / its gradient factor alone
    n = 5003
    rng = np.random.default_rng(3)
    base = synth_inputs.make_random(1, n_v=50, n_b=8)
    sid = rng.integers(0, 3, n).astype(np.uint8)
    prob = synth_inputs.Problem("ident-n", n, n, np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), np.ones(n, np.float32),
                                sid, base.t_under, base.t_over, base.w_under, base.w_over, np.ones(n, np.float32))
    plan = m.Plan(prob, max_iters=2)
    x = rng.uniform(0, 90, n).astype(np.float32)
    d, r, g, G = plan.eval(x)
    np.testing.assert_array_equal(d.cpu().numpy(), x)
    d_o, r_o, G_o = oracle.eval_objective(prob, x.astype(np.float64))
    assert np.abs(r.cpu().numpy() - r_o).max() <= 1e-6 * np.abs(r_o).max()      # one fp32 rounding or two per element
    assert abs(G - G_o) <= 1e-6 * G_o                                           # fp64 accumulation of fp32 u, o
    check_eval_batch(m, plan, prob, np.stack([x, 0.5 * x, 2 * x, np.zeros_like(x)]))
    plan.close()


@pytest.mark.parametrize("seed,n_v,n_b,density", [(1, 50, 8, 0.4), (2, 1000, 37, 0.3), (3, 4099, 130, 0.5), (4, 30000, 300, 0.2),
                                                   (5, 3, 1, 1.0), (6, 2500, 2000, 0.02)])
def test_eval_parity_random_shapes(m, seed, n_v, n_b, density):
    # ragged shapes: nnz not a multiple of 4, empty / single-entry / full rows, short D^T rows, one-column matrices
    prob = synth_inputs.make_random(seed, n_v=n_v, n_b=n_b, density=density, empty_row_frac=0.15, full_rows=min(2, n_v))
    plan = m.Plan(prob, max_iters=4)
    x = np.random.default_rng(seed).uniform(0, 80, prob.n_b).astype(np.float32)
    check_eval(m, plan, prob, x)
    check_eval(m, plan, prob, np.zeros(prob.n_b, np.float32))
    plan.close()


def test_eval_all_rows_empty_and_leading_trailing_empty(m):
    rng = np.random.default_rng(0)
    base = synth_inputs.make_random(11, n_v=600, n_b=20, density=0.3)
    # 500 empty rows in front and behind
    rp = np.concatenate([np.zeros(500, np.int32), base.row_ptr, np.full(500, base.row_ptr[-1], np.int32)])
    sid = np.concatenate([rng.integers(0, 3, 500).astype(np.uint8), base.sid, rng.integers(0, 3, 500).astype(np.uint8)])
    prob = synth_inputs.Problem("padded", 1600, 20, rp, base.col, base.val, sid, base.t_under, base.t_over, base.w_under,
                                base.w_over, base.x0, lambda0=base.lambda0)
    plan = m.Plan(prob, max_iters=4)
    check_eval(m, plan, prob, prob.x0)   # zero-dose PTV rows contribute w- T^2 each and a constant residual
    plan.close()
    empty = synth_inputs.Problem("empty", 100, 5, np.zeros(101, np.int32), np.zeros(0, np.int32), np.zeros(0, np.float32),
                                 sid[:100], base.t_under, base.t_over, base.w_under, base.w_over, np.ones(5, np.float32))
    plan = m.Plan(empty, max_iters=4)
    d, r, g, G = plan.eval(empty.x0)
    d_o, r_o, G_o = oracle.eval_objective(empty, empty.x0.astype(np.float64))
    assert G == G_o and not d.cpu().numpy().any() and not g.cpu().numpy().any()
    np.testing.assert_array_equal(r.cpu().numpy(), r_o.astype(np.float32))
    plan.set_x(empty.x0)
    plan.run_iters(3)
    tr = plan.trace()
    assert tr.n_iters == 0 and tr.stop_reason == oracle.STOP_STATIONARY   # zero gradient: first trial equals x_k
    plan.close()


# ---------------------------------------------------------------------------------------------- the loop
def run_gpu(m, prob, n_iters, driver, delta=0.0, ls_batch=0, **options):
    plan = m.Plan(prob, max_iters=max(n_iters, 1), driver=driver, ls_batch=ls_batch, **options)
    plan.set_x(prob.x0)
    if delta > 0:
        plan.run_to_tol(delta, n_iters)
    else:
        plan.run_iters(n_iters)
    tr = plan.trace()
    x = plan.get_x().cpu().numpy()
    d = plan.get_dose().cpu().numpy()
    cnt = plan.counters()
    return plan, tr, x, d, cnt


def test_three_drivers_are_bit_identical(m):
    # plans are compared with each other: tune_level 0 (the default) gives every plan of a problem the same partition
    prob = phantom(0)
    res = [run_gpu(m, prob, 25, drv) for drv in (m.DRIVER_HOST, m.DRIVER_GRAPH, m.DRIVER_PERSISTENT)]
    _, tr0, x0, d0, c0 = res[0]
    assert tr0.n_iters == 25 and tr0.n_trials.max() > 1
    for _, tr, x, d, c in res[1:]:
        assert tr.n_iters == tr0.n_iters and tr.stop_reason == tr0.stop_reason
        np.testing.assert_array_equal(tr.obj, tr0.obj)
        np.testing.assert_array_equal(tr.n_trials, tr0.n_trials)
        np.testing.assert_array_equal(tr.lam, tr0.lam)
        np.testing.assert_array_equal(tr.step_sq, tr0.step_sq)
        np.testing.assert_array_equal(x, x0)
        np.testing.assert_array_equal(d, d0)
        assert c == c0
    for r in res:
        r[0].close()


@pytest.mark.parametrize("cfg,n", [(0, 50), (2, 40)])
def test_batched_line_search_is_bit_identical_to_sequential(m, cfg, n):
    # Plans are compared with each other, so they must share one CTA partition: the measured rebalancing of plan
    # creation (timing dependent; it changes the order in which objective partials are summed) stays off (tune_level 0).
    # imrt_params.ls_batch: 1 = one trial point per pass over D (steps 2-4 of PAPER.md:109-111 literally), 2 / 4 = the
    # next 2 / 4 trial points in one pass.  Same iterates, objectives, step sizes and trial counts, bit for bit.
    prob = phantom(cfg)
    res = {R: run_gpu(m, prob, n, m.DRIVER_PERSISTENT, ls_batch=R) for R in (1, 2, 4)}
    _, tr1, x1, d1, (fwd1, trp1) = res[1]
    assert tr1.n_iters == n and fwd1 == 1 + tr1.n_trials.sum() and tr1.n_trials.max() > 1
    for R in (2, 4):
        plan, tr, x, d, (fwd, trp) = res[R]
        assert plan.info()["ls_batch"] == R
        np.testing.assert_array_equal(tr.obj, tr1.obj)
        np.testing.assert_array_equal(tr.n_trials, tr1.n_trials)
        np.testing.assert_array_equal(tr.lam, tr1.lam)
        np.testing.assert_array_equal(tr.step_sq, tr1.step_sq)
        np.testing.assert_array_equal(x, x1)
        np.testing.assert_array_equal(d, d1)
        assert trp == trp1 and fwd == 1 + np.ceil(tr.n_trials / R).sum()
    for r in res.values():
        r[0].close()


def test_runs_are_reproducible_and_resumable(m):
    prob = phantom(0)
    p1, tr1, x1, _, _ = run_gpu(m, prob, 20, m.DRIVER_PERSISTENT)
    plan = m.Plan(prob, max_iters=20, driver=m.DRIVER_PERSISTENT)
    plan.set_x(prob.x0)
    plan.run_iters(7)
    plan.run_iters(13)   # 7 + 13 accepted iterations in two launches == 20 in one
    tr2 = plan.trace()
    np.testing.assert_array_equal(tr2.obj, tr1.obj)
    np.testing.assert_array_equal(plan.get_x().cpu().numpy(), x1)
    plan.run_iters(5)    # trace capacity reached: nothing more happens, and the caller is told why
    assert plan.trace().n_iters == 20 and m.STOP_NAMES[plan.trace().stop_reason] == "TRACE_FULL"
    p1.close()
    plan.close()


@pytest.mark.parametrize("cfg,driver", [(0, 2), (0, 0), (1, 2), (2, 2), (2, 0)])
def test_trajectory_parity_follow_mode(m, cfg, driver):
    # Every config at ITS OWN run length (SURVEY.md 8(d) "Run lengths"): cfg0 50 and cfg1 200 fixed iterations; cfg2 under its
    # rule "delta = 1e-6 or 500 iterations", compared at the GPU's own stopping count.  (cfg3 / cfg4: test_full_size_parity.)
    prob = phantom(cfg)
    plan, tr, x, d, (fwd, trp) = run_gpu(m, prob, prob.n_iters, driver, delta=prob.delta)
    n = tr.n_iters
    if prob.delta > 0:
        print("cfg%d: GPU stopped after %d iterations (%s)" % (cfg, n, m.STOP_NAMES[tr.stop_reason]))
        assert tr.stop_reason in (oracle.STOP_MAX_ITERS, oracle.STOP_TOLERANCE) and n > 100
    else:
        assert n == prob.n_iters and tr.stop_reason == oracle.STOP_MAX_ITERS
    R = plan.info()["ls_batch"]     # one dose pass evaluates up to R trial points
    assert fwd == 1 + np.ceil(tr.n_trials / R).sum()
    assert (np.diff(tr.obj) < 0).all() and (x >= 0).all()
    fol = oracle.run(prob, n_iters=n, follow_trials=tr.n_trials, tau_rel=1e-6)
    assert fol.n_follow_violations == 0, "GPU accepted/rejected a trial the oracle would not (first at iteration %d)" % fol.first_violation
    np.testing.assert_array_equal(tr.lam, fol.lam)
    assert abs(tr.obj[-1] - fol.obj[-1]) <= TOL_G_FINAL * fol.obj[-1]
    assert (np.abs(tr.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()
    # DVH points of the final plans
    d_o, _, _ = oracle.eval_objective(prob, fol.x)
    dp_o, mean_o = oracle.dvh_points(prob.sid, d_o, prob.n_structures)
    dp_g, mean_g = oracle.dvh_points(prob.sid, d.astype(np.float64), prob.n_structures)
    assert np.nanmax(np.abs(dp_g - dp_o)) <= TOL_DVH_GY and np.nanmax(np.abs(mean_g - mean_o)) <= TOL_DVH_GY
    # and the library's own DVH kernel gives exactly the order statistics of its own dose
    dp_k, mean_k = plan.dvh(oracle.DVH_PCTS)
    np.testing.assert_array_equal(dp_k, dp_g)
    np.testing.assert_allclose(mean_k, mean_g, rtol=1e-6)
    # free-running oracle: report where (if anywhere) the trial counts first part ways
    free = oracle.run(prob, n_iters=n)
    same = free.n_trials[:n] == tr.n_trials
    if not same.all():
        k = int(np.argmin(same))
        print("cfg%d: free-running oracle and GPU first differ in trial count at iteration %d (margin %.3e)" % (cfg, k, free.margin[k]))
    plan.close()


@pytest.mark.parametrize("cfg,delta", [(0, 1e-3), (1, 1e-3), (2, 3e-3), (2, 1e-3)])
def test_run_to_tolerance_matches_oracle_stop(m, cfg, delta):
    # step 5 (reading R5): the TOLERANCE exit fires on both sides, at the same iteration (+-1: the two
    # relative changes are compared with delta in different precisions)
    prob = phantom(cfg)
    plan, tr, x, d, _ = run_gpu(m, prob, 500, m.DRIVER_PERSISTENT, delta=delta)
    ref = oracle.run(prob, n_iters=500, delta=delta)
    assert tr.stop_reason == oracle.STOP_TOLERANCE and ref.stop_reason == oracle.STOP_TOLERANCE
    rel = np.abs(np.diff(tr.obj)) / tr.obj[1:]
    assert rel[-1] < delta and (rel[:-1] >= delta).all()
    assert abs(tr.n_iters - ref.n_iters) <= 1, (tr.n_iters, ref.n_iters)
    fol = oracle.run(prob, n_iters=tr.n_iters, follow_trials=tr.n_trials, tau_rel=1e-6)
    assert fol.n_follow_violations == 0 and abs(tr.obj[-1] - fol.obj[-1]) <= TOL_G_FINAL * fol.obj[-1]
    plan.close()


def test_identity_two_trials_then_stationary(m):
    # tests/golden/hand_cases.json "identity_two_trials", now through the CUDA path
    T = np.array([10.0, 20.0, 30.0], np.float32)
    prob = synth_inputs.Problem("ident", 3, 3, np.array([0, 1, 2, 3], np.int32), np.array([0, 1, 2], np.int32),
                                np.ones(3, np.float32), np.array([0, 1, 2], np.uint8), T, T, np.ones(3, np.float32),
                                np.ones(3, np.float32), np.array([12.0, 16.0, 30.0], np.float32), eps=0.2, alpha=2.0, lambda0=1.0)
    for drv in (0, 1, 2):
        for R in (1, 2, 4):
            plan, tr, x, d, (fwd, trp) = run_gpu(m, prob, 5, drv, ls_batch=R)
            assert tr.n_iters == 1 and tr.stop_reason == oracle.STOP_STATIONARY
            assert list(tr.obj) == [20.0, 0.0] and list(tr.n_trials) == [2] and list(tr.lam) == [0.5] and list(tr.step_sq) == [20.0]
            assert list(x) == [10.0, 20.0, 30.0] and fwd == (3 if R == 1 else 2) and trp == 2
            plan.close()


def test_linesearch_stall_and_bad_inputs(m):
    import torch
    T = np.array([5.0], np.float32)
    prob = synth_inputs.Problem("stall", 2, 2, np.array([0, 1, 2], np.int32), np.array([0, 1], np.int32), np.ones(2, np.float32),
                                np.zeros(2, np.uint8), T, T, np.ones(1, np.float32), np.ones(1, np.float32),
                                np.array([1.0, 9.0], np.float32), lambda0=1024.0, max_ls=2)
    for R in (1, 2, 4):
        plan, tr, x, d, (fwd, trp) = run_gpu(m, prob, 3, m.DRIVER_PERSISTENT, ls_batch=R)
        assert tr.n_iters == 0 and tr.stop_reason == oracle.STOP_LS_STALLED and fwd == 1 + {1: 3, 2: 2, 4: 1}[R]
        np.testing.assert_array_equal(x, prob.x0)
        if R < 4:
            plan.close()
    with pytest.raises(m.ImrtError) as e:
        plan.set_x(np.array([1.0, -1.0], np.float32))
    assert e.value.status_name == "BAD_X"
    plan.close()
    bad = synth_inputs.Problem(**{**prob.__dict__})
    bad.col = np.array([0, 2], np.int32)
    with pytest.raises(m.ImrtError) as e:
        m.Plan(bad)
    assert e.value.status_name == "BAD_CSR"
    bad = synth_inputs.Problem(**{**prob.__dict__})
    bad.row_ptr = np.array([0, 2, 1], np.int32)
    with pytest.raises(m.ImrtError) as e:
        m.Plan(bad)
    assert e.value.status_name == "BAD_CSR"
    dup = synth_inputs.Problem("dup", 2, 3, np.array([0, 2, 3], np.int32), np.array([1, 1, 0], np.int32), np.ones(3, np.float32),
                               np.zeros(2, np.uint8), T, T, np.ones(1, np.float32), np.ones(1, np.float32), np.ones(3, np.float32))
    with pytest.raises(m.ImrtError) as e:          # a repeated column (and, equally, descending columns)
        m.Plan(dup)
    assert e.value.status_name == "BAD_CSR"
    bad = synth_inputs.Problem(**{**prob.__dict__})
    bad.sid = np.array([0, 3], np.uint8)
    with pytest.raises(m.ImrtError) as e:
        m.Plan(bad)
    assert e.value.status_name == "BAD_STRUCTURE"
    bad = synth_inputs.Problem(**{**prob.__dict__})
    bad.val = np.array([1.0, np.inf], np.float32)
    with pytest.raises(m.ImrtError) as e:
        m.Plan(bad)
    assert e.value.status_name == "BAD_CSR"
    assert torch.cuda.is_available()


# (the full-size cases, cfg3 and cfg4, live in tests/test_zz_full_size.py: they take minutes and sort after the cheap tests)


# ---------------------------------------------------------------------------------------------- per-voxel limits
@pytest.mark.parametrize("cfg", [0, 2])
def test_per_voxel_limits_parity(m, cfg):
    # the paper's own model: every voxel has its own T_j (here the structure's limit perturbed per voxel, both sides,
    # including voxels whose row of D is empty: their constant penalty and residual must follow the per-voxel limits)
    import copy
    prob = copy.copy(phantom(cfg))
    rng = np.random.default_rng(100 + cfg)
    prob.tv_under = (prob.t_under[prob.sid] * rng.uniform(0.9, 1.1, prob.n_v)).astype(np.float32)
    prob.tv_over = (prob.t_over[prob.sid] * rng.uniform(0.9, 1.1, prob.n_v)).astype(np.float32)
    plan = m.Plan(prob, max_iters=20)
    check_eval(m, plan, prob, prob.x0)
    plan.set_x(prob.x0)
    plan.run_iters(20)
    tr = plan.trace()
    fol = oracle.run(prob, n_iters=20, follow_trials=tr.n_trials, tau_rel=1e-6)
    assert tr.n_iters == 20 and fol.n_follow_violations == 0
    assert (np.abs(tr.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()
    # back to per-structure limits: the plan behaves as if the call had never happened
    plan.set_voxel_limits(None, None)
    base = phantom(cfg)
    check_eval(m, plan, base, base.x0)
    # only the upper limits per voxel
    half = copy.copy(base)
    half.tv_over = prob.tv_over
    plan.set_voxel_limits(None, half.tv_over)
    check_eval(m, plan, half, half.x0)
    with pytest.raises(m.ImrtError):
        plan.run_iters(1)                 # the iterate was invalidated: set_x first
    plan.close()


# ---------------------------------------------------------------------------------------------- the fallback layouts
@pytest.mark.parametrize("opt", [{"dose_format": 1}, {"col_bits": 32}, {"transpose_format": 1}, {"transpose_format": 2},
                                 {"tune_level": 1}, {"tune_level": 2}, {"quad_cap": 64}])
def test_fallback_layouts_parity(m, opt):
    # the layouts a plan falls back to when the matrix does not suit the packed ones: row-format records everywhere,
    # 32-bit column indices (n_b > 65,536), single rows of D^T instead of row pairs, the 32-bit D^T stream (a group of 32
    # entries wider than 65,535 voxels); the measured partitions; small records --
    # forced here through imrt_options
    for prob in (phantom(0), phantom(1),
                 synth_inputs.make_random(21, n_v=4099, n_b=130, density=0.5, empty_row_frac=0.15, full_rows=2)):
        plan = m.Plan(prob, max_iters=12, **opt)
        info = plan.info()
        if opt.get("dose_format") == 1:
            assert info["quad_rows"] == 0
        if opt.get("col_bits") == 32:
            assert info["col16"] == 0 and info["quad_rows"] == 0
        if opt.get("transpose_format") == 1:
            assert info["tr_format"] == 1
        if opt.get("transpose_format") == 2:
            assert info["tr_format"] == 0
        x = np.random.default_rng(5).uniform(0, 60, prob.n_b).astype(np.float32)
        check_eval(m, plan, prob, x)
        plan.set_x(prob.x0)
        plan.run_iters(12)
        tr = plan.trace()
        fol = oracle.run(prob, n_iters=12, follow_trials=tr.n_trials, tau_rel=1e-6)
        assert tr.n_iters == fol.n_iters and fol.n_follow_violations == 0
        assert (np.abs(tr.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()
        plan.close()


@pytest.mark.parametrize("seed,n_quads,n_b,tail", [(1, 1, 40, 0), (2, 2, 64, 1), (3, 3, 300, 2), (4, 257, 512, 3), (5, 4001, 900, 0),
                                                     (6, 1500, 2304, 1)])
def test_quad_pairs_edge_cases(m, seed, n_quads, n_b, tail):
    # The dose pass takes the quads of a record two at a time (one per half-warp): single quads, odd counts, an
    # incomplete last group, empty groups between long ones, neighbours of very different length, rows without entries.
    prob = synth_inputs.make_quad_blocks(seed, n_quads, n_b, tail)
    x = np.random.default_rng(seed).uniform(0, 3, prob.n_b).astype(np.float32)
    ref = None
    for R in (4, 2, 1):
        plan = m.Plan(prob, max_iters=8, ls_batch=R)
        if n_quads >= 100:
            assert plan.info()["quad_rows"] > 0          # the case really exercises the quad records
        check_eval(m, plan, prob, x)
        check_eval_batch(m, plan, prob, np.stack([x * f for f in (1.0, 0.5, 0.25, 0.0)][:R]))
        plan.set_x(prob.x0)
        plan.run_iters(8)
        tr = plan.trace()
        x_end = plan.get_x().cpu().numpy()
        assert (np.diff(tr.obj) < 0).all() and (x_end >= 0).all()
        # the loop's own (batched) dose pass against the oracle at the point it ended in (trajectories themselves are
        # compared on the phantoms: reading R15)
        G_o = oracle.eval_objective(prob, x_end.astype(np.float64))[2]
        assert abs(tr.obj[-1] - G_o) <= TOL_KERNEL * abs(G_o) + 1e-300
        cur = (tr.obj.copy(), x_end)
        if ref is not None:                               # every batch width: the same bits
            np.testing.assert_array_equal(cur[0], ref[0])
            np.testing.assert_array_equal(cur[1], ref[1])
        ref = cur
        plan.close()


def test_wide_transpose_groups_use_the_32_bit_stream(m):
    # a beamlet whose voxels lie more than 65,535 rows apart inside one group of 32 entries: no 16-bit offsets possible
    n_v, n_b = 200000, 6
    rows = np.arange(0, n_v, 2500)                     # 80 rows, 2,500 apart: 32 consecutive entries span 77,500 voxels
    rp = np.zeros(n_v + 1, np.int32)
    rp[rows + 1] = n_b
    rp = np.cumsum(rp).astype(np.int32)
    rng = np.random.default_rng(9)
    col = np.tile(np.arange(n_b, dtype=np.int32), rows.shape[0])
    val = rng.uniform(0.1, 1.0, col.shape[0]).astype(np.float32)
    sid = (np.arange(n_v) % 3).astype(np.uint8)
    base = synth_inputs.make_random(1, n_v=50, n_b=8)
    prob = synth_inputs.Problem("wide", n_v, n_b, rp, col, val, sid, base.t_under, base.t_over, base.w_under, base.w_over,
                                rng.uniform(0.5, 1.5, n_b).astype(np.float32))
    prob.lambda0, _ = synth_inputs.pick_lambda0(rp, col, val, sid, base.w_under, base.w_over)
    plan = m.Plan(prob, max_iters=8)
    assert plan.info()["tr_format"] == 0
    check_eval(m, plan, prob, prob.x0 * 30)
    plan.set_x(prob.x0)
    plan.run_iters(8)
    tr = plan.trace()
    fol = oracle.run(prob, n_iters=8, follow_trials=tr.n_trials, tau_rel=1e-6)
    assert fol.n_follow_violations == 0 and (np.abs(tr.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()
    plan.close()


# ---------------------------------------------------------------------------------------------- mixed resolution
def test_mixed_resolution_workflow(m):
    # "For unspecified tissue we increased the voxel size in each dimension by a factor of 2 ... The full resolution was
    # used when evaluating the treatment quality": optimise on the mixed-resolution matrix, evaluate dose and DVH with a
    # second plan on the full-resolution matrix.  (The row merging is input preparation: synth_inputs.mixed_resolution.)
    import copy
    import torch
    fine = phantom(1)
    # the merge is a library call (imrt_merge_rows_count / _fill): bit-exact against the oracle's plain merge
    group, n_groups, sid_g = synth_inputs.mixed_resolution_groups(fine)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    m_rp, m_col, m_val = m.imrt_merge_rows(fine.n_b, dev(fine.row_ptr), dev(fine.col), dev(fine.val), dev(group), n_groups)
    o_rp, o_col, o_val = oracle.merge_rows(fine.n_b, fine.row_ptr, fine.col, fine.val, group, n_groups)
    np.testing.assert_array_equal(m_rp.cpu().numpy(), o_rp)
    np.testing.assert_array_equal(m_col.cpu().numpy(), o_col)
    np.testing.assert_array_equal(m_val.cpu().numpy(), o_val)
    mixed = copy.copy(fine)
    mixed.name, mixed.n_v, mixed.sid, mixed.voxel_ids = fine.name + "-mixed", n_groups, sid_g, None
    mixed.row_ptr, mixed.col, mixed.val = m_rp.cpu().numpy(), m_col.cpu().numpy(), m_val.cpu().numpy()
    mixed.lambda0, _ = synth_inputs.pick_lambda0(mixed.row_ptr, mixed.col, mixed.val, mixed.sid, mixed.w_under, mixed.w_over)
    assert mixed.n_v < fine.n_v // 4 and int((sid_g != 3).sum()) == int((fine.sid != 3).sum())
    n = 40
    plan = m.Plan(mixed, max_iters=n)
    check_eval(m, plan, mixed, mixed.x0)
    plan.set_x(mixed.x0)
    plan.run_iters(n)
    tr = plan.trace()
    fol = oracle.run(mixed, n_iters=n, follow_trials=tr.n_trials, tau_rel=1e-6)
    assert tr.n_iters == n and fol.n_follow_violations == 0
    assert (np.abs(tr.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()
    x = plan.get_x()
    # full-resolution evaluation of that plan
    full = m.Plan(fine, max_iters=1)
    d, r, g, G = full.eval(x)
    d_o, r_o, G_o = oracle.eval_objective(fine, x.cpu().numpy().astype(np.float64))
    assert relerr(d.cpu().numpy(), d_o) <= TOL_KERNEL and abs(G - G_o) <= TOL_KERNEL * G_o
    full.set_x(x)
    dp_g, mean_g = full.dvh(oracle.DVH_PCTS)
    dp_o, mean_o = oracle.dvh_points(fine.sid, d_o, fine.n_structures)
    assert np.nanmax(np.abs(dp_g - dp_o)) <= TOL_DVH_GY and np.nanmax(np.abs(mean_g - mean_o)) <= TOL_DVH_GY
    plan.close()
    full.close()


# ---------------------------------------------------------------------------------------------- randomised shapes
def test_randomised_shapes_layouts_batches_and_drivers(m):
    # 36 seeded problems: banded (neighbouring rows overlap: quad records), unstructured, with per-voxel limits; sizes from
    # 7 rows to 60,000, 1 to 2,500 beamlets, empty-row fractions up to 70 %; every batch width and driver.  Per-kernel
    # parity at a random x; the loop must run, decrease the objective and stay feasible.  (Trajectory parity needs a
    # problem that has not converged to machine precision -- reading R15 -- and is covered on the phantoms.)
    rng = np.random.default_rng(2024)
    for case in range(36):
        seed = int(rng.integers(1 << 30))
        n_v = int(rng.choice([7, 130, 1000, 5000, 20000, 60000]))
        n_b = int(rng.choice([1, 5, 33, 200, 700, 2500]))
        if case % 3 == 1:
            prob = synth_inputs.make_random(seed, n_v=min(n_v, 20000), n_b=n_b, density=float(rng.choice([0.02, 0.2, 0.6])),
                                            empty_row_frac=float(rng.choice([0.0, 0.3])), full_rows=int(rng.integers(0, 3)))
        else:
            prob = synth_inputs.make_banded(seed, n_v, n_b, width=int(rng.choice([3, 20, 90, 400])),
                                            jitter=float(rng.choice([0.3, 2.0, 15.0])), empty_frac=float(rng.choice([0.0, 0.2, 0.7])))
        if case % 3 == 2:
            r2 = np.random.default_rng(seed)
            prob.tv_under = (prob.t_under[prob.sid] * r2.uniform(0.8, 1.2, prob.n_v)).astype(np.float32)
            prob.tv_over = (prob.t_over[prob.sid] * r2.uniform(0.8, 1.2, prob.n_v)).astype(np.float32)
        plan = m.Plan(prob, max_iters=10, driver=int(rng.choice([0, 1, 2])), ls_batch=int(rng.choice([1, 2, 4])))
        x = np.random.default_rng(seed + 1).uniform(0, 80, prob.n_b).astype(np.float32)
        check_eval(m, plan, prob, x)
        plan.set_x(prob.x0)
        plan.run_iters(10)
        tr = plan.trace()
        assert (np.diff(tr.obj) < 0).all() and (plan.get_x().cpu().numpy() >= 0).all(), prob.name
        plan.close()


# ---------------------------------------------------------------------------------------------- tuning blobs, dense quads
def test_tuned_partition_can_be_exported_and_reinjected(m):
    # tune_level >= 1 balances the passes from measured times, so two tuned plans may differ in the last bits; a plan
    # created from the first one's blob (imrt_plan_get_tuning -> imrt_options.host_tuning) reproduces it bit for bit
    prob = phantom(2)
    p1, tr1, x1, d1, _ = run_gpu(m, prob, 30, m.DRIVER_PERSISTENT, tune_level=2)
    blob = p1.tuning()
    p2 = m.Plan(prob, max_iters=30, tuning=blob)
    p2.set_x(prob.x0)
    p2.run_iters(30)
    tr2 = p2.trace()
    np.testing.assert_array_equal(tr2.obj, tr1.obj)
    np.testing.assert_array_equal(p2.get_x().cpu().numpy(), x1)
    with pytest.raises(m.ImrtError):
        m.Plan(phantom(0), max_iters=4, tuning=blob)          # another problem's blob is refused
    p1.close()
    p2.close()


def test_dense_quads_fall_back_to_row_records(m):
    # 4 full rows of a wide matrix: one quad record would not fit in the ring twice, so those rows go to row-format records
    prob = synth_inputs.make_random(31, n_v=64, n_b=8000, density=0.02, empty_row_frac=0.0, full_rows=4)
    plan = m.Plan(prob, max_iters=4)
    x = np.random.default_rng(1).uniform(0, 2, prob.n_b).astype(np.float32)
    check_eval(m, plan, prob, x)
    plan.close()


@pytest.mark.parametrize("seed,n_v,n_b,n_groups", [(1, 300, 40, 37), (2, 5000, 700, 1200), (3, 64, 30000, 9), (4, 2000, 5, 2500)])
def test_merge_rows_matches_oracle_bit_for_bit(m, seed, n_v, n_b, n_groups):
    # rows scattered over the groups at random (not neighbours), groups without rows, empty rows, one very wide matrix
    import torch
    prob = synth_inputs.make_random(seed, n_v=n_v, n_b=n_b, density=0.1 if n_b < 1000 else 0.003, empty_row_frac=0.2, full_rows=1)
    group = np.random.default_rng(seed).integers(0, n_groups, n_v).astype(np.int32)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    m_rp, m_col, m_val = m.imrt_merge_rows(n_b, dev(prob.row_ptr), dev(prob.col), dev(prob.val), dev(group), n_groups)
    o_rp, o_col, o_val = oracle.merge_rows(n_b, prob.row_ptr, prob.col, prob.val, group, n_groups)
    np.testing.assert_array_equal(m_rp.cpu().numpy(), o_rp)
    np.testing.assert_array_equal(m_col.cpu().numpy(), o_col)
    np.testing.assert_array_equal(m_val.cpu().numpy(), o_val)
    bad = group.copy()
    bad[0] = n_groups
    with pytest.raises(m.ImrtError):
        m.imrt_merge_rows(n_b, dev(prob.row_ptr), dev(prob.col), dev(prob.val), dev(bad), n_groups)
    # the raw CSR is validated here too (merging runs before imrt_plan_create): a column outside [0, n_b) must not reach the
    # shared-memory column bitmap, a decreasing row_ptr must not be followed
    if prob.col.size:
        bad_col = prob.col.copy()
        bad_col[bad_col.size // 2] = n_b
        with pytest.raises(m.ImrtError) as e:
            m.imrt_merge_rows(n_b, dev(prob.row_ptr), dev(bad_col), dev(prob.val), dev(group), n_groups)
        assert e.value.status_name == "BAD_CSR"
        bad_col[bad_col.size // 2] = -1
        with pytest.raises(m.ImrtError) as e:
            m.imrt_merge_rows(n_b, dev(prob.row_ptr), dev(bad_col), dev(prob.val), dev(group), n_groups)
        assert e.value.status_name == "BAD_CSR"
    bad_rp = prob.row_ptr.copy()
    bad_rp[n_v // 2] = bad_rp[-1] + 7
    with pytest.raises(m.ImrtError) as e:
        m.imrt_merge_rows(n_b, dev(bad_rp), dev(prob.col), dev(prob.val), dev(group), n_groups)
    assert e.value.status_name == "BAD_CSR"
