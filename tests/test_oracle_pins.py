"""Pins for the fp64 CPU oracle (oracle/imrt_oracle.c) -- CPU only.

The paper prints no worked numerical example, no eps/alpha/lambda0 and no iteration counts
(SURVEY.md 8(c.3)), so the oracle is pinned to what the paper's definitions and the mathematics
fix: hand-derived closed forms (tests/golden/hand_cases.json), brute-force dense products,
central finite differences, Armijo / monotonicity invariants, KKT at convergence, reduction to
textbook NNLS (scipy.optimize.nnls) and scale invariance.
"""
import json
import os

import numpy as np
import pytest

import oracle
import synth_inputs
from synth_inputs import Problem

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_cases.json")))


def dense_problem(D, sid, t_u, t_o, w_u, w_o, x0, **kw):
    """CSR problem from a small dense matrix (exact zeros dropped)."""
    D = np.asarray(D, dtype=np.float32)
    n_v, n_b = D.shape
    row_ptr, col, val = [0], [], []
    for j in range(n_v):
        for i in range(n_b):
            if D[j, i] != 0.0:
                col.append(i)
                val.append(D[j, i])
        row_ptr.append(len(col))
    f32 = lambda a: np.asarray(a, dtype=np.float32)
    return Problem("dense", n_v, n_b, np.asarray(row_ptr, np.int32), np.asarray(col, np.int32), f32(val),
                   np.asarray(sid, np.uint8), f32(t_u), f32(t_o), f32(w_u), f32(w_o), f32(x0), **kw)


def to_dense(prob):
    D = np.zeros((prob.n_v, prob.n_b), dtype=np.float64)
    for j in range(prob.n_v):
        for p in range(prob.row_ptr[j], prob.row_ptr[j + 1]):
            D[j, prob.col[p]] += float(prob.val[p])
    return D


# ------------------------------------------------------------------ d = D x
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_dose_matches_brute_force_dense(seed):
    prob = synth_inputs.make_random(seed, n_v=50, n_b=8, density=0.4, empty_row_frac=0.2, full_rows=2)
    rl = np.diff(prob.row_ptr)
    assert (rl == 0).any() and (rl == 1).any() and (rl == prob.n_b).any()  # empty, single-entry, full rows
    x = np.random.default_rng(seed).uniform(0, 3, prob.n_b)
    d, _, _ = oracle.eval_objective(prob, x)
    D = to_dense(prob)
    ref = np.array([sum(D[j, i] * x[i] for i in range(prob.n_b)) for j in range(prob.n_v)])
    np.testing.assert_allclose(d, ref, rtol=1e-14, atol=1e-14)


# ------------------------------------------------------------------ G, r closed forms  (Eq. (1)-(2))
def test_one_by_one_hand_case():
    c = GOLD["one_by_one"]
    prob = dense_problem(c["D"], [0], [c["T"]], [c["T"]], [1.0], [1.0], c["x"])
    d, r, G = oracle.eval_objective(prob, np.array(c["x"]))
    g = oracle.gradient(prob, r)
    assert G == c["G"] and list(r) == c["r"] and list(g) == c["g"] and d[0] == 1.0


def test_zero_penalty_when_every_voxel_at_bound():
    # rows with one entry 1.0, x = T  =>  d = T  =>  G = 0, r = 0, g = 0     (north-star check)
    n = 7
    T = np.array([70, 50, 50, 60, 70, 50, 60], dtype=np.float64)
    sid = [0, 1, 2, 3, 0, 1, 3]
    prob = dense_problem(np.eye(n), sid, [70, 0, 0, 0], [70, 50, 50, 60], [100, 0, 0, 0], [100, 10, 10, 1], T)
    d, r, G = oracle.eval_objective(prob, T)
    assert G == 0.0 and not r.any() and not oracle.gradient(prob, r).any()
    np.testing.assert_array_equal(d, T)


def test_one_sided_terms():
    # (iii) an OAR voxel below its limit contributes 0; above it, w+ (d-T+)^2
    # (iv) a target voxel above T+ contributes only the over term, below T- only the under term
    prob = dense_problem(np.eye(4), [1, 1, 0, 0], [70, 0], [72, 50], [100, 0], [30, 10], [40, 55, 75, 64])
    d, r, G = oracle.eval_objective(prob, np.array([40.0, 55.0, 75.0, 64.0]))
    terms = [0.0, 10 * 5.0 ** 2, 30 * 3.0 ** 2, 100 * 6.0 ** 2]
    assert G == sum(terms)
    np.testing.assert_array_equal(r, [0.0, 2 * 10 * 5.0, 2 * 30 * 3.0, -2 * 100 * 6.0])
    # in the dead band of a target (T- <= d <= T+) nothing is charged
    _, r2, G2 = oracle.eval_objective(prob, np.array([0.0, 0.0, 71.0, 71.0]))
    assert G2 == 0.0 and not r2.any()


def test_union_read_as_sum_matches_paper_model():
    # unweighted, T- = T+ = T_j; targets get both terms, non-targets only F+   (reading R1)
    rng = np.random.default_rng(5)
    D = rng.uniform(0, 1, (12, 4)) * (rng.random((12, 4)) < 0.6)
    sid = [0] * 5 + [1] * 7
    prob = dense_problem(D, sid, [30, 0], [30, 30], [1, 0], [1, 1], np.ones(4))
    # per-voxel T is emulated by one structure per class here: T = 30 for everyone
    x = rng.uniform(0, 40, 4)
    z = D.astype(np.float32).astype(np.float64) @ x
    G_paper = sum(max(0, 30 - z[j]) ** 2 for j in range(5)) + sum(max(0, z[j] - 30) ** 2 for j in range(12))
    _, _, G = oracle.eval_objective(prob, x)
    assert abs(G - G_paper) <= 1e-12 * G_paper


# ------------------------------------------------------------------ gradient  (reading R3)
@pytest.mark.parametrize("seed", [10, 11, 12])
def test_gradient_matches_central_finite_differences(seed):
    prob = synth_inputs.make_random(seed, n_v=40, n_b=6, density=0.5)
    rng = np.random.default_rng(seed)
    x = rng.uniform(20, 60, prob.n_b)
    d, r, _ = oracle.eval_objective(prob, x)
    # keep instances where no voxel sits within the FD step of a kink
    s = prob.sid
    margin = np.minimum(np.abs(d - prob.t_under[s]), np.abs(d - prob.t_over[s]))
    assert margin[np.diff(prob.row_ptr) > 0].min() > 1e-2
    assert (r != 0).sum() > 5
    g = oracle.gradient(prob, r)
    fd = np.empty_like(g)
    for i in range(prob.n_b):
        h = 1e-5 * (1 + abs(x[i]))
        xp, xm = x.copy(), x.copy()
        xp[i] += h
        xm[i] -= h
        fd[i] = (oracle.eval_objective(prob, xp)[2] - oracle.eval_objective(prob, xm)[2]) / (2 * h)
    np.testing.assert_allclose(g, fd, rtol=1e-6, atol=1e-6 * np.abs(g).max())


def test_gradient_scatter_equals_dense_transpose():
    prob = synth_inputs.make_random(21, n_v=50, n_b=8, density=0.4, full_rows=1)
    r = np.random.default_rng(3).normal(size=prob.n_v)
    g = oracle.gradient(prob, r)
    Dt = to_dense(prob).T.copy()
    ref = np.array([sum(Dt[i, j] * r[j] for j in range(prob.n_v)) for i in range(prob.n_b)])
    np.testing.assert_allclose(g, ref, rtol=1e-13, atol=1e-13)


# ------------------------------------------------------------------ projection
def test_projection_feasible_and_sticky_at_zero():
    x = np.array([0.0, 0.0, 1.0, 2.0, 0.5])
    g = np.array([3.0, -1.0, 4.0, -2.0, 1.0])
    xn, delta = oracle.trial_point(x, g, 0.5)
    np.testing.assert_array_equal(xn, [0.0, 0.5, 0.0, 3.0, 0.0])
    assert (xn >= 0).all() and xn[0] == 0.0
    assert delta == 0.25 + 1.0 + 1.0 + 0.25
    assert not np.signbit(xn).any()  # max(0, -0.0) -> +0


# ------------------------------------------------------------------ Armijo
def test_identity_hand_trace_two_trials_then_stationary():
    c = GOLD["identity_two_trials"]
    T = c["T"]
    prob = dense_problem(np.eye(3), [0, 1, 2], T, T, [1, 1, 1], [1, 1, 1], c["x1"],
                         eps=0.2, alpha=2.0, lambda0=1.0, n_iters=5)
    _, r, G1 = oracle.eval_objective(prob, np.array(c["x1"]))
    assert G1 == c["G1"] and list(oracle.gradient(prob, r)) == c["g1"]
    for lam, t in ((1.0, c["trial1"]), (0.5, c["trial2"])):
        xn, delta = oracle.trial_point(np.array(c["x1"]), np.array(c["g1"]), lam)
        assert list(xn) == t["x"] and delta == t["Delta"]
        assert oracle.eval_objective(prob, xn)[2] == t["G"]
        assert c["G1"] - 0.2 / lam * delta == t["C"]
    res = oracle.run(prob)
    assert res.n_iters == 1 and res.stop_reason == oracle.STOP_STATIONARY
    assert list(res.n_trials) == c["n_trials"] and list(res.lam) == c["lambda"] and list(res.obj) == c["obj"]
    assert list(res.x) == T
    assert res.fwd_passes == 3 and res.tr_passes == 2


def replay_armijo(prob, res):
    """Re-derive every accept/reject of a trace from eval/grad/trial_point alone."""
    x = prob.x0.astype(np.float64)
    for k in range(res.n_iters):
        _, r, Gk = oracle.eval_objective(prob, x)
        assert Gk == res.obj[k]
        g = oracle.gradient(prob, r)
        lam = prob.lambda0
        for m in range(res.n_trials[k]):
            xn, delta = oracle.trial_point(x, g, lam)
            Gn = oracle.eval_objective(prob, xn)[2]
            C = Gk - prob.eps / lam * delta
            if m + 1 < res.n_trials[k]:
                assert not (Gn < C)          # every earlier trial fails the test
                lam = lam / prob.alpha
            else:
                assert Gn < C                # the accepted one passes it
                assert lam == res.lam[k] and Gn == res.obj[k + 1] and delta == res.step_sq[k]
        x = xn
    np.testing.assert_array_equal(x, res.x)


def test_trace_invariants_on_tiny_phantom(phantom0):
    res = oracle.run(phantom0, n_iters=12)
    assert res.n_iters == 12 and res.stop_reason == oracle.STOP_MAX_ITERS
    assert (np.diff(res.obj) < 0).all()                    # strictly decreasing (north-star: monotone)
    assert (res.x >= 0).all()
    assert (res.n_trials >= 1).all() and res.n_trials.max() > 1   # backtracking is exercised
    assert res.fwd_passes == 1 + res.n_trials.sum() and res.tr_passes == 12
    replay_armijo(phantom0, res)


def test_follow_mode_reproduces_free_run_and_flags_wrong_counts(phantom0):
    free = oracle.run(phantom0, n_iters=10)
    fol = oracle.run(phantom0, n_iters=10, follow_trials=free.n_trials)
    assert fol.n_follow_violations == 0
    np.testing.assert_array_equal(fol.obj, free.obj)
    wrong = free.n_trials.copy()
    wrong[3] += 1
    bad = oracle.run(phantom0, n_iters=10, follow_trials=wrong)
    assert bad.n_follow_violations >= 1 and bad.first_violation == 3


def test_stationary_and_stall_exits():
    # x already optimal: G = 0 -> STATIONARY without a single trial
    prob = dense_problem(np.eye(2), [0, 0], [5], [5], [1], [1], [5, 5], n_iters=3)
    res = oracle.run(prob)
    assert res.n_iters == 0 and res.stop_reason == oracle.STOP_STATIONARY and res.fwd_passes == 1
    # g > 0 on a coordinate at 0 and nothing else to move: zero step -> STATIONARY (reading R4)
    prob = dense_problem([[1.0]], [0], [0], [1], [0], [1], [0.0], n_iters=3)
    prob.t_over[:] = -1.0   # d = 0 > T+ = -1: over-dosed, gradient +2, x stays at 0
    res = oracle.run(prob)
    assert res.n_iters == 0 and res.stop_reason == oracle.STOP_STATIONARY
    # max_ls cap: lambda0 far too large and only 2 backtracks allowed
    prob = dense_problem(np.eye(2), [0, 0], [5], [5], [1], [1], [1, 9], lambda0=1024.0, max_ls=2, n_iters=3)
    res = oracle.run(prob)
    assert res.n_iters == 0 and res.stop_reason == oracle.STOP_LS_STALLED and res.fwd_passes == 1 + 3


# ------------------------------------------------------------------ whole optimiser
def nnls_problem(seed, n_v=30, n_b=6):
    rng = np.random.default_rng(seed)
    D = rng.uniform(0.1, 1.0, (n_v, n_b)) * (rng.random((n_v, n_b)) < 0.7)
    D[:, 0] = D[:, 1] * 0.5 + 0.3          # make some coordinates want to be negative -> active bounds
    T = rng.uniform(5, 40, n_v).astype(np.float32)
    # one structure per voxel => per-voxel prescription T_j, the paper's literal model
    prob = dense_problem(D, np.arange(n_v), T, T, np.full(n_v, 3.0), np.full(n_v, 3.0),
                         rng.uniform(0.5, 1.5, n_b), n_iters=200000, delta=1e-14)
    prob.lambda0, _ = synth_inputs.pick_lambda0(prob.row_ptr, prob.col, prob.val, prob.sid, prob.w_under, prob.w_over)
    return prob, to_dense(prob), T.astype(np.float64)


@pytest.mark.parametrize("seed", [0, 1])
def test_reduces_to_nnls(seed):
    from scipy.optimize import nnls
    prob, D, T = nnls_problem(seed)
    res = oracle.run(prob)
    assert res.stop_reason in (oracle.STOP_TOLERANCE, oracle.STOP_STATIONARY)
    x_ref, rnorm = nnls(D, T)
    G_ref = 3.0 * rnorm ** 2
    assert abs(res.obj[-1] - G_ref) <= 1e-8 * G_ref
    assert (x_ref == 0).any()              # a bound is active, so the projection matters
    # KKT at convergence (north-star check): g_i >= -tol where x_i = 0, |g_i| <= tol where x_i > 0
    _, r, _ = oracle.eval_objective(prob, res.x)
    g = oracle.gradient(prob, r)
    tol = 1e-4 * np.abs(oracle.gradient(prob, oracle.eval_objective(prob, prob.x0.astype(np.float64))[1])).max()
    assert (g[res.x == 0] >= -tol).all() and (np.abs(g[res.x > 0]) <= tol).all()
    assert np.abs(res.x - np.maximum(0, res.x - g)).max() <= tol


def test_scale_invariance(phantom0):
    # weights * c, lambda0 / c  =>  same x trajectory, G scaled by c      (c a power of two: exact in fp)
    c = 4.0
    res1 = oracle.run(phantom0, n_iters=8)
    scaled = Problem(**{**phantom0.__dict__})
    scaled.w_under = phantom0.w_under * np.float32(c)
    scaled.w_over = phantom0.w_over * np.float32(c)
    scaled.lambda0 = phantom0.lambda0 / c
    res2 = oracle.run(scaled, n_iters=8)
    np.testing.assert_array_equal(res1.n_trials, res2.n_trials)
    np.testing.assert_allclose(res2.x, res1.x, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(res2.obj, c * res1.obj, rtol=1e-12)


def test_tolerance_stop_rule(phantom0):
    # step 5 (reading R5): stop at the first k with |G_new - G_old| / G_new < delta
    res = oracle.run(phantom0, n_iters=400, delta=1e-3)
    assert res.stop_reason == oracle.STOP_TOLERANCE
    rel = np.abs(np.diff(res.obj)) / res.obj[1:]
    assert rel[-1] < 1e-3 and (rel[:-1] >= 1e-3).all()


# ------------------------------------------------------------------ DVH points
def test_dvh_hand_case():
    c = GOLD["dvh_1_to_10"]
    doses = np.array(c["doses"] + [100.0, 200.0], dtype=np.float64)
    sid = np.array([0] * 10 + [1, 1], dtype=np.uint8)
    dp, mean = oracle.dvh_points(sid, doses, 3, c["pcts"])
    assert list(dp[0]) == c["D_p"] and mean[0] == c["mean"]
    assert list(dp[1]) == [200.0, 200.0, 200.0, 100.0, 100.0] and mean[1] == 150.0
    assert np.isnan(dp[2]).all() and np.isnan(mean[2])


# ------------------------------------------------------------------ per-voxel limits  (reading R16)
def test_per_voxel_limits_are_the_papers_literal_model():
    # Eq. (1) with its own T_j per voxel: F-_j = max(0, T_j - z_j)^2 on targets, F+_j = max(0, z_j - T_j)^2 on all voxels,
    # written out here independently of the oracle; gradient 2 D^T (o - u [targets]) checked by central differences.
    rng = np.random.default_rng(21)
    D = rng.uniform(0, 1, (15, 5)) * (rng.random((15, 5)) < 0.6)
    sid = [0] * 6 + [1] * 9                       # structure 0 = targets
    T = rng.uniform(5, 60, 15).astype(np.float32)
    prob = dense_problem(D, sid, [999, 999], [999, 999], [1, 0], [1, 1], np.ones(5))   # per-structure limits unused
    prob.tv_under, prob.tv_over = T.copy(), T.copy()
    x = rng.uniform(0, 40, 5)
    z = D.astype(np.float32).astype(np.float64) @ x
    G_paper = sum(max(0.0, T[j] - z[j]) ** 2 for j in range(6)) + sum(max(0.0, z[j] - T[j]) ** 2 for j in range(15))
    d, r, G = oracle.eval_objective(prob, x)
    assert abs(G - G_paper) <= 1e-12 * G_paper
    g = oracle.gradient(prob, r)
    for i in range(5):
        h = 1e-5 * (1 + abs(x[i]))
        xp, xm = x.copy(), x.copy()
        xp[i] += h
        xm[i] -= h
        fd = (oracle.eval_objective(prob, xp)[2] - oracle.eval_objective(prob, xm)[2]) / (2 * h)
        assert abs(fd - g[i]) <= 1e-6 * max(1.0, abs(g[i]))
    # per-voxel arrays that repeat the structure's limits change nothing, bit for bit
    base = synth_inputs.make_phantom(0)
    ref = oracle.run(base, n_iters=8)
    base.tv_under, base.tv_over = base.t_under[base.sid].copy(), base.t_over[base.sid].copy()
    same = oracle.run(base, n_iters=8)
    np.testing.assert_array_equal(ref.obj, same.obj)
    np.testing.assert_array_equal(ref.x, same.x)
    # only one side given: the other keeps the structure's limit
    base.tv_under = None
    base.tv_over = (base.t_over[base.sid] * 0.9).astype(np.float32)
    x_hot = np.full(base.n_b, 40.0)               # hot enough for voxels to sit above their upper limits
    G_tight = oracle.eval_objective(base, x_hot)[2]
    base.tv_over = None
    G_plain = oracle.eval_objective(base, x_hot)[2]
    assert G_tight > G_plain                      # tighter upper limits, same lower limits: a larger penalty


# ------------------------------------------------------------------ input preparation: mixed resolution
def test_mixed_resolution_rows_are_block_means(phantom0):
    # harness check: a coarse voxel's dose is the mean dose of the fine body voxels in its 2x2x2 block, target / OAR rows
    # are untouched, and the beamlet side is unchanged
    mixed = synth_inputs.mixed_resolution(phantom0)
    x = np.random.default_rng(3).uniform(0, 30, phantom0.n_b)
    d_fine = oracle.eval_objective(phantom0, x)[0]
    d_mixed = oracle.eval_objective(mixed, x)[0]
    nx, ny, nz = phantom0.meta["grid"]
    vid = phantom0.voxel_ids
    key = (vid % nx) // 2 + ((nx + 1) // 2) * (((vid // nx) % ny) // 2 + ((ny + 1) // 2) * ((vid // (nx * ny)) // 2))
    body = phantom0.sid == 3
    n_fine = int((~body).sum())
    np.testing.assert_allclose(d_mixed[:n_fine], d_fine[~body], rtol=1e-6, atol=1e-9)
    means = {}
    for k, dv in zip(key[body], d_fine[body]):
        means.setdefault(int(k), []).append(dv)
    expect = np.array([np.mean(means[k]) for k in sorted(means)])
    assert mixed.n_v == n_fine + expect.shape[0] and mixed.n_b == phantom0.n_b
    np.testing.assert_allclose(d_mixed[n_fine:], expect, rtol=1e-5, atol=1e-7)     # fp32 rounding of the merged values
    assert (mixed.sid[n_fine:] == 3).all() and (mixed.sid[:n_fine] != 3).all()


def test_merge_rows_hand_case_and_block_means(phantom0):
    # oracle.merge_rows (reading R17) pinned by (i) a hand case, (ii) the independently built scipy block
    # means of synth_inputs.mixed_resolution: same structure, values within one fp32 ulp (scipy adds in another order)
    rp = np.array([0, 2, 3, 4, 4], np.int32)
    col = np.array([0, 2, 0, 1], np.int32)
    val = np.array([1.0, 3.0, 3.0, 5.0], np.float32)
    group = np.array([0, 0, 2, 0], np.int32)             # rows 0, 1 and the empty row 3 -> group 0; group 1 has no rows
    orp, oc, ov = oracle.merge_rows(3, rp, col, val, group, 3)
    assert orp.tolist() == [0, 2, 2, 3] and oc.tolist() == [0, 2, 1]
    np.testing.assert_array_equal(ov, np.array([4.0 / 3.0, 1.0, 5.0], np.float32))      # (1 + 3) / 3, 3 / 3, 5 / 1
    group, n_groups, sid_g = synth_inputs.mixed_resolution_groups(phantom0)
    orp, oc, ov = oracle.merge_rows(phantom0.n_b, phantom0.row_ptr, phantom0.col, phantom0.val, group, n_groups)
    mixed = synth_inputs.mixed_resolution(phantom0)
    np.testing.assert_array_equal(sid_g, mixed.sid)
    np.testing.assert_array_equal(orp, mixed.row_ptr)
    np.testing.assert_array_equal(oc, mixed.col)
    assert (np.abs(ov - mixed.val) <= np.spacing(np.abs(mixed.val))).all()
