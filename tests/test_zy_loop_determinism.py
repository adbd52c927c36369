"""The persistent loop is race-free: repeated runs of ONE plan give the same bits, whatever the CTA count.

include/imrtgp.h promises bit-reproducible results per plan.  Two runs of one plan that differ are a race by definition.
The transpose stages overlay the shared-memory trial points and gradient, so the case that
stresses the hand-over hardest is a plan with FEW CTAs: with n_ctas = 1 the one CTA publishes the whole accepted
iterate from shared memory right before its producer warp starts the next transpose pass over the same bytes.
(The full-size repeats -- cfg3 / cfg4, tuned partition, ten runs -- are part of tests/test_zz_full_size.py.)
"""
import numpy as np
import pytest

import oracle
from test_gpu_parity import TOL_G_FINAL, m, phantom  # noqa: F401

pytestmark = pytest.mark.gpu


def one_run(plan, prob, n):
    plan.set_x(prob.x0)
    plan.run_iters(n)
    return plan.trace(), plan.get_x().cpu().numpy()


@pytest.mark.parametrize("cfg,n_ctas,n,reps", [(0, 1, 50, 10), (0, 2, 50, 10), (0, 37, 50, 10), (1, 1, 60, 6), (2, 4, 60, 6), (2, 0, 200, 10)])
def test_repeated_runs_of_one_plan_are_bit_identical(m, cfg, n_ctas, n, reps):
    prob = phantom(cfg)
    plan = m.Plan(prob, max_iters=n, driver=m.DRIVER_PERSISTENT, n_ctas=n_ctas)
    tr0, x0 = one_run(plan, prob, n)
    assert tr0.n_iters == n and m.STOP_NAMES[tr0.stop_reason] == "MAX_ITERS" and tr0.n_trials.max() > 1
    for rep in range(reps - 1):
        tr, x = one_run(plan, prob, n)
        assert tr.n_iters == n and tr.stop_reason == tr0.stop_reason, "run %d stopped after %d iterations" % (rep + 2, tr.n_iters)
        np.testing.assert_array_equal(tr.n_trials, tr0.n_trials)
        np.testing.assert_array_equal(tr.obj, tr0.obj)
        np.testing.assert_array_equal(tr.step_sq, tr0.step_sq)
        np.testing.assert_array_equal(x, x0)
    # and the trajectory is the oracle's (follow mode), so "identical" is not "identically wrong"
    fol = oracle.run(prob, n_iters=n, follow_trials=tr0.n_trials, tau_rel=1e-6)
    assert fol.n_follow_violations == 0
    assert (np.abs(tr0.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()
    plan.close()


def test_a_launch_that_does_no_iteration_changes_nothing(m):
    # imrt_plan_run_iters(0): the loop body never runs; the iterate, the trace and the objective stay as they were
    prob = phantom(0)
    plan = m.Plan(prob, max_iters=10, driver=m.DRIVER_PERSISTENT)
    tr0, x0 = one_run(plan, prob, 5)
    plan.run_iters(0)
    tr = plan.trace()
    np.testing.assert_array_equal(tr.obj, tr0.obj)
    np.testing.assert_array_equal(plan.get_x().cpu().numpy(), x0)
    plan.run_iters(5)                                    # and the run resumes as if nothing had happened
    ref = m.Plan(prob, max_iters=10, driver=m.DRIVER_PERSISTENT)
    tr_ref, x_ref = one_run(ref, prob, 10)
    np.testing.assert_array_equal(plan.trace().obj, tr_ref.obj)
    np.testing.assert_array_equal(plan.get_x().cpu().numpy(), x_ref)
    plan.close()
    ref.close()
