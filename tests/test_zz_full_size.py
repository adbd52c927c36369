"""Full-size GPU parity and run-to-run bit identity: BASELINE.json configs[3] (headline) and configs[4] (stress), in the
launch configuration bench.py times (persistent driver, one CTA per SM, tuned partition).

These take minutes (the serial fp64 oracle replays 300-500 iterations), so the file sorts after every cheap GPU test:
with `pytest -x` a failure here hides nothing but the tests of this file and tests/test_zz_no_alloc.py.

On a failure of the trajectory the tuning blob (imrt_plan_get_tuning), the trace and plan.info() are written to
gpurun_out/fail_dumps/ so that the failing partition can be replayed (imrt_options.host_tuning).
"""
import json
import os

import numpy as np
import pytest

import oracle
from test_gpu_parity import (TOL_DVH_GY, TOL_G_FINAL, check_eval, check_eval_batch, m, phantom, relerr, trial_points,  # noqa: F401
                             _phantoms)

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def dump_on_failure(tag, plan, tr, blob):
    d = os.path.join(ROOT, "gpurun_out", "fail_dumps")
    os.makedirs(d, exist_ok=True)
    with open(os.path.join(d, tag + ".tuning.bin"), "wb") as f:
        f.write(blob)
    np.savez(os.path.join(d, tag + ".trace.npz"), obj=tr.obj, lam=tr.lam, n_trials=tr.n_trials, step_sq=tr.step_sq,
             n_iters=tr.n_iters, stop_reason=tr.stop_reason)
    with open(os.path.join(d, tag + ".info.json"), "w") as f:
        json.dump(plan.info(), f)
    print("dumped %s.{tuning.bin,trace.npz,info.json} to %s" % (tag, d))


def run_from_x0(plan, prob):
    plan.set_x(prob.x0)
    if prob.delta > 0:
        plan.run_to_tol(prob.delta, prob.n_iters)
    else:
        plan.run_iters(prob.n_iters)
    return plan.trace(), plan.get_x().cpu().numpy()


def assert_same_run(tr, x, tr0, x0, what):
    assert tr.n_iters == tr0.n_iters and tr.stop_reason == tr0.stop_reason, \
        "%s: %d iterations (stop %d) against %d (stop %d)" % (what, tr.n_iters, tr.stop_reason, tr0.n_iters, tr0.stop_reason)
    np.testing.assert_array_equal(tr.n_trials, tr0.n_trials, err_msg=what)
    np.testing.assert_array_equal(tr.obj, tr0.obj, err_msg=what)
    np.testing.assert_array_equal(tr.lam, tr0.lam, err_msg=what)
    np.testing.assert_array_equal(tr.step_sq, tr0.step_sq, err_msg=what)
    np.testing.assert_array_equal(x, x0, err_msg=what)


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_parity(m, cfg):
    # the configs' own run lengths: cfg3 "delta = 1e-6 or 500 iterations", cfg4 300 fixed iterations -- the oracle replays
    # the GPU's iteration count in follow mode (about 2 and 4 minutes of serial fp64 work).  The oracle's eval / gradient
    # take well under a second per call even at these sizes, so every output element is compared, not a sample.
    prob = phantom(cfg)
    plan = m.Plan(prob, max_iters=prob.n_iters, driver=m.DRIVER_PERSISTENT, tune_level=2)     # as bench.py creates it
    blob = plan.tuning()
    info = plan.info()
    assert info["fwd_grid"] == info["n_sm"] and info["tr_grid"] == info["n_sm"]   # what bench.py launches
    check_eval(m, plan, prob, prob.x0)
    xo = oracle.run(prob, n_iters=3).x.astype(np.float32)
    check_eval(m, plan, prob, xo)
    check_eval_batch(m, plan, prob, trial_points(prob, xo, 4))     # the R = 4 pass bench.py times, on four trial points

    # trajectory from x0 under the config's own rule
    tr, x = run_from_x0(plan, prob)
    n_iters = tr.n_iters
    print("cfg%d: GPU stopped after %d iterations (%s)" % (cfg, n_iters, m.STOP_NAMES[tr.stop_reason]))
    try:
        assert tr.stop_reason in (oracle.STOP_MAX_ITERS, oracle.STOP_TOLERANCE) and n_iters >= min(300, prob.n_iters)
        assert (np.diff(tr.obj) < 0).all() and (x >= 0).all()
        # Run-to-run bit identity (include/imrtgp.h "Conventions"): the same plan, the same x0, ten times -- any
        # difference between two runs of one plan is a race -- and a second plan built from the first one's partition.
        for rep in range(9):
            tr_r, x_r = run_from_x0(plan, prob)
            assert_same_run(tr_r, x_r, tr, x, "cfg%d, run %d of the same plan" % (cfg, rep + 2))
        twin = m.Plan(prob, max_iters=prob.n_iters, driver=m.DRIVER_PERSISTENT, tuning=blob)
        for rep in range(2):
            tr_t, x_t = run_from_x0(twin, prob)
            assert_same_run(tr_t, x_t, tr, x, "cfg%d, run %d of a plan created from the tuning blob" % (cfg, rep + 1))
        twin.close()
        del twin
        tr_r, x_r = run_from_x0(plan, prob)             # leave `plan` at the end of a run for the checks below
        assert_same_run(tr_r, x_r, tr, x, "cfg%d, last run" % cfg)
    except AssertionError:
        dump_on_failure("cfg%d" % cfg, plan, tr, blob)
        raise

    # the oracle in follow mode
    fol = oracle.run(prob, n_iters=n_iters, follow_trials=tr.n_trials, tau_rel=1e-6)
    try:
        assert fol.n_follow_violations == 0, "first violation at iteration %d" % fol.first_violation
        np.testing.assert_array_equal(tr.lam, fol.lam)
        assert (np.abs(tr.obj - fol.obj) <= TOL_G_FINAL * fol.obj).all()      # every entry, relative to itself
    except AssertionError:
        dump_on_failure("cfg%d" % cfg, plan, tr, blob)
        raise
    d = plan.get_dose().cpu().numpy()
    d_o, _, _ = oracle.eval_objective(prob, fol.x)
    dp_o, mean_o = oracle.dvh_points(prob.sid, d_o, prob.n_structures)
    dp_g, mean_g = plan.dvh(oracle.DVH_PCTS)
    assert np.nanmax(np.abs(dp_g - dp_o)) <= TOL_DVH_GY and np.nanmax(np.abs(mean_g - mean_o)) <= TOL_DVH_GY
    # dose of the two final plans, voxel by voxel: the DVH tolerance (0.5 % of the prescription) applied to EVERY voxel.
    # (The minimiser is not unique -- reading R14 -- so the fp32 and fp64 trajectories may drift apart along directions
    # the objective does not see; DESIGN.md section 6 records the measured drift per iteration.)
    print("cfg%d: dose drift after %d iterations: normwise %.2e, largest voxel %.4f Gy" % (cfg, n_iters, relerr(d, d_o), np.abs(d - d_o).max()))
    assert np.abs(d - d_o).max() <= TOL_DVH_GY
    assert relerr(d, d_o) <= 1e-4      # the bound of round 1's first version, at the full run length
    plan.close()
    _phantoms.pop(cfg, None)        # free ~1-3 GB of host memory
