"""imrt_dvh_static: DVH points without any device allocation by the library or for the library.

Some users of libimrtgp cannot give it device memory to work in: their own memory pool already owns the whole GPU (so one
more cudaMalloc fails), or they sit in a stretch of code where the device-wide stall of cudaMalloc / cudaFree is not
acceptable.  For them imrt_dvh_static keeps its histograms in a ~1.1 MB array compiled into the library.  This file
checks that entry point against the existing one, imrt_plan_dvh (scratch in the caller's workspace): same dose in, the
same D_p and mean doses out -- exactly for the D_p (order statistics of the same fp32 doses; the tolerance the other DVH
tests use) and to 1e-12 relative for the means (same kernels, same summation order).  Two calls in a row on different
doses show that what one call leaves in the shared array does not leak into the next; then the first dose again.

The file name sorts last on purpose: `pytest -x` stops at the first failure and this test must not hide the others.
It needs nothing from the tests before it and passes alone in a fresh process as well.
"""

import numpy as np
import pytest

import synth_inputs

pytestmark = pytest.mark.gpu

PCTS = (2.0, 5.0, 50.0, 95.0, 98.0)


@pytest.fixture(scope="module")
def m():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_0908_4421_b200 as mod
    mod.lib()
    return mod


def test_static_scratch_dvh_matches_plan_dvh_on_two_calls_in_a_row(m):
    import torch
    prob = synth_inputs.make_phantom(0)
    plan = m.Plan(prob, max_iters=12)
    n_s = plan.n_structures

    # dose A: the starting point x0 (every voxel far from its limits);  dose B: after 12 GP iterations
    plan.set_x(prob.x0)
    dose_a = plan.get_dose().clone()
    dp_a, mean_a = plan.dvh(PCTS)                       # existing path, scratch in the plan's workspace
    plan.run_iters(12)
    dose_b = plan.get_dose().clone()
    dp_b, mean_b = plan.dvh(PCTS)
    torch.cuda.synchronize()
    assert not np.array_equal(dp_a, dp_b)               # the two calls below really see different inputs

    before = torch.cuda.memory_allocated()
    for dose, dp_ref, mean_ref in ((dose_a, dp_a, mean_a), (dose_b, dp_b, mean_b), (dose_a, dp_a, mean_a)):
        dp, mean = m.imrt_dvh_static(dose, plan.sid, n_s, PCTS, plan.stream.cuda_stream)
        np.testing.assert_array_equal(dp, dp_ref)
        np.testing.assert_allclose(mean, mean_ref, rtol=1e-12, atol=0.0)
    assert torch.cuda.memory_allocated() == before      # and torch was not asked for memory on the way either

    # a single percentage: another histogram count on the same (now dirty) array
    dp1, mean1 = m.imrt_dvh_static(dose_b, plan.sid, n_s, (50.0,), plan.stream.cuda_stream)
    np.testing.assert_array_equal(dp1[:, 0], dp_b[:, PCTS.index(50.0)])
    np.testing.assert_allclose(mean1, mean_b, rtol=1e-12, atol=0.0)
    plan.close()


def test_static_scratch_dvh_refuses_what_does_not_fit(m):
    import torch
    d = torch.ones(1000, dtype=torch.float32, device="cuda:0")
    sid = torch.zeros(1000, dtype=torch.uint8, device="cuda:0")
    with pytest.raises(m.ImrtError) as e:               # 17 structures: beyond the built-in array
        m.imrt_dvh_static(d, sid, 17, PCTS)
    assert e.value.status_name == "UNSUPPORTED" and "at most 16 structures" in str(e.value)
    with pytest.raises(m.ImrtError) as e:               # 16 x 9 = 144 > 128 structure x percentage pairs
        m.imrt_dvh_static(d, sid, 16, np.linspace(1, 99, 9))
    assert e.value.status_name == "UNSUPPORTED" and "128" in str(e.value)
    with pytest.raises(m.ImrtError) as e:               # 17 percentages
        m.imrt_dvh_static(d, sid, 2, np.linspace(1, 99, 17))
    assert e.value.status_name == "UNSUPPORTED"
    sid[123] = 5                                        # a structure id the caller did not announce
    with pytest.raises(m.ImrtError) as e:
        m.imrt_dvh_static(d, sid, 4, PCTS)
    assert e.value.status_name == "BAD_STRUCTURE"
    L = m.lib()
    assert m.STATUS_NAMES[L.imrt_dvh_static(None, None, 10, 2, None, 1, None, None, None)] == "INVALID_ARG"
    # the largest shape that fits: 16 structures x 8 percentages; doses 1..n, so D_p is known in closed form
    n = 4096
    d = torch.arange(1, n + 1, dtype=torch.float32, device="cuda:0")
    sid = (torch.arange(n, device="cuda:0") % 16).to(torch.uint8)
    pcts = np.array([1, 10, 25, 50, 75, 90, 99, 100], np.float64)
    dp, mean = m.imrt_dvh_static(d, sid, 16, pcts)
    per = n // 16
    for s in range(16):
        doses = np.arange(1, n + 1)[s::16]              # ascending
        rank = np.clip(np.ceil(pcts * per / 100.0).astype(int), 1, per)
        np.testing.assert_array_equal(dp[s], doses[::-1][rank - 1])
        assert mean[s] == doses.mean()
