"""The boundary: libimrtgp.so loads and exports every symbol include/imrtgp.h declares, the Python
binding carries the same names, the host-only entry points follow the paper's scalar rules, and nothing on the product
path can fall back to the oracle or to a CPU implementation.  No compute call is made: all of this runs without a GPU.
"""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_0908_4421_b200 as imrt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_in_header():
    src = open(os.path.join(ROOT, "include", "imrtgp.h")).read()
    src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)                  # comments mention the calls too
    return re.findall(r"\b(?:imrt_status|int32_t|const\s+char\s*\*)\s*(imrt_[a-z_0-9]+)\s*\(", src)


def test_every_declared_symbol_is_exported_and_bound():
    names = declared_in_header()
    assert len(names) == len(set(names)) >= 20
    assert set(names) == set(imrt.EXPORTS)                           # the binding's list is the header's list
    L = imrt.lib()
    for n in names:
        assert getattr(L, n) is not None                             # dlsym: raises AttributeError when missing
    # the binding has a function of the same name for every call (imrt_last_error surfaces as ImrtError's message)
    for n in names:
        if n != "imrt_last_error":
            assert callable(getattr(imrt, n)), n
    assert imrt.imrt_version().startswith("imrtgp") and "sm_100a" in imrt.imrt_version()


def test_signatures_carry_no_torch_or_cxx_types():
    src = open(os.path.join(ROOT, "include", "imrtgp.h")).read()
    assert 'extern "C"' in src
    code = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)
    for banned in ("torch", "at::", "std::", "template", "class "):
        assert banned not in code, banned


def test_workspace_bytes_is_host_arithmetic():
    small = imrt.imrt_workspace_bytes(1000, 10, 5000, 3, 50)
    big = imrt.imrt_workspace_bytes(1187328, 2304, 62869568, 4, 500)   # cfg3
    assert 0 < small < big
    assert big > 2 * 8 * 62869568 * 0.5                                # room for both re-encoded matrices
    assert big < 8 * (1 << 30)                                         # and nowhere near the 180 GB of HBM
    with pytest.raises(imrt.ImrtError) as e:
        imrt.imrt_workspace_bytes(-1, 10, 5000, 3, 50)
    assert e.value.status_name == "INVALID_ARG"


def test_armijo_and_stop_rules_by_hand():
    # PAPER.md:92-95 Eq. (5): C = G_k - (eps / lambda) * ||x+ - x||^2, accept iff G_new < C (strict).
    # G_k = 10, eps = 0.5, lambda = 1, step_sq = 1 -> C = 9.5
    assert imrt.imrt_armijo_accepts(10.0, 9.0, 1.0, 0.5, 1.0) == 1
    assert imrt.imrt_armijo_accepts(10.0, 9.5, 1.0, 0.5, 1.0) == 0     # equality is a rejection
    assert imrt.imrt_armijo_accepts(10.0, 9.6, 1.0, 0.5, 1.0) == 0
    # a smaller lambda raises the bar: eps / lambda = 4 -> C = 6
    assert imrt.imrt_armijo_accepts(10.0, 6.5, 1.0, 0.5, 0.125) == 0
    assert imrt.imrt_armijo_accepts(10.0, 5.5, 1.0, 0.5, 0.125) == 1
    # PAPER.md:112-114 step 5 (reading R5): |G_new - G_old| / G_new < delta; G_new = 0 stops
    assert imrt.imrt_stop_test(10.0, 9.0, 1e-3) == 0                   # 1/9
    assert imrt.imrt_stop_test(10.0, 9.995, 1e-3) == 1                 # 5.0e-4
    assert imrt.imrt_stop_test(8.0, 10.0, 0.25) == 1                   # 0.2: relative to the NEW value
    assert imrt.imrt_stop_test(10.0, 8.0, 0.25) == 0                   # 0.25 is not < 0.25
    assert imrt.imrt_stop_test(10.0, 0.0, 1e-3) == 1


def test_null_and_undersized_arguments_are_refused_with_a_message():
    L = imrt.lib()
    out = ctypes.c_void_p()
    prm = imrt.Params(0.2, 2.0, 1e-3, 30, 10, imrt.DRIVER_PERSISTENT, 0)
    s = L.imrt_plan_create(ctypes.byref(out), 10, 2, 5, None, None, None, None, 1, None, None, None, None, ctypes.byref(prm), None, None, 0, None)
    assert imrt.STATUS_NAMES[s] == "INVALID_ARG" and b"null" in L.imrt_last_error(None) and out.value is None
    assert imrt.STATUS_NAMES[L.imrt_plan_run_iters(None, 3)] == "INVALID_ARG"
    assert imrt.STATUS_NAMES[L.imrt_plan_destroy(None)] == "INVALID_ARG"
    # a workspace smaller than imrt_workspace_bytes() says how much is needed (checked before anything is touched)
    hp = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rp, ci, v, sid = np.array([0, 1, 2], np.int32), np.zeros(2, np.int32), np.ones(2, np.float32), np.zeros(2, np.uint8)
    t, ws = np.ones(1, np.float32), np.zeros(1 << 16, np.uint8)
    s = L.imrt_plan_create(ctypes.byref(out), 2, 1, 2, hp(rp), hp(ci), hp(v), hp(sid), 1, hp(t), hp(t), hp(t), hp(t), ctypes.byref(prm),
                           None, hp(ws), ws.nbytes, None)
    assert imrt.STATUS_NAMES[s] == "WORKSPACE_TOO_SMALL" and b"needed" in L.imrt_last_error(None)


def test_no_device_is_an_error_not_a_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    L = imrt.lib()
    out = ctypes.c_void_p()
    prm = imrt.Params(0.2, 2.0, 1e-3, 30, 10, imrt.DRIVER_PERSISTENT, 0)
    hp = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rp, ci, v, sid = np.array([0, 1, 2], np.int32), np.zeros(2, np.int32), np.ones(2, np.float32), np.zeros(2, np.uint8)
    t = np.ones(1, np.float32)
    ws = np.zeros(imrt.imrt_workspace_bytes(2, 1, 2, 1, 10), np.uint8)
    s = L.imrt_plan_create(ctypes.byref(out), 2, 1, 2, hp(rp), hp(ci), hp(v), hp(sid), 1, hp(t), hp(t), hp(t), hp(t), ctypes.byref(prm),
                           None, hp(ws), ws.nbytes, None)
    assert imrt.STATUS_NAMES[s] in ("CUDA_ERROR", "UNSUPPORTED_DEVICE") and out.value is None
    assert L.imrt_last_error(None)


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_0908_4421_b200 import build as b

    def no_nvcc():
        raise RuntimeError("nvcc not found")
    monkeypatch.setattr(imrt, "_lib", None)
    monkeypatch.setattr(b, "build", no_nvcc)
    monkeypatch.setattr(b, "LIB", str(tmp_path / "libimrtgp.so"))
    with pytest.raises(ImportError, match="not built"):
        imrt.imrt_version()


def test_product_and_oracle_share_nothing():
    pkg = os.path.join(ROOT, "paper_0908_4421_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "imrt_oracle" not in text and "oracle/" not in text, f
    assert "oracle" not in open(os.path.join(ROOT, "include", "imrtgp.h")).read().lower()
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_0908_4421_b200" not in text and "from paper_0908_4421_b200" not in text, f
            assert "imrtgp.h" not in text and "libimrtgp" not in text, f


def test_the_library_reads_no_environment_variables():
    # every switch of the library is a field of imrt_params / imrt_options (include/imrtgp.h): no getenv in csrc/
    import glob
    for path in glob.glob(os.path.join(ROOT, "paper_0908_4421_b200", "csrc", "*")):
        with open(path) as f:
            assert "getenv" not in f.read(), path


def test_shard_inbox_size_and_refusals_host_only():
    # imrt_shard_inbox_bytes is host arithmetic: flags for 16 ranks (2 x 128 B), the objective slots
    # (2 parities x 16 ranks x 4 trial points x 8 B) and 2 parities x world x n_b (padded to 32) fp32 gradient partials
    assert imrt.imrt_shard_inbox_bytes(2304, 2) == 256 + 1024 + 2 * 2 * 2304 * 4
    assert imrt.imrt_shard_inbox_bytes(5, 3) == 256 + 1024 + 2 * 3 * 32 * 4
    L = imrt.lib()
    n = ctypes.c_size_t(0)
    assert imrt.STATUS_NAMES[L.imrt_shard_inbox_bytes(100, 17, ctypes.byref(n))] == "INVALID_ARG"      # at most 16 ranks
    assert imrt.STATUS_NAMES[L.imrt_plan_set_shard(None, 0, 2, None)] == "INVALID_ARG"
    assert imrt.STATUS_NAMES[L.imrt_plan_run_ranks(None, 2, 1, 0.0)] == "INVALID_ARG"
    assert imrt.STATUS_NAMES[L.imrt_merge_rows_workspace_bytes(0, 1, ctypes.byref(n))] == "INVALID_ARG"
    assert imrt.imrt_merge_rows_workspace_bytes(1000, 10) > 5 * 4 * 1000
