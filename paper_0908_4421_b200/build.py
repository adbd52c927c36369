"""Build libimrtgp.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_0908_4421_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libimrtgp.so")
SOURCES = ["imrtgp.cu"]
HEADERS = ["kernels.cuh", "pipeline.cuh", "dvh.cuh", "merge.cuh", "layout.cuh", os.path.join("..", "..", "include", "imrtgp.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/imrtgp.cu -> libimrtgp.so (idempotent).  Raises CalledProcessError on a compile error."""
    if force or is_stale():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.check_call(cmd, cwd=CSRC)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
