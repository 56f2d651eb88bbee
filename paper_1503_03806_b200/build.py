"""Builds paper_1503_03806_b200/libhk.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "csrc", "hk_kernels.cu"), os.path.join(HERE, "csrc", "hk_sort.cu"),
       os.path.join(HERE, "csrc", "hk_kdist.cu"), os.path.join(HERE, "csrc", "hk_resample.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "hk_voigt.cuh"), os.path.join(HERE, "csrc", "hk_internal.h"),
              os.path.join(HERE, "..", "include", "hk.h")]
LIB = os.path.join(HERE, "libhk.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=true"]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: the hk CUDA library cannot be built")
    return p


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build_library(force: bool = False, verbose: bool = False) -> str:
    """HK_DEBUG_CHECKS=1 in the environment compiles the index checks (HK_CHECK: a trap instead of an out-of-range access) and the
    ring watchdog in: the build the GPU test suite is run against once per round in place of compute-sanitizer, which is
    closed on this GPU pool."""
    if force or is_stale():
        dbg = ["-DHK_DEBUG_CHECKS", "-DHK_WATCHDOG"] if os.environ.get("HK_DEBUG_CHECKS") == "1" else []
        cmd = [nvcc_path()] + NVCC_FLAGS + dbg + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SRC
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
