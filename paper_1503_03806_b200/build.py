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


LIB_CHECKED = os.path.join(HERE, "libhk_dbg.so")
DEBUG_FLAGS = ["-DHK_DEBUG_CHECKS", "-DHK_WATCHDOG"]


def is_stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build_library(force: bool = False, verbose: bool = False, out: str | None = None, debug: bool | None = None) -> str:
    """Release build -> libhk.so.  The CHECKED build (debug=True, or HK_DEBUG_CHECKS=1 in the environment) compiles in the index
    checks (HK_CHECK: a trap instead of an out-of-range access) and the watchdogs of the mbarrier / ring spin loops, and goes
    to a file of its own — libhk_dbg.so, or `out` — so that it can never stand in for the release library in a bench run;
    hk_version() of such a library says "checked".  It is what tests/test_gpu_debug_build.py runs a slice of the GPU suite
    against, in place of compute-sanitizer, which is closed on this GPU pool."""
    if debug is None:
        debug = os.environ.get("HK_DEBUG_CHECKS") == "1"
    lib = out or (LIB_CHECKED if debug else LIB)
    if force or is_stale(lib):
        cmd = [nvcc_path()] + NVCC_FLAGS + (DEBUG_FLAGS if debug else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + SRC
        subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
