"""The checked build of the library (-DHK_DEBUG_CHECKS -DHK_WATCHDOG) under a slice of the GPU suite.

compute-sanitizer is closed on the GPU pool this repo is developed on (SURVEY.md Appendix B item 9 asks for memcheck and
racecheck on the mbarrier ring and the shared-memory sort).  In its place the sources carry index checks (HK_CHECK: a trap
instead of an out-of-range shared- or global-memory access in a1, the far kernel's ring and the near kernel's queues) and a
watchdog on every mbarrier / ring spin loop (a trap after ~2 s instead of a hung GPU).  This test compiles that build to a
temporary file — libhk.so is not touched — and runs, in a child process whose binding loads it through HK_LIB, the cases that
reach every such check: the five small full-grid cases (incl. the ragged N = 3333), a dense list on the one-warp far shape
with the near kernel, the unsorted list with large pressure shifts, hk_kdist at 1000 / 10000 / 1025 points per bin, the
ranged host path, the no-alloc entry point.  Each case compares against the oracle or the device form as it does in the
release suite; a trap surfaces as a CUDA error in the child and fails it.
"""
import os
import shutil
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = [
    "tests/test_gpu_debug_build.py::test_the_loaded_library_is_the_checked_build",
    "tests/test_gpu_opacity.py::test_small_cases_full_grid",
    "tests/test_gpu_debug_build.py::test_dense_list_one_warp_far_shape_and_near_kernel",
    "tests/test_gpu_line_physics.py::test_large_pressure_shifts_on_a_dense_unsorted_list",
    "tests/test_gpu_kdist.py::test_random_bins_same_kappa",
    "tests/test_gpu_opacity.py::test_host_buffer_form_on_a_grid_wide_enough_for_the_ranged_path",
    "tests/test_gpu_opacity.py::test_host_buffer_form_ranged_path_with_the_k_table",
    "tests/test_zz_no_alloc.py::test_same_kappa_as_hk_opacity_on_calls_in_a_row",
]


def test_the_loaded_library_is_the_checked_build():
    if not os.environ.get("HK_LIB"):
        pytest.skip("runs in the child process of test_checked_build_runs_the_cases_without_a_trap")
    assert "checked" in hk.hk_version()


def test_dense_list_one_warp_far_shape_and_near_kernel():
    # 1e6 lines on 3e5 grid points: 17 500 lines reach every 256-point span, which selects the far kernel's dense shape
    # (one warp per CTA with a ring of its own, >= 1e4 lines per span) — config 3's launch configuration at a size the
    # checked build finishes in a moment; the near kernel lists hundreds of rounds of 32 lines per span
    import torch
    wl = workloads.small(seed=41, n_lines=1_000_000, nu_max=3000.0, cutoff=25.0, T=2500.0, P_atm=1.0 / workloads.BAR_PER_ATM,
                         logS=(-32.0, -20.0))
    T, P = wl.T[0], wl.P_atm[0]
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    got = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    got32 = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, precision=hk.HK_FP32)
    torch.cuda.synchronize()
    got, got32 = got.cpu().numpy(), got32.cpu().numpy()
    rng = np.random.default_rng(41)
    for s in np.concatenate(([0, wl.n_points - 48], rng.integers(0, wl.n_points - 48, 4))):
        js = np.arange(s, s + 48, dtype=np.int64)
        lo = np.searchsorted(wl.nu0, wl.nu_min + js[0] * wl.dnu - wl.cutoff - 1.0, "left")
        hi = np.searchsorted(wl.nu0, wl.nu_min + js[-1] * wl.dnu + wl.cutoff + 1.0, "right")
        ref = oracle.opacity_points(wl.nu0[lo:hi], wl.S[lo:hi], wl.gamma0[lo:hi], T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, js)
        assert np.abs(got[js] / ref - 1.0).max() <= 1e-6
        assert np.abs(got32[js] / ref - 1.0).max() <= 1e-4


def test_checked_build_runs_the_cases_without_a_trap(tmp_path):
    if os.environ.get("HK_LIB"):
        pytest.skip("already inside the child process")
    if not (shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc")):
        pytest.skip("nvcc is needed to compile the checked build")
    from paper_1503_03806_b200.build import build_library
    lib = build_library(force=True, out=str(tmp_path / "libhk_checked.so"), debug=True)
    env = dict(os.environ, HK_LIB=lib)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "gpu", "-p", "no:cacheprovider", *CASES], cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=900)
    tail = (r.stdout + r.stderr)[-4000:]
    assert r.returncode == 0, tail
    assert " passed" in r.stdout and "skipped" not in r.stdout.splitlines()[-1], tail
