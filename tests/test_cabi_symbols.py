"""The C-ABI library loads and exports every symbol include/hk.h declares; host-only entry points work (no GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1503_03806_b200 as hk


@pytest.fixture(scope="module")
def lib():
    from paper_1503_03806_b200.build import build_library
    build_library()
    return hk.load_library()


def test_exports_every_declared_symbol(lib):
    names = hk.declared_symbols()
    assert {"hk_opacity", "hk_kdist", "hk_voigt_K", "hk_gauss_legendre", "hk_count_evals", "hk_grid_size",
            "hk_create", "hk_opacity_ctx", "hk_destroy", "hk_strerror"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_sass_is_sm100a_with_tma_bulk_copy(lib):
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    from paper_1503_03806_b200._binding import LIB_PATH
    out = subprocess.run([cuobjdump, "-sass", LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert "UBLKCP" in out          # cp.async.bulk (1-D TMA) stages the line records
    assert "MUFU.RCP64H" in out     # FP64 reciprocal seed
    assert "DFMA" in out


def test_grid_size_host():
    assert hk.hk_grid_size(0.0, 3000.0, 0.01) == 300000
    assert hk.hk_grid_size(0.0, 30000.0, 0.01) == 3000000
    assert hk.hk_grid_size(0.0, 1.0, 0.0) == -1


def test_gauss_legendre_host():
    for n in (1, 2, 3, 20, 64, 128):
        g, w = hk.hk_gauss_legendre(n)
        t, wt = np.polynomial.legendre.leggauss(n)
        assert np.abs(g - 0.5 * (1 + t)).max() < 1e-15
        assert np.abs(w - 0.5 * wt).max() < 1e-14
        assert abs(w.sum() - 1.0) < 1e-14
    g, w = hk.hk_gauss_legendre(20)
    for p in range(40):
        assert abs(np.sum(w * g ** p) - 1.0 / (p + 1)) < 1e-14
    with pytest.raises(hk.HKError):
        hk.hk_gauss_legendre(0)


def test_count_evals_host_bruteforce():
    rng = np.random.default_rng(0)
    nu0 = rng.uniform(-30.0, 130.0, 500)
    N, dnu, cutoff = 10000, 0.01, 25.0
    nu = np.arange(N) * dnu
    brute = sum(int(np.count_nonzero(np.abs(nu - c) <= cutoff)) for c in nu0)
    assert hk.hk_count_evals(nu0, 0.0, N, dnu, cutoff) == brute
    assert hk.hk_count_evals([50.0], 0.0, N, dnu, cutoff) == 5001


def test_strerror_and_version():
    assert hk.hk_strerror(0) == "ok"
    assert "invalid" in hk.hk_strerror(-1)
    assert "sm_100a" in hk.hk_version()


def test_compute_call_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        hk.hk_fp64_peak()
    with pytest.raises(RuntimeError):
        hk.Lines.from_numpy([1.0], [1.0], [0.05])


@pytest.mark.parametrize("ppb,n_c", [(1000, 20), (10000, 20), (37, 5), (64, 8), (20, 20)])
def test_cheb_projection_host_against_the_oracle(ppb, n_c):
    # host logic of hk_kdist_cheb (Householder Q-R in long double): C = P D must be the least-squares solution
    import oracle
    from paper_1503_03806_b200.build import build_library
    build_library()
    P = hk.hk_cheb_projection(ppb, n_c)
    assert P.shape == (n_c, ppb)
    A = oracle.cheb_design(ppb, n_c)
    tol = 1e-9 if n_c < ppb else 1e-4         # as many polynomials as equispaced points: interpolation, cond(A) ~ 1e9
    assert np.abs(P @ A - np.eye(n_c)).max() < tol                                   # left inverse of the design matrix
    rng = np.random.default_rng(ppb)
    kappa = np.sort(10 ** rng.uniform(-8, 4, ppb))
    C = oracle.kdist_cheb(kappa, ppb, n_c)[0]
    assert np.abs(P @ np.log(kappa) - C).max() < tol * max(1.0, np.abs(C).max())
    with pytest.raises(hk.HKError):
        hk.hk_cheb_projection(10, 20)


def test_sass_of_the_hot_kernels():
    """What the kernels are claimed to be built from shows in the SASS of libhk.so (cuobjdump works without a GPU): the far
    kernel stages line records by 1-D TMA bulk copies completing on mbarriers (UBLKCP, SYNCS) and takes FP64 reciprocals from
    MUFU.RCP64H; the FP32 variant's far kernel uses sm_100's packed float arithmetic (FFMA2 / FMUL2 / FADD2)."""
    import shutil
    import subprocess
    from paper_1503_03806_b200.build import build_library
    from paper_1503_03806_b200.build import is_stale, LIB
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    filt = shutil.which("cu++filt") or "/usr/local/cuda/bin/cu++filt"
    if not (os.path.exists(cuobjdump) and os.path.exists(filt)):
        pytest.skip("cuobjdump / cu++filt not available")
    have_nvcc = bool(shutil.which("nvcc")) or os.path.exists("/usr/local/cuda/bin/nvcc")
    if not have_nvcc and is_stale():
        pytest.skip("no nvcc and no up-to-date libhk.so to inspect")
    lib = build_library() if have_nvcc else LIB
    sass = subprocess.run([cuobjdump, "-sass", lib], capture_output=True, text=True, check=True).stdout
    funcs = {}
    name = None
    for line in sass.splitlines():
        if "Function :" in line:
            name = line.split("Function :")[1].strip()
            funcs[name] = []
        elif name is not None:
            funcs[name].append(line)
    # demangled names: the last template argument of FarShape says FP32 variant or not ("(bool)1" / "true")
    names = list(funcs)
    plain = subprocess.run([filt], input="\n".join(names), capture_output=True, text=True, check=True).stdout.splitlines()
    assert len(plain) == len(names)
    funcs = {p: funcs[n] for n, p in zip(names, plain)}
    far = {n: "\n".join(b) for n, b in funcs.items() if "voigt_far_kernel" in n}
    assert len(far) == 3, sorted(far)                                 # sparse and dense FP64 shapes, FP32 variant
    for n, body in far.items():
        assert "UBLKCP" in body and "SYNCS" in body, n                # TMA bulk copy + mbarrier
    is32 = lambda n: re.search(r"(\(bool\)\s*1|true)\s*>\s*>", n) is not None
    f32 = [b for n, b in far.items() if is32(n)]
    f64 = [b for n, b in far.items() if not is32(n)]
    assert len(f32) == 1 and len(f64) == 2
    assert all(k in f32[0] for k in ("FFMA2", "FMUL2", "FADD2"))
    assert all("MUFU.RCP64H" in b and "DFMA" in b for b in f64)
    near = [("\n".join(b)) for n, b in funcs.items() if "voigt_near_kernel" in n]
    assert len(near) == 1 and "DFMA" in near[0] and "LDGSTS" in near[0]   # cp.async prefetch of the kappa strip
