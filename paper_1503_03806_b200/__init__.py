"""paper_1503_03806_b200 — B200-native HELIOS-K hot path (Grimm & Heng 2015, arXiv:1503.03806).

Thin Python binding over the C ABI of include/hk.h (libhk.so, hand-written sm_100a CUDA).  Argument marshalling
only: every step of the path runs in the library's kernels.  PyTorch supplies device memory and streams.
There is no CPU fallback: importing works without a GPU (so the symbols can be inspected), but every compute
call raises if the library or a CUDA device is missing.
"""
from ._binding import (HKError, Lines, Context, load_library, declared_symbols, hk_grid_size, hk_count_evals, hk_regime_census,
                       hk_gauss_legendre, hk_opacity, hk_kdist, hk_voigt_K, hk_lines_check_sorted, hk_fp64_peak, hk_fp32_peak,
                       hk_set_timing, hk_trim, hk_last_stage_ms, hk_strerror, hk_version, hk_opacity_host, hk_kdist_cheb, hk_cheb_projection, hk_cheb_eval, hk_transmission,
                       hk_transmission_direct, HK_FP64, HK_FP32, hk_opacity_noalloc, HK_NOALLOC_MAX_LINES,
                       HK_NOALLOC_MAX_POINTS)

__all__ = ["HKError", "Lines", "Context", "load_library", "declared_symbols", "hk_grid_size", "hk_count_evals", "hk_regime_census",
           "hk_gauss_legendre", "hk_opacity", "hk_kdist", "hk_voigt_K", "hk_lines_check_sorted", "hk_fp64_peak", "hk_fp32_peak",
           "hk_set_timing", "hk_trim", "hk_last_stage_ms", "hk_strerror", "hk_version", "hk_opacity_host", "hk_kdist_cheb", "hk_cheb_projection", "hk_cheb_eval", "hk_transmission",
           "hk_transmission_direct", "HK_FP64", "HK_FP32", "hk_opacity_noalloc", "HK_NOALLOC_MAX_LINES", "HK_NOALLOC_MAX_POINTS"]
