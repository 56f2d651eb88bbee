"""ctypes binding of include/hk.h.  Same names as the C entry points; marshalling only."""
from __future__ import annotations

import ctypes as C
import os
import re
from dataclasses import dataclass

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# HK_LIB names another build of the library (tests/test_gpu_debug_build.py points it at the checked build); HK_DEBUG_CHECKS=1
# selects the in-tree checked build libhk_dbg.so (paper_1503_03806_b200.build)
LIB_PATH = os.environ.get("HK_LIB") or os.path.join(HERE, "libhk_dbg.so" if os.environ.get("HK_DEBUG_CHECKS") == "1" else "libhk.so")
HEADER = os.path.join(HERE, "..", "include", "hk.h")

HK_FP64, HK_FP32 = 0, 1
_dp = C.POINTER(C.c_double)
_i64 = C.c_int64


class HKError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        super().__init__(f"{where}: {hk_strerror(code)} ({code}){' — ' + detail if detail else ''}")


class _hk_lines(C.Structure):
    _fields_ = [("nu0", C.c_void_p), ("S", C.c_void_p), ("gamma0", C.c_void_p), ("n_T", C.c_void_p), ("E_low", C.c_void_p),
                ("gamma_self", C.c_void_p), ("A21", C.c_void_p), ("delta", C.c_void_p)]


class _hk_params(C.Structure):
    _fields_ = [("mass_amu", C.c_double), ("q_ratio", C.c_double), ("precision", C.c_int), ("lines_sorted", C.c_int),
                ("stream", C.c_void_p), ("self_fraction", C.c_double), ("abundance", C.c_double), ("cutoff_widths", C.c_double),
                ("accumulate", C.c_int)]


def _params(mass_amu, q_ratio, precision, lines_sorted, stream, self_fraction=0.5, abundance=1.0, accumulate=False,
            cutoff_widths=0.0):
    return _hk_params(float(mass_amu), float(q_ratio), int(precision), int(bool(lines_sorted)), _stream_ptr(stream),
                      float(self_fraction), float(abundance), float(cutoff_widths), int(bool(accumulate)))


_lib = None


def declared_symbols() -> list:
    """Entry points declared in include/hk.h (used by the CPU test that checks the library exports them all)."""
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(hk_[A-Za-z0-9_]+)\s*\(", txt)))


def load_library():
    """Loads libhk.so (built in-tree by paper_1503_03806_b200.build / __graft_entry__.build()).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.hk_grid_size.restype = _i64
    L.hk_grid_size.argtypes = [C.c_double] * 3
    L.hk_opacity.restype = C.c_int
    L.hk_opacity.argtypes = [C.POINTER(_hk_lines), _i64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                             C.c_double, C.c_void_p, C.POINTER(_hk_params)]
    L.hk_opacity_noalloc.restype = C.c_int
    L.hk_opacity_noalloc.argtypes = L.hk_opacity.argtypes
    L.hk_opacity_host.restype = C.c_int
    L.hk_opacity_host.argtypes = [C.POINTER(_hk_lines), _i64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                  C.c_double, C.c_void_p, C.c_double, C.c_int, C.c_void_p, C.POINTER(_hk_params)]
    L.hk_lines_check_sorted.restype = C.c_int
    L.hk_lines_check_sorted.argtypes = [C.c_void_p, _i64, C.c_void_p]
    L.hk_count_evals.restype = _i64
    L.hk_count_evals.argtypes = [_dp, _i64, C.c_double, _i64, C.c_double, C.c_double]
    L.hk_kdist.restype = C.c_int
    L.hk_kdist.argtypes = [C.c_void_p, _i64, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
    L.hk_kdist_cheb.restype = C.c_int
    L.hk_kdist_cheb.argtypes = [C.c_void_p, _i64, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
    L.hk_cheb_projection.restype = C.c_int
    L.hk_cheb_projection.argtypes = [C.c_int, C.c_int, _dp]
    L.hk_cheb_eval.restype = C.c_int
    L.hk_cheb_eval.argtypes = [C.c_void_p, _i64, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
    L.hk_transmission.restype = C.c_int
    L.hk_transmission.argtypes = [C.c_void_p, _i64, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
    L.hk_transmission_direct.restype = C.c_int
    L.hk_transmission_direct.argtypes = [C.c_void_p, _i64, C.c_double, C.c_double, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
    L.hk_regime_census.restype = C.c_int
    L.hk_regime_census.argtypes = [_dp, _dp, _i64, C.c_double, C.c_double, C.c_double, C.c_double, _i64, C.c_double,
                                   C.c_double, C.c_int, C.POINTER(_i64)]
    L.hk_gauss_legendre.restype = C.c_int
    L.hk_gauss_legendre.argtypes = [C.c_int, _dp, _dp]
    L.hk_voigt_K.restype = C.c_int
    L.hk_voigt_K.argtypes = [C.c_void_p, C.c_void_p, _i64, C.c_void_p, C.c_int, C.c_void_p]
    L.hk_create.restype = C.c_int
    L.hk_create.argtypes = [C.POINTER(_hk_lines), _i64, C.POINTER(_hk_params), C.POINTER(C.c_void_p)]
    L.hk_opacity_ctx.restype = C.c_int
    L.hk_opacity_ctx.argtypes = [C.c_void_p] + [C.c_double] * 7 + [C.c_void_p]
    L.hk_destroy.restype = C.c_int
    L.hk_destroy.argtypes = [C.c_void_p]
    L.hk_fp64_peak.restype = C.c_int
    L.hk_fp64_peak.argtypes = [_dp, C.c_void_p]
    L.hk_fp32_peak.restype = C.c_int
    L.hk_fp32_peak.argtypes = [_dp, C.c_void_p]
    L.hk_set_timing.restype = C.c_int
    L.hk_set_timing.argtypes = [C.c_int]
    L.hk_last_stage_ms.restype = C.c_int
    L.hk_last_stage_ms.argtypes = [C.POINTER(C.c_float)]
    L.hk_trim.restype = C.c_int
    L.hk_trim.argtypes = []
    L.hk_strerror.restype = C.c_char_p
    L.hk_strerror.argtypes = [C.c_int]
    L.hk_last_cuda_error.restype = C.c_char_p
    L.hk_version.restype = C.c_char_p
    _lib = L
    return L


def hk_strerror(code: int) -> str:
    try:
        return load_library().hk_strerror(int(code)).decode()
    except ImportError:
        return "libhk.so not loaded"


def hk_version() -> str:
    return load_library().hk_version().decode()


def _check(rc, where):
    if rc != 0:
        detail = load_library().hk_last_cuda_error().decode() if rc == -2 else ""
        raise HKError(rc, where, detail)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1503_03806_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _dev_ptr(t, name, allow_none=False):
    if t is None:
        if allow_none:
            return None
        raise ValueError(f"{name} is required")
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float64 CUDA tensor")
    return t.data_ptr()


def _stream_ptr(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


@dataclass
class Lines:
    """Line list on the device (hk_lines): float64 CUDA tensors of equal length."""
    nu0: object
    S: object
    gamma0: object
    n_T: object = None
    E_low: object = None
    gamma_self: object = None      # eq. 20: self broadening (gamma0 is then the air-broadening coefficient)
    A21: object = None             # eq. 20: Einstein A (natural width)
    delta: object = None           # eq. 21: pressure shift

    @staticmethod
    def from_numpy(nu0, S, gamma0, n_T=None, E_low=None, gamma_self=None, A21=None, delta=None, device="cuda"):
        torch = _torch()
        f = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(device)
        return Lines(f(nu0), f(S), f(gamma0), f(n_T), f(E_low), f(gamma_self), f(A21), f(delta))

    @property
    def n(self) -> int:
        return int(self.nu0.numel())

    def _c(self):
        n = self.n
        for name in ("S", "gamma0", "n_T", "E_low", "gamma_self", "A21", "delta"):
            t = getattr(self, name)
            if t is not None and int(t.numel()) != n:
                raise ValueError(f"{name} has {int(t.numel())} entries, nu0 has {n}")
        return _hk_lines(_dev_ptr(self.nu0, "nu0"), _dev_ptr(self.S, "S"), _dev_ptr(self.gamma0, "gamma0"),
                         _dev_ptr(self.n_T, "n_T", True), _dev_ptr(self.E_low, "E_low", True),
                         _dev_ptr(self.gamma_self, "gamma_self", True), _dev_ptr(self.A21, "A21", True),
                         _dev_ptr(self.delta, "delta", True))


def hk_grid_size(nu_min: float, nu_max: float, dnu: float) -> int:
    return int(load_library().hk_grid_size(nu_min, nu_max, dnu))


def hk_count_evals(nu0_host, nu_min: float, N: int, dnu: float, cutoff: float) -> int:
    a = np.ascontiguousarray(nu0_host, dtype=np.float64)
    return int(load_library().hk_count_evals(a.ctypes.data_as(_dp), a.size, nu_min, int(N), dnu, cutoff))


def hk_regime_census(nu0_host, gamma0_host, T, P_atm, mass_amu, nu_min, N, dnu, cutoff, precision=HK_FP64) -> dict:
    """Line-point evaluations per regime of the device Voigt routine (bench.py's roofline numerator).  Host arrays."""
    a = np.ascontiguousarray(nu0_host, dtype=np.float64)
    g = np.ascontiguousarray(gamma0_host, dtype=np.float64)
    if a.size != g.size:
        raise ValueError("nu0 and gamma0 differ in length")
    c = (_i64 * 5)()
    _check(load_library().hk_regime_census(a.ctypes.data_as(_dp), g.ctypes.data_as(_dp), a.size, T, P_atm, mass_amu, nu_min,
                                           int(N), dnu, cutoff, int(precision), c), "hk_regime_census")
    return dict(zip(("gh1", "gh2", "gh3", "gh6", "series"), (int(v) for v in c)))


def hk_gauss_legendre(n_g: int):
    g = np.empty(n_g)
    w = np.empty(n_g)
    _check(load_library().hk_gauss_legendre(int(n_g), g.ctypes.data_as(_dp), w.ctypes.data_as(_dp)), "hk_gauss_legendre")
    return g, w


def hk_opacity(lines: Lines, T, P_atm, nu_min, nu_max, dnu, cutoff, mass_amu=18.0, q_ratio=1.0, lines_sorted=True,
               out=None, stream=None, precision=HK_FP64, self_fraction=0.5, abundance=1.0, accumulate=False,
               cutoff_widths=0.0):
    """kappa[N] on the device (hk_opacity of include/hk.h).  Asynchronous on the current (or given) torch stream.
    accumulate=True adds abundance * kappa of this species to `out` (mixtures)."""
    torch = _torch()
    L = load_library()
    N = hk_grid_size(nu_min, nu_max, dnu)
    if out is None:
        if N < 1 or accumulate:
            raise HKError(-1, "hk_opacity")
        out = torch.empty(N, dtype=torch.float64, device=lines.nu0.device)
    elif N >= 1 and int(out.numel()) != N:       # (N < 1: let the library report HK_ERR_INVALID)
        raise ValueError(f"out has {int(out.numel())} entries, the grid has {N}")
    cl = lines._c()
    prm = _params(mass_amu, q_ratio, precision, lines_sorted, stream, self_fraction, abundance, accumulate, cutoff_widths)
    _check(L.hk_opacity(C.byref(cl), lines.n, T, P_atm, nu_min, nu_max, dnu, cutoff, _dev_ptr(out, "out"), C.byref(prm)),
           "hk_opacity")
    return out


HK_NOALLOC_MAX_LINES, HK_NOALLOC_MAX_POINTS = 65536, 4194304


def hk_opacity_noalloc(lines: Lines, T, P_atm, nu_min, nu_max, dnu, cutoff, out, mass_amu=18.0, q_ratio=1.0, stream=None,
                       precision=HK_FP64, self_fraction=0.5, abundance=1.0, accumulate=False, cutoff_widths=0.0):
    """hk_opacity for a caller that may not allocate GPU memory when it calls (its process gave the whole device to an arena
    of its own, or it sits in a latency-bound loop, or allocation after start-up is forbidden to it): hk_opacity_noalloc of
    include/hk.h.  Same kernels and bit-for-bit the same kappa as hk_opacity, with the library's work space in a fixed
    ~11 MiB array inside libhk.so instead of its memory pool.  `out` (float64 CUDA tensor, one entry per grid point) is
    required: this binding allocates nothing either.  At most HK_NOALLOC_MAX_LINES lines, ascending in nu0, no pressure
    shift (lines.delta), at most HK_NOALLOC_MAX_POINTS grid points; beyond that HKError (unsupported) names the limit.
    Asynchronous on the current (or given) torch stream.  All calls on a device share the one array: keep them on one
    stream or order them, overlapping calls corrupt each other.  Make the first call on a device at start-up (it does the
    one-time set-up), outside any stream capture."""
    L = load_library()
    N = hk_grid_size(nu_min, nu_max, dnu)
    if out is None:
        raise ValueError("out is required: hk_opacity_noalloc allocates nothing")
    if N >= 1 and int(out.numel()) != N:
        raise ValueError(f"out has {int(out.numel())} entries, the grid has {N}")
    cl = lines._c()
    prm = _params(mass_amu, q_ratio, precision, True, stream, self_fraction, abundance, accumulate, cutoff_widths)
    rc = L.hk_opacity_noalloc(C.byref(cl), lines.n, T, P_atm, nu_min, nu_max, dnu, cutoff, _dev_ptr(out, "out"), C.byref(prm))
    if rc == -5:
        raise HKError(rc, "hk_opacity_noalloc", L.hk_last_cuda_error().decode())
    _check(rc, "hk_opacity_noalloc")
    return out


def hk_kdist(kappa, dnu, bin_width, n_g, out=None, stream=None):
    """k_out[n_bins, n_g] on the device (hk_kdist of include/hk.h)."""
    torch = _torch()
    L = load_library()
    n = int(kappa.numel())
    ppb = int(round(bin_width / dnu))
    if out is None:
        if ppb < 1 or n % ppb or n_g < 1:
            raise HKError(-1, "hk_kdist")
        out = torch.empty((n // ppb, n_g), dtype=torch.float64, device=kappa.device)
    _check(L.hk_kdist(_dev_ptr(kappa, "kappa"), n, dnu, bin_width, int(n_g), _dev_ptr(out, "out"), _stream_ptr(stream)),
           "hk_kdist")
    return out


def hk_kdist_cheb(kappa, dnu, bin_width, n_c=20, n_g=None, stream=None):
    """Chebyshev coefficients [n_bins, n_c] of ln kappa(y) per bin (hk_kdist_cheb); with n_g also the Gauss-Legendre k-table
    [n_bins, n_g] from the same launch.  Returns coef, or (coef, k_table)."""
    torch = _torch()
    n = int(kappa.numel())
    ppb = int(round(bin_width / dnu))
    if ppb < 1 or n % ppb or n_c < 1:
        raise HKError(-1, "hk_kdist_cheb")
    coef = torch.empty((n // ppb, n_c), dtype=torch.float64, device=kappa.device)
    ktab = None if n_g is None else torch.empty((n // ppb, n_g), dtype=torch.float64, device=kappa.device)
    _check(load_library().hk_kdist_cheb(_dev_ptr(kappa, "kappa"), n, dnu, bin_width, int(n_c), _dev_ptr(coef, "coef"),
                                        int(n_g or 0), _dev_ptr(ktab, "k_out", True), _stream_ptr(stream)), "hk_kdist_cheb")
    return coef if ktab is None else (coef, ktab)


def hk_cheb_projection(ppb: int, n_c: int):
    """P[n_c, ppb] with C = P D, the host-side Q-R product hk_kdist_cheb uploads (host arithmetic, no GPU needed)."""
    P = np.empty((int(n_c), int(ppb)))
    _check(load_library().hk_cheb_projection(int(ppb), int(n_c), P.ctypes.data_as(_dp)), "hk_cheb_projection")
    return P


def hk_cheb_eval(coef, y, stream=None):
    """kappa(y) [n_bins, n_y] reconstructed from Chebyshev coefficients [n_bins, n_c] (hk_cheb_eval)."""
    torch = _torch()
    n_bins, n_c = (int(v) for v in coef.shape)
    out = torch.empty((n_bins, int(y.numel())), dtype=torch.float64, device=coef.device)
    _check(load_library().hk_cheb_eval(_dev_ptr(coef, "coef"), n_bins, n_c, _dev_ptr(y, "y"), int(y.numel()),
                                       _dev_ptr(out, "out"), _stream_ptr(stream)), "hk_cheb_eval")
    return out


def hk_transmission(k_table, mcol, stream=None):
    """T[n_bins, n_m] = sum_q w_q exp(-k_table[b][q] m~) (hk_transmission; eq. 5 on the k-distribution side)."""
    torch = _torch()
    n_bins, n_g = (int(v) for v in k_table.shape)
    out = torch.empty((n_bins, int(mcol.numel())), dtype=torch.float64, device=k_table.device)
    _check(load_library().hk_transmission(_dev_ptr(k_table, "k_table"), n_bins, n_g, _dev_ptr(mcol, "mcol"), int(mcol.numel()),
                                          _dev_ptr(out, "out"), _stream_ptr(stream)), "hk_transmission")
    return out


def hk_transmission_direct(kappa, dnu, bin_width, mcol, stream=None):
    """T[n_bins, n_m] = mean over each bin's grid points of exp(-kappa_j m~) (hk_transmission_direct; eq. 5, Riemann side)."""
    torch = _torch()
    n = int(kappa.numel())
    ppb = int(round(bin_width / dnu))
    if ppb < 1 or n % ppb:
        raise HKError(-1, "hk_transmission_direct")
    out = torch.empty((n // ppb, int(mcol.numel())), dtype=torch.float64, device=kappa.device)
    _check(load_library().hk_transmission_direct(_dev_ptr(kappa, "kappa"), n, dnu, bin_width, _dev_ptr(mcol, "mcol"),
                                                 int(mcol.numel()), _dev_ptr(out, "out"), _stream_ptr(stream)),
           "hk_transmission_direct")
    return out


def hk_voigt_K(x, y, out=None, stream=None, precision=HK_FP64):
    """K(x,y) = Re w(x+iy) through the device Voigt routine (test hook)."""
    torch = _torch()
    if out is None:
        out = torch.empty_like(x)
    _check(load_library().hk_voigt_K(_dev_ptr(x, "x"), _dev_ptr(y, "y"), int(x.numel()), _dev_ptr(out, "out"),
                                     int(precision), _stream_ptr(stream)), "hk_voigt_K")
    return out


def hk_lines_check_sorted(nu0, stream=None) -> bool:
    rc = load_library().hk_lines_check_sorted(_dev_ptr(nu0, "nu0"), int(nu0.numel()), _stream_ptr(stream))
    if rc == -4:
        return False
    _check(rc, "hk_lines_check_sorted")
    return True


def hk_fp64_peak(stream=None) -> float:
    """Measured FP64 FMA thread-instructions per second of this GPU (roofline denominator, measured live)."""
    v = C.c_double(0.0)
    _check(load_library().hk_fp64_peak(C.byref(v), _stream_ptr(stream)), "hk_fp64_peak")
    return v.value


def hk_fp32_peak(stream=None) -> float:
    """Measured FP32 FMA thread-instructions per second of this GPU (roofline denominator of the FP32 variant)."""
    v = C.c_double(0.0)
    _check(load_library().hk_fp32_peak(C.byref(v), _stream_ptr(stream)), "hk_fp32_peak")
    return v.value


def hk_trim() -> None:
    _check(load_library().hk_trim(), "hk_trim")


def hk_set_timing(on: bool) -> None:
    _check(load_library().hk_set_timing(int(bool(on))), "hk_set_timing")


def hk_last_stage_ms():
    a = (C.c_float * 3)()
    _check(load_library().hk_last_stage_ms(a), "hk_last_stage_ms")
    return [float(v) for v in a]


class Context:
    """hk_create / hk_opacity_ctx / hk_destroy: line list bound once, scratch kept across (T,P) calls.

    A Context is bound to ONE stream, the one given (or current) at creation: opacity() launches on it and allocates its
    result under it, whatever stream is current at the time of the call; a consumer on another stream has to wait for it."""

    def __init__(self, lines: Lines, mass_amu=18.0, lines_sorted=True, stream=None, precision=HK_FP64, self_fraction=0.5,
                 abundance=1.0, accumulate=False, cutoff_widths=0.0):
        self._lines = lines      # keep the tensors alive
        self._stream = stream if stream is not None else _torch().cuda.current_stream()
        stream = self._stream
        self._h = C.c_void_p()
        cl = lines._c()
        prm = _params(mass_amu, 1.0, precision, lines_sorted, stream, self_fraction, abundance, accumulate, cutoff_widths)
        _check(load_library().hk_create(C.byref(cl), lines.n, C.byref(prm), C.byref(self._h)), "hk_create")

    def opacity(self, T, P_atm, nu_min, nu_max, dnu, cutoff, q_ratio=1.0, out=None):
        torch = _torch()
        N = hk_grid_size(nu_min, nu_max, dnu)
        if out is None:
            with torch.cuda.stream(self._stream):
                out = torch.empty(N, dtype=torch.float64, device=self._lines.nu0.device)
        _check(load_library().hk_opacity_ctx(self._h, T, P_atm, q_ratio, nu_min, nu_max, dnu, cutoff, _dev_ptr(out, "out")),
               "hk_opacity_ctx")
        return out

    def close(self):
        if self._h:
            load_library().hk_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _host_ptr(t, name, allow_none=False):
    if t is None:
        if allow_none:
            return None
        raise ValueError(f"{name} is required")
    import torch
    if isinstance(t, np.ndarray):
        if t.dtype != np.float64 or not t.flags.c_contiguous:
            raise TypeError(f"{name} must be a contiguous float64 array")
        return t.ctypes.data
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float64 HOST tensor or numpy array")
    return t.data_ptr()


def hk_opacity_host(nu0, S, gamma0, T, P_atm, nu_min, nu_max, dnu, cutoff, mass_amu=18.0, n_T=None, E_low=None, q_ratio=1.0,
                    lines_sorted=True, bin_width=None, n_g=20, kappa_out=None, k_out=None, want_kappa=True, stream=None,
                    precision=HK_FP64, gamma_self=None, A21=None, delta=None, self_fraction=0.5, abundance=1.0,
                    accumulate=False, cutoff_widths=0.0):
    """End-to-end call with HOST buffers (hk_opacity_host of include/hk.h): host line arrays -> device, hk_opacity
    (+ hk_kdist when bin_width is given), kappa / k-table -> host.  Buffers are host torch tensors (pinned for
    asynchronous copies) or numpy arrays.  Returns (kappa_host or None, k_host or None).  Synchronous."""
    torch = _torch()
    L = load_library()
    N = hk_grid_size(nu_min, nu_max, dnu)
    n = int(nu0.shape[0])
    for name, t in (("S", S), ("gamma0", gamma0), ("n_T", n_T), ("E_low", E_low), ("gamma_self", gamma_self), ("A21", A21),
                    ("delta", delta)):
        if t is not None and int(t.shape[0]) != n:
            raise ValueError(f"{name} has {int(t.shape[0])} entries, nu0 has {n}")
    if want_kappa and kappa_out is None and N >= 1:
        kappa_out = torch.empty(N, dtype=torch.float64, pin_memory=True)
    if kappa_out is not None and N >= 1 and int(kappa_out.shape[0]) != N:
        raise ValueError(f"kappa_out has {int(kappa_out.shape[0])} entries, the grid has {N}")
    if bin_width is not None:
        ppb = int(round(bin_width / dnu))
        if ppb < 1 or N < 1 or N % ppb or n_g < 1:
            raise HKError(-1, "hk_opacity_host")
        if k_out is None:
            k_out = torch.empty((N // ppb, n_g), dtype=torch.float64, pin_memory=True)
        elif tuple(k_out.shape) != (N // ppb, n_g):
            raise ValueError(f"k_out has shape {tuple(k_out.shape)}, expected {(N // ppb, n_g)}")
    else:
        k_out = None
    cl = _hk_lines(_host_ptr(nu0, "nu0"), _host_ptr(S, "S"), _host_ptr(gamma0, "gamma0"), _host_ptr(n_T, "n_T", True),
                   _host_ptr(E_low, "E_low", True), _host_ptr(gamma_self, "gamma_self", True), _host_ptr(A21, "A21", True),
                   _host_ptr(delta, "delta", True))
    prm = _params(mass_amu, q_ratio, precision, lines_sorted, stream, self_fraction, abundance, accumulate, cutoff_widths)
    _check(L.hk_opacity_host(C.byref(cl), n, T, P_atm, nu_min, nu_max, dnu, cutoff, _host_ptr(kappa_out, "kappa_out", True),
                             float(bin_width or 0.0), int(n_g), _host_ptr(k_out, "k_out", True), C.byref(prm)),
           "hk_opacity_host")
    return kappa_out, k_out
