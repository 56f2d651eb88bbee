"""CPU oracle (TEST INFRASTRUCTURE — see the header of hk_oracle.c).

Thin ctypes wrapper around `oracle/hk_oracle.c`.  Only tests/, `__graft_entry__.smoke()` and
bench.py's cpu_baseline / `--impl reference` leg may import this module; the CUDA path under
`paper_1503_03806_b200/` never does, and this module never imports that package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hk_oracle.c")
_LIB = os.path.join(_HERE, "libhk_oracle.so")
_lib = None

_dp = C.POINTER(C.c_double)
_i64 = C.c_int64


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP).  No fast-math: the arithmetic is as written."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_faddeeva_re.restype = C.c_double
        L.orc_faddeeva_re.argtypes = [C.c_double, C.c_double]
        L.orc_voigt_K.restype = None
        L.orc_voigt_K.argtypes = [_dp, _dp, _i64, _dp]
        L.orc_voigt_V.restype = C.c_double
        L.orc_voigt_V.argtypes = [C.c_double] * 3
        L.orc_line_strength.restype = C.c_double
        L.orc_line_strength.argtypes = [C.c_double] * 5
        L.orc_gauss_legendre.restype = C.c_int
        L.orc_gauss_legendre.argtypes = [C.c_int, _dp, _dp]
        L.orc_count_evals.restype = _i64
        L.orc_count_evals.argtypes = [_dp, _i64, C.c_double, _i64, C.c_double, C.c_double]
        L.orc_opacity.restype = C.c_int
        L.orc_opacity.argtypes = [_dp, _dp, _dp, _dp, _dp, _i64, C.c_double, C.c_double, C.c_double, _i64,
                                  C.c_double, C.c_double, C.c_double, C.c_double, _i64, _i64, _dp]
        L.orc_opacity_points.restype = C.c_int
        L.orc_opacity_points.argtypes = [_dp, _dp, _dp, _dp, _dp, _i64, C.c_double, C.c_double, C.c_double, _i64,
                                         C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(_i64), _i64, _dp]
        L.orc_opacity_points_full.restype = C.c_int
        L.orc_opacity_points_full.argtypes = [_dp] * 8 + [_i64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                              _i64, C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(_i64), _i64, _dp]
        L.orc_opacity_points_rel.restype = C.c_int
        L.orc_opacity_points_rel.argtypes = [_dp] * 8 + [_i64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                             _i64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                             C.POINTER(_i64), _i64, _dp]
        L.orc_kdist.restype = C.c_int
        L.orc_kdist.argtypes = [_dp, _i64, _i64, C.c_int, _dp]
        _lib = L
    return _lib


def _arr(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def set_threads(n: int) -> None:
    """Number of OpenMP threads the oracle uses (default: all cores)."""
    os.environ["OMP_NUM_THREADS"] = str(n)
    try:
        C.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
    except OSError:
        pass


def faddeeva_re(x, y):
    """K(x,y) = Re w(x+iy), elementwise (H_V is the real part of the Faddeeva function)."""
    x, y = np.broadcast_arrays(_arr(x), _arr(y))
    x, y = _arr(x), _arr(y)
    out = np.empty(x.shape, dtype=np.float64)
    lib().orc_voigt_K(_p(x), _p(y), x.size, _p(out))
    return out


def voigt_V(dv: float, alpha: float, gamma: float) -> float:
    """V(dv; alpha, gamma) = K(dv/alpha, gamma/alpha)/(alpha sqrt(pi))  (eq. 19)."""
    return lib().orc_voigt_V(float(dv), float(alpha), float(gamma))


def line_strength(S, nu0, E_low, T, q_ratio) -> float:
    """S(T) from S(296 K), eq. 18 in the DESIGN.md G1 reading."""
    return lib().orc_line_strength(float(S), float(nu0), float(E_low), float(T), float(q_ratio))


def gauss_legendre(n_g: int):
    g = np.empty(n_g)
    w = np.empty(n_g)
    rc = lib().orc_gauss_legendre(int(n_g), _p(g), _p(w))
    if rc != 0:
        raise ValueError(f"orc_gauss_legendre: {rc}")
    return g, w


def grid_size(nu_min: float, nu_max: float, dnu: float) -> int:
    return int(round((nu_max - nu_min) / dnu))


def count_evals(nu0, nu_min, N, dnu, cutoff) -> int:
    nu0 = _arr(nu0)
    return int(lib().orc_count_evals(_p(nu0), nu0.size, nu_min, int(N), dnu, cutoff))


def opacity(nu0, S, gamma0, T, P_atm, nu_min, nu_max, dnu, cutoff, mass_amu=18.0, n_T=None, E_low=None,
            q_ratio=1.0, j_begin=0, j_end=None):
    """kappa(nu_j), j in [j_begin, j_end), on nu_j = nu_min + j*dnu  (eq. 16 + 19)."""
    nu0, S, gamma0 = _arr(nu0), _arr(S), _arr(gamma0)
    n_T = None if n_T is None else _arr(n_T)
    E_low = None if E_low is None else _arr(E_low)
    N = grid_size(nu_min, nu_max, dnu)
    if j_end is None:
        j_end = N
    out = np.empty(max(j_end - j_begin, 0), dtype=np.float64)
    rc = lib().orc_opacity(_p(nu0), _p(S), _p(gamma0), _p(n_T), _p(E_low), nu0.size, T, P_atm, nu_min, N, dnu, cutoff,
                           mass_amu, q_ratio, j_begin, j_end, _p(out))
    if rc != 0:
        raise ValueError(f"orc_opacity: error {rc}")
    return out


def opacity_points(nu0, S, gamma0, T, P_atm, nu_min, nu_max, dnu, cutoff, js, mass_amu=18.0, n_T=None, E_low=None,
                   q_ratio=1.0):
    """kappa at an arbitrary list of grid indices `js` (same definition as `opacity`)."""
    nu0, S, gamma0 = _arr(nu0), _arr(S), _arr(gamma0)
    n_T = None if n_T is None else _arr(n_T)
    E_low = None if E_low is None else _arr(E_low)
    js = np.ascontiguousarray(js, dtype=np.int64)
    N = grid_size(nu_min, nu_max, dnu)
    out = np.empty(js.size, dtype=np.float64)
    rc = lib().orc_opacity_points(_p(nu0), _p(S), _p(gamma0), _p(n_T), _p(E_low), nu0.size, T, P_atm, nu_min, N, dnu,
                                  cutoff, mass_amu, q_ratio, js.ctypes.data_as(C.POINTER(_i64)), js.size, _p(out))
    if rc != 0:
        raise ValueError(f"orc_opacity_points: error {rc}")
    return out


def opacity_full(nu0, S, gamma_air, T, P_atm, nu_min, nu_max, dnu, cutoff, mass_amu=18.0, gamma_self=None, A21=None,
                 delta=None, n_T=None, E_low=None, q_ratio=1.0, self_fraction=0.5, abundance=1.0, js=None,
                 cutoff_widths=0.0):
    """kappa with the full line physics of eqs. 20-21 and an abundance weight;
    on the whole grid, or at the grid indices `js`.  cutoff_widths > 0: line i is truncated at
    min(cutoff, cutoff_widths * gamma_i) ("500 Lorentz widths")."""
    f = lambda a: None if a is None else _arr(a)
    nu0, S, gamma_air = _arr(nu0), _arr(S), _arr(gamma_air)
    gamma_self, A21, delta, n_T, E_low = f(gamma_self), f(A21), f(delta), f(n_T), f(E_low)
    N = grid_size(nu_min, nu_max, dnu)
    js = np.arange(N, dtype=np.int64) if js is None else np.ascontiguousarray(js, dtype=np.int64)
    out = np.empty(js.size, dtype=np.float64)
    rc = lib().orc_opacity_points_rel(_p(nu0), _p(S), _p(gamma_air), _p(gamma_self), _p(A21), _p(delta), _p(n_T), _p(E_low),
                                      nu0.size, T, P_atm, self_fraction, abundance, nu_min, N, dnu, cutoff, cutoff_widths,
                                      mass_amu, q_ratio, js.ctypes.data_as(C.POINTER(_i64)), js.size, _p(out))
    if rc != 0:
        raise ValueError(f"orc_opacity_points_rel: error {rc}")
    return out


def kdist(kappa, ppb: int, n_g: int):
    """k_out[n_bins, n_g]: per-bin sorted kappa resampled at the Gauss-Legendre nodes (eqs. 14-15)."""
    kappa = _arr(kappa)
    if kappa.size % ppb:
        raise ValueError("n_points is not a multiple of ppb")
    out = np.empty((kappa.size // ppb, n_g), dtype=np.float64)
    rc = lib().orc_kdist(_p(kappa), kappa.size, int(ppb), int(n_g), _p(out))
    if rc != 0:
        raise ValueError(f"orc_kdist: error {rc}")
    return out


# ---------------------------------------------------------------------------------------------------------
# SURVEY.md §8(f) "next" rows: Chebyshev resampling (f1) and the transmission function (f2).  Plain numpy, FP64.
# ---------------------------------------------------------------------------------------------------------
KAPPA_FLOOR = 1.0e-300   # DESIGN.md reading C1: ln(kappa) is taken of max(kappa, 1e-300) (the paper is silent on kappa = 0)


def cheb_design(ppb: int, n_c: int):
    """A[k][n] = T_n(2 y_k - 1) at the cell centres y_k = (k + 1/2)/ppb (A7), by the recurrence
    T_0 = 1, T_1 = t, T_{n+1} = 2 t T_n - T_{n-1}  ("exploit the recurrence relations")."""
    t = 2.0 * ((np.arange(ppb) + 0.5) / ppb) - 1.0
    A = np.empty((ppb, n_c))
    A[:, 0] = 1.0
    if n_c > 1:
        A[:, 1] = t
    for n in range(2, n_c):
        A[:, n] = 2.0 * t * A[:, n - 1] - A[:, n - 2]
    return A


def kdist_cheb(kappa, ppb: int, n_c: int):
    """C[n_bins, n_c]: least-squares fit of ln kappa(y) of every bin with n_c Chebyshev polynomials, solved through the
    Q-R decomposition of the design matrix ("solving A C = D ... we implement Q-R decomposition")."""
    kappa = _arr(kappa)
    if kappa.size % ppb:
        raise ValueError("n_points is not a multiple of ppb")
    A = cheb_design(ppb, n_c)
    Q, R = np.linalg.qr(A)                                    # library primitive (LAPACK Householder QR), thin form
    out = np.empty((kappa.size // ppb, n_c))
    for b in range(kappa.size // ppb):
        s = np.sort(kappa[b * ppb:(b + 1) * ppb])             # kappa(y) of the bin (eqs. 14-15)
        D = np.log(np.maximum(s, KAPPA_FLOOR))
        out[b] = np.linalg.solve(R, Q.T @ D)                  # R C = Q^T D
    return out


def cheb_eval(C, y):
    """kappa(y) = exp(sum_n C_n T_n(2y - 1)) for every bin (rows of C) at the abscissae y in [0,1]."""
    C = np.atleast_2d(_arr(C))
    y = _arr(y)
    t = 2.0 * y - 1.0
    T = np.empty((y.size, C.shape[1]))
    T[:, 0] = 1.0
    if C.shape[1] > 1:
        T[:, 1] = t
    for n in range(2, C.shape[1]):
        T[:, n] = 2.0 * t * T[:, n - 1] - T[:, n - 2]
    return np.exp(C @ T.T)


def transmission_kdist(k_table, mcol):
    """T[b][m] = int_0^1 exp(-kappa(y) m~) dy (eq. 5, second equality) by the Gauss-Legendre rule whose nodes
    the k-table holds: sum_q w_q exp(-k[b][q] m~_m)."""
    k_table = np.atleast_2d(_arr(k_table))
    mcol = _arr(mcol)
    _, w = gauss_legendre(k_table.shape[1])
    return np.einsum("q,bqm->bm", w, np.exp(-k_table[:, :, None] * mcol[None, None, :]))


def transmission_direct(kappa, ppb: int, mcol):
    """T[b][m] = (1/Delta x) int exp(-kappa(x) m~) dx over the bin (eq. 5, first equality), on the grid: the mean of
    exp(-kappa_j m~_m) over the bin's ppb points (each point stands for delta x)."""
    kappa = _arr(kappa)
    mcol = _arr(mcol)
    if kappa.size % ppb:
        raise ValueError("n_points is not a multiple of ppb")
    kb = kappa.reshape(-1, ppb)
    out = np.empty((kb.shape[0], mcol.size))
    for b in range(kb.shape[0]):
        out[b] = np.exp(-kb[b][:, None] * mcol[None, :]).mean(axis=0)
    return out
