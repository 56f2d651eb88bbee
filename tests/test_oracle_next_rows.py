"""Pins for the oracle's SURVEY §8(f) rows: Chebyshev resampling of ln kappa(y) and the transmission
function (eq. 5).  Closed forms, library routines of a different algorithm, invariants."""
import numpy as np
import pytest

import oracle


# ---- f1: Chebyshev least-squares fit -----------------------------------------------------------------------------------
def test_design_matrix_is_chebyshev():
    A = oracle.cheb_design(50, 7)
    t = 2.0 * (np.arange(50) + 0.5) / 50 - 1.0
    for n in range(7):
        assert np.allclose(A[:, n], np.cos(n * np.arccos(t)), atol=1e-13)          # T_n(cos th) = cos(n th)


def test_polynomial_ln_kappa_is_recovered_exactly():
    # ln kappa(y) = a polynomial of degree < n_c in t = 2y - 1, monotone increasing so that the sort is the identity
    ppb, n_c = 1000, 20
    t = 2.0 * (np.arange(ppb) + 0.5) / ppb - 1.0
    c_true = np.zeros(n_c)
    c_true[:6] = [-3.0, 4.0, 0.3, 0.2, -0.05, 0.02]
    lnk = np.polynomial.chebyshev.chebval(t, c_true)
    assert np.all(np.diff(lnk) > 0)
    rng = np.random.default_rng(0)
    kappa = np.exp(lnk)[rng.permutation(ppb)]                                       # order within the bin must not matter
    C = oracle.kdist_cheb(kappa, ppb, n_c)
    assert C.shape == (1, n_c)
    assert np.abs(C[0] - c_true).max() < 1e-11


@pytest.mark.parametrize("ppb,n_c", [(1000, 20), (10000, 20), (100, 8), (64, 1)])
def test_against_numpy_chebfit_and_normal_equations(ppb, n_c):
    rng = np.random.default_rng(ppb)
    kappa = 10 ** rng.uniform(-8, 4, 3 * ppb)
    C = oracle.kdist_cheb(kappa, ppb, n_c)
    A = oracle.cheb_design(ppb, n_c)
    t = 2.0 * (np.arange(ppb) + 0.5) / ppb - 1.0
    for b in range(3):
        D = np.log(np.sort(kappa[b * ppb:(b + 1) * ppb]))
        ref = np.polynomial.chebyshev.chebfit(t, D, n_c - 1)                        # library least squares (SVD, scaled columns)
        assert np.abs(C[b] - ref).max() < 1e-9 * max(1.0, np.abs(ref).max())
        r = A @ C[b] - D
        assert np.abs(A.T @ r).max() < 1e-8 * np.abs(D).sum()                       # residual orthogonal to the basis


def test_constant_bin_and_floor():
    C = oracle.kdist_cheb(np.full(500, 3.5), 500, 12)
    assert abs(C[0, 0] - np.log(3.5)) < 1e-13 and np.abs(C[0, 1:]).max() < 1e-13
    C0 = oracle.kdist_cheb(np.zeros(500), 500, 4)                                   # kappa = 0: ln of the floor (reading C1)
    assert abs(C0[0, 0] - np.log(1e-300)) < 1e-10 and np.abs(C0[0, 1:]).max() < 1e-10


def test_eval_reproduces_smooth_kappa_of_y():
    # resampling error << 1 % for N_nu >= 1e3: a smooth ln kappa(y) spanning 6 decades
    ppb = 1000
    y = (np.arange(ppb) + 0.5) / ppb
    kappa = 10 ** (-3 + 6 * y ** 3)
    C = oracle.kdist_cheb(kappa, ppb, 20)
    assert np.abs(oracle.cheb_eval(C, y)[0] / kappa - 1.0).max() < 1e-9
    assert oracle.cheb_eval(C, y).shape == (1, ppb)


# ---- f2: transmission function -----------------------------------------------------------------------------------------
def test_transmission_closed_forms():
    m = 10 ** np.linspace(-4, 2, 31)
    # constant opacity: T = exp(-kappa m) by both routes
    kap = np.full(1000, 0.37)
    kt = oracle.kdist(kap, 1000, 20)
    assert np.abs(oracle.transmission_kdist(kt, m)[0] / np.exp(-0.37 * m) - 1.0).max() < 1e-13
    assert np.abs(oracle.transmission_direct(kap, 1000, m)[0] / np.exp(-0.37 * m) - 1.0).max() < 1e-13
    # m = 0: T = 1
    assert np.array_equal(oracle.transmission_direct(10 ** np.linspace(-3, 3, 1000), 1000, [0.0])[0], [1.0])
    assert abs(oracle.transmission_kdist(kt, [0.0])[0, 0] - 1.0) < 1e-15
    # kappa uniformly distributed on [a, b]: T = (exp(-a m) - exp(-b m)) / ((b - a) m)
    a, b, ppb = 0.5, 2.5, 4000
    kap = a + (b - a) * (np.arange(ppb) + 0.5) / ppb
    mm = np.array([0.01, 0.3, 1.0, 3.0])
    exact = (np.exp(-a * mm) - np.exp(-b * mm)) / ((b - a) * mm)
    rng = np.random.default_rng(5)
    shuffled = kap[rng.permutation(ppb)]
    assert np.abs(oracle.transmission_direct(shuffled, ppb, mm)[0] / exact - 1.0).max() < 1e-7     # midpoint rule, O(1/ppb^2)
    kt = oracle.kdist(shuffled, ppb, 20)
    assert np.abs(oracle.transmission_kdist(kt, mm)[0] / exact - 1.0).max() < 1e-12              # Gauss-Legendre: exact for smooth


def test_transmission_invariants_and_lebesgue_equals_riemann():
    rng = np.random.default_rng(11)
    ppb = 1000
    y = (np.arange(ppb) + 0.5) / ppb
    kap = np.concatenate([10 ** (-2 + 3 * y ** 2), 10 ** (1 - 2 * y)])[np.r_[rng.permutation(ppb), ppb + rng.permutation(ppb)]]
    m = 10 ** np.linspace(-3, 3, 25)
    Td = oracle.transmission_direct(kap, ppb, m)
    Tk = oracle.transmission_kdist(oracle.kdist(kap, ppb, 20), m)
    assert Td.shape == Tk.shape == (2, 25)
    assert np.all(np.diff(Td, axis=1) < 0) and np.all((Td > 0) & (Td <= 1))
    assert np.abs(Tk - Td).max() < 1e-5                                            # eq. 5: int F dx = int F dy
    # numpy brute force of the definition
    ref = np.array([[np.mean(np.exp(-kap[b * ppb:(b + 1) * ppb] * mm)) for mm in m] for b in range(2)])
    assert np.abs(Td / ref - 1.0).max() < 1e-13


# ---- f3: full line physics (eqs. 20-21) and species mixing -------------------------
def _draw(n=60, seed=4):
    rng = np.random.default_rng(seed)
    nu0 = np.sort(rng.uniform(5.0, 95.0, n))
    return (nu0, 10 ** rng.uniform(-22, -19, n), rng.uniform(0.02, 0.1, n), rng.uniform(0.1, 0.5, n),
            10 ** rng.uniform(-2, 2, n), rng.uniform(-0.02, 0.02, n), rng.uniform(0.3, 0.8, n))


GRID = (0.0, 100.0, 0.01, 25.0)


def test_full_physics_reduces_to_the_simple_law():
    nu0, S, ga, gs, A, dl, nT = _draw()
    base = oracle.opacity(nu0, S, ga, 900.0, 2.0, *GRID, n_T=nT)
    assert np.array_equal(oracle.opacity_full(nu0, S, ga, 900.0, 2.0, *GRID, n_T=nT), base)
    # gamma_self == gamma_air: the self fraction drops out of eq. 20
    for f in (0.0, 0.5, 1.0):
        k = oracle.opacity_full(nu0, S, ga, 900.0, 2.0, *GRID, n_T=nT, gamma_self=ga, self_fraction=f)
        assert np.abs(k / base - 1.0).max() < 1e-13
    # self_fraction = 0: air only; = 1: the simple law with gamma_self in place of gamma_air
    k0 = oracle.opacity_full(nu0, S, ga, 900.0, 2.0, *GRID, n_T=nT, gamma_self=gs, self_fraction=0.0)
    assert np.abs(k0 / base - 1.0).max() < 1e-13
    k1 = oracle.opacity_full(nu0, S, ga, 900.0, 2.0, *GRID, n_T=nT, gamma_self=gs, self_fraction=1.0)
    assert np.abs(k1 / oracle.opacity(nu0, S, gs, 900.0, 2.0, *GRID, n_T=nT) - 1.0).max() < 1e-13
    # equal proportions: the pressure term is the mean of the two coefficients
    kh = oracle.opacity_full(nu0, S, ga, 900.0, 2.0, *GRID, n_T=nT, gamma_self=gs, self_fraction=0.5)
    assert np.abs(kh / oracle.opacity(nu0, S, 0.5 * (ga + gs), 900.0, 2.0, *GRID, n_T=nT) - 1.0).max() < 1e-12


def test_natural_width_adds_to_the_lorentz_width():
    # a line at nu0 -> 0 is a pure Lorentzian (alpha = 0): peak = amp/(pi gamma), so gamma is read off the peak
    c, amu = 2.99792458e10, 1.66053906660e-24
    S, ga, A, T, P = 1e-20, 0.05, 3.0e9, 296.0, 1e-3
    k = oracle.opacity_full([0.0], [S], [ga], T, P, 0.0, 10.0, 0.01, 25.0, A21=[A])
    gamma = ga * P + A / (4 * np.pi * c)
    assert abs(k[0] / (S / (18.0 * amu) / (np.pi * gamma)) - 1.0) < 1e-13
    assert A / (4 * np.pi * c) > 0.1 * ga * P                                    # the natural width matters in this case
    j = 137
    lor = S / (18.0 * amu) * gamma / (np.pi * ((j * 0.01) ** 2 + gamma ** 2))
    assert abs(k[j] / lor - 1.0) < 1e-13


def test_pressure_shift_is_a_translation_of_the_centre():
    nu0, S, ga, gs, A, dl, nT = _draw()
    P = 7.0
    k = oracle.opacity_full(nu0, S, ga, 1200.0, P, *GRID, delta=dl)
    ref = oracle.opacity(nu0 + dl * P, S, ga, 1200.0, P, *GRID)                  # the shifted list is no longer ordered
    assert np.any(np.diff(nu0 + dl * P) < 0)
    assert np.abs(k / ref - 1.0).max() < 1e-13
    one = oracle.opacity_full([50.0], [1e-20], [0.05], 300.0, 10.0, *GRID, delta=[-0.031])
    assert np.argmax(one) == 5000 - 31


def test_abundance_weight_and_mixing_is_linear():
    nu0, S, ga, gs, A, dl, nT = _draw()
    kw = dict(gamma_self=gs, A21=A, delta=dl, n_T=nT)
    k1 = oracle.opacity_full(nu0, S, ga, 800.0, 0.5, *GRID, **kw)
    kx = oracle.opacity_full(nu0, S, ga, 800.0, 0.5, *GRID, abundance=0.25, **kw)
    assert np.abs(kx / (0.25 * k1) - 1.0).max() < 1e-14
    js = np.array([0, 17, 5000, 9999])
    assert np.array_equal(oracle.opacity_full(nu0, S, ga, 800.0, 0.5, *GRID, js=js, **kw), k1[js])


# ---- f4: relative line-wing cutoff --------------------------------------------------------------------
def test_relative_cutoff_support_and_reductions():
    nu0, S, ga, gs, A, dl, nT = _draw(n=40, seed=9)
    T, P, W = 296.0, 1.0, 40.0                     # gamma_i = ga_i at 296 K, 1 atm (simple law): W gamma = 0.8 .. 4 cm^-1
    k_abs = oracle.opacity(nu0, S, ga, T, P, *GRID)
    # a relative cutoff wider than the absolute one never binds
    assert np.array_equal(oracle.opacity_full(nu0, S, ga, T, P, *GRID, cutoff_widths=1e6), k_abs)
    assert np.array_equal(oracle.opacity_full(nu0, S, ga, T, P, *GRID, cutoff_widths=0.0), k_abs)
    # single lines: the support is |nu_j - nu0| <= W gamma exactly (brute force on the grid), the values inside are untouched
    nu = np.arange(10000) * 0.01
    for i in (0, 7, 23):
        k = oracle.opacity_full(nu0[i:i + 1], S[i:i + 1], ga[i:i + 1], T, P, 0.0, 100.0, 0.01, 1e4, cutoff_widths=W)
        full = oracle.opacity(nu0[i:i + 1], S[i:i + 1], ga[i:i + 1], T, P, 0.0, 100.0, 0.01, 1e4)
        lo = np.ceil(((nu0[i] - W * ga[i]) - 0.0) / 0.01)
        hi = np.floor(((nu0[i] + W * ga[i]) - 0.0) / 0.01)
        inside = (np.arange(10000) >= lo) & (np.arange(10000) <= hi)
        assert np.array_equal(k != 0.0, inside) and np.array_equal(k[inside], full[inside])
        assert abs(inside.sum() - 2 * W * ga[i] / 0.01) <= 2
    # the sum over lines of the single-line results is the multi-line result (each line keeps its own cutoff)
    parts = sum(oracle.opacity_full(nu0[i:i + 1], S[i:i + 1], ga[i:i + 1], T, P, *GRID, cutoff_widths=W) for i in range(40))
    allk = oracle.opacity_full(nu0, S, ga, T, P, *GRID, cutoff_widths=W)
    assert np.abs(allk - parts).max() <= 1e-12 * allk.max()
    # the absolute cutoff stays an upper bound: min(cutoff, W gamma)
    assert W * ga[0] > 0.5
    capped = oracle.opacity_full(nu0[:1], S[:1], ga[:1], T, P, 0.0, 100.0, 0.01, 0.5, cutoff_widths=W)
    assert np.array_equal(capped, oracle.opacity(nu0[:1], S[:1], ga[:1], T, P, 0.0, 100.0, 0.01, 0.5))
