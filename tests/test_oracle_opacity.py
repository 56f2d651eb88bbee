"""Pins for the oracle's line parameters, window, Voigt profile and kappa (eqs. 16-20).

Expected values come from closed forms / limits / invariants and from a numpy + scipy.special.wofz brute force
(a library Faddeeva, not the oracle's), with the cutoff window decided independently.
"""
import math

import numpy as np
import pytest

import oracle
import workloads

C_LIGHT = 2.99792458e10
K_B = 1.380649e-16
AMU = 1.66053906660e-24


def _alpha(nu0, T, m=18.0):
    return nu0 / C_LIGHT * np.sqrt(2 * K_B * T / (m * AMU))


def test_bruteforce_numpy_wofz_small_opacity():
    from scipy.special import wofz
    wl = workloads.small(seed=11, n_lines=120, nu_max=300.0, cutoff=25.0)
    T, P = wl.T[0], wl.P_atm[0]
    kap = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    N = wl.n_points
    assert kap.shape == (N,)
    nu = wl.nu_min + np.arange(N) * wl.dnu
    alpha = _alpha(wl.nu0, T)
    gamma = wl.gamma0 * P * math.sqrt(296.0 / T)
    ref = np.zeros(N)
    for i in range(wl.n_lines):
        dv = nu - wl.nu0[i]
        inside = np.abs(dv) <= wl.cutoff                    # window decided in value space here
        V = wofz((dv + 1j * gamma[i]) / alpha[i]).real / (alpha[i] * math.sqrt(math.pi))
        ref += np.where(inside, wl.S[i] / (18.0 * AMU) * V, 0.0)
    assert np.abs(kap / ref - 1.0).max() < 1e-12
    assert kap.min() > 0.0


def test_config0_spot_check_against_wofz():
    # full config 0 in the oracle, 400 seeded grid points re-done with wofz
    from scipy.special import wofz
    wl = workloads.config(0)
    T, P = wl.T[0], wl.P_atm[0]
    rng = np.random.default_rng(0)
    js = np.sort(rng.choice(wl.n_points, 400, replace=False))
    alpha = _alpha(wl.nu0, T)
    gamma = wl.gamma0 * P * math.sqrt(296.0 / T)
    for j in js[:40]:
        k1 = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, j_begin=int(j), j_end=int(j) + 1)[0]
        nu = wl.nu_min + j * wl.dnu
        dv = nu - wl.nu0
        m = np.abs(dv) <= wl.cutoff
        ref = np.sum(wl.S[m] / (18.0 * AMU) * wofz((dv[m] + 1j * gamma[m]) / alpha[m]).real / (alpha[m] * math.sqrt(math.pi)))
        assert abs(k1 / ref - 1.0) < 1e-12


def test_gaussian_limit():
    # gamma -> 0: V -> exp(-(dv/alpha)^2)/(alpha sqrt(pi))   (Doppler profile)
    alpha, gamma = 0.05, 0.05 * 1e-12
    for dv in np.linspace(-0.15, 0.15, 31):
        v = oracle.voigt_V(dv, alpha, gamma)
        g = math.exp(-(dv / alpha) ** 2) / (alpha * math.sqrt(math.pi))
        assert abs(v / g - 1.0) < 1e-8


def test_lorentzian_limit():
    # alpha -> 0: V -> gamma/(pi (dv^2 + gamma^2)); also exactly alpha == 0 (a line at nu0 = 0)
    gamma = 0.03
    for alpha in (1e-9, 1e-14, 0.0):
        for dv in (0.0, 1e-3, 0.02, 0.5, 7.0, 90.0):
            v = oracle.voigt_V(dv, alpha, gamma)
            l = gamma / (math.pi * (dv * dv + gamma * gamma))
            assert abs(v / l - 1.0) < 1e-9


def test_unit_area():
    # dnu * sum V over [-W, W] = 1 - Lorentz tails; tails = (2/pi) atan-like ~ 2 gamma/(pi W) for W >> alpha, gamma
    alpha, gamma, W, h = 0.06, 0.03, 200.0, 0.002
    dv = np.arange(-W, W + h / 2, h)
    v = np.array([oracle.voigt_V(d, alpha, gamma) for d in dv[:: 1]])
    area = h * (v.sum() - 0.5 * (v[0] + v[-1]))
    tail = 1.0 - (2.0 / math.pi) * math.atan(W / gamma)      # exact tail of the Lorentzian; Voigt differs by O(alpha^2/W^2)
    assert abs(area - (1.0 - tail)) < 1e-7


def test_single_line_is_amplitude_times_profile():
    nu0, S, g0, T, P = 1234.5678, 3e-21, 0.07, 1500.0, 1.0
    kap = oracle.opacity([nu0], [S], [g0], T, P, 1200.0, 1270.0, 0.01, 25.0)
    a = float(_alpha(nu0, T))
    gam = g0 * P * math.sqrt(296.0 / T)
    for j in (0, 1000, 3456, 3457, 5000, 6999):
        nu = 1200.0 + j * 0.01
        expect = S / (18.0 * AMU) * oracle.voigt_V(nu - nu0, a, gam) if abs(nu - nu0) <= 25.0 else 0.0
        assert kap[j] == pytest.approx(expect, rel=1e-15, abs=0.0)
    assert kap[0] == 0.0 and kap[-1] == 0.0                  # outside the +-25 cm^-1 window
    # symmetric about nu0 to the extent the grid allows: peak at the nearest node
    assert abs(np.argmax(kap) - round((nu0 - 1200.0) / 0.01)) <= 1


def test_linearity_additivity_and_order_independence():
    wl = workloads.small(seed=5, n_lines=60, nu_max=100.0, cutoff=25.0)
    args = (wl.T[0], wl.P_atm[0], wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    k = oracle.opacity(wl.nu0, wl.S, wl.gamma0, *args)
    k2 = oracle.opacity(wl.nu0, 2.0 * wl.S, wl.gamma0, *args)
    assert np.array_equal(k2, 2.0 * k)
    ka = oracle.opacity(wl.nu0[:25], wl.S[:25], wl.gamma0[:25], *args)
    kb = oracle.opacity(wl.nu0[25:], wl.S[25:], wl.gamma0[25:], *args)
    assert np.abs((ka + kb) / k - 1.0).max() < 1e-14
    perm = np.random.default_rng(1).permutation(wl.n_lines)
    kp = oracle.opacity(wl.nu0[perm], wl.S[perm], wl.gamma0[perm], *args)
    assert np.array_equal(kp, k)


def test_subrange_equals_full():
    wl = workloads.small(seed=6, n_lines=40, nu_max=60.0, cutoff=25.0)
    args = (wl.nu0, wl.S, wl.gamma0, wl.T[0], wl.P_atm[0], wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    k = oracle.opacity(*args)
    ks = oracle.opacity(*args, j_begin=1234, j_end=2345)
    assert np.array_equal(ks, k[1234:2345])


def test_window_is_inclusive_in_index_space():
    # a line exactly on a grid node, cutoff an exact multiple of dnu: 2*cutoff/dnu + 1 points, edges included
    nu0 = 50.0
    kap = oracle.opacity([nu0], [1e-20], [0.05], 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0)
    nz = np.nonzero(kap)[0]
    assert nz[0] == 2500 and nz[-1] == 7500 and nz.size == 5001
    assert oracle.count_evals([nu0], 0.0, 10000, 0.01, 25.0) == 5001
    # a line outside the grid but within the cutoff still contributes; beyond the cutoff it does not
    kap = oracle.opacity([-10.0], [1e-20], [0.05], 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0)
    assert np.nonzero(kap)[0][-1] == 1500 and kap[0] > 0.0
    kap = oracle.opacity([130.0], [1e-20], [0.05], 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0)
    assert not kap.any()
    assert oracle.count_evals([130.0], 0.0, 10000, 0.01, 25.0) == 0
    # no lines at all: kappa == 0
    assert not oracle.opacity([], [], [], 1000.0, 1.0, 0.0, 10.0, 0.01, 25.0).any()


def test_count_evals_bruteforce():
    wl = workloads.small(seed=8, n_lines=300, nu_max=50.0, cutoff=7.0)
    N = wl.n_points
    nu = wl.nu_min + np.arange(N) * wl.dnu
    brute = sum(int(np.count_nonzero(np.abs(nu - c) <= wl.cutoff)) for c in wl.nu0)
    assert oracle.count_evals(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff) == brute
    kap_mask = np.zeros(N, dtype=np.int64)
    for c in wl.nu0:
        kap_mask += np.abs(nu - c) <= wl.cutoff
    assert kap_mask.sum() == brute


def test_line_strength_scaling_special_cases():
    # eq. 18 (G1 reading): T = 296 -> 1; E'' = 0 -> no Boltzmann factor; nu0 -> 0 -> stimulated ratio -> 296/T
    assert oracle.line_strength(2.5e-22, 1500.0, 3000.0, 296.0, 1.0) == pytest.approx(2.5e-22, rel=1e-15)
    c2 = 1.4388
    T = 1200.0
    s = oracle.line_strength(1.0, 2000.0, 0.0, T, 0.5)
    assert s == pytest.approx(0.5 * (1 - math.exp(-c2 * 2000 / T)) / (1 - math.exp(-c2 * 2000 / 296.0)), rel=1e-14)
    assert oracle.line_strength(1.0, 1e-9, 0.0, T, 1.0) == pytest.approx(296.0 / T, rel=1e-9)
    assert oracle.line_strength(1.0, 0.0, 0.0, T, 1.0) == pytest.approx(296.0 / T, rel=1e-15)
    # hot band: raising T raises a high-E'' line (Boltzmann factor > 1 for T > 296)
    assert oracle.line_strength(1.0, 1000.0, 20000.0, 3000.0, 1.0) > 1e30
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    S, nu0, E, T, q = 3e-24, 4321.0, 8765.0, 777.0, (296.0 / 777.0) ** 1.5
    e = mp.mpf(S) * mp.mpf(q) * mp.exp(-mp.mpf(c2) * E * (mp.mpf(1) / T - mp.mpf(1) / 296)) * \
        (1 - mp.exp(-mp.mpf(c2) * nu0 / T)) / (1 - mp.exp(-mp.mpf(c2) * nu0 / 296))
    assert oracle.line_strength(S, nu0, E, T, q) == pytest.approx(float(e), rel=1e-13)


def test_opacity_with_E_low_uses_scaled_strength():
    wl = workloads.small(seed=9, n_lines=30, nu_max=40.0, cutoff=25.0, with_E=True, T=900.0)
    T, P = wl.T[0], wl.P_atm[0]
    q = wl.q_ratio(T)
    k = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, E_low=wl.E_low, q_ratio=q)
    ST = np.array([oracle.line_strength(s, n, e, T, q) for s, n, e in zip(wl.S, wl.nu0, wl.E_low)])
    k_ref = oracle.opacity(wl.nu0, ST, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    assert np.array_equal(k, k_ref)


def test_temperature_exponent_and_pressure_scaling():
    # gamma = gamma0 * P * (296/T)^n : in the far wing kappa is proportional to gamma
    nu0, S, g0 = 500.0, 1e-20, 0.05
    base = oracle.opacity([nu0], [S], [g0], 296.0, 1.0, 400.0, 600.0, 0.5, 100.0)
    dbl = oracle.opacity([nu0], [S], [g0], 296.0, 2.0, 400.0, 600.0, 0.5, 100.0)
    j = 20                                                    # 90 cm^-1 from the centre
    assert dbl[j] / base[j] == pytest.approx(2.0, rel=1e-5)
    n1 = oracle.opacity([nu0], [S], [g0], 1184.0, 1.0, 400.0, 600.0, 0.5, 100.0, n_T=[1.0])
    n05 = oracle.opacity([nu0], [S], [g0], 1184.0, 1.0, 400.0, 600.0, 0.5, 100.0)
    assert n05[j] / n1[j] == pytest.approx(2.0, rel=1e-4)    # (296/1184)^0.5 / (296/1184)^1 = 2


def test_rejects_bad_arguments():
    with pytest.raises(ValueError):
        oracle.opacity([1.0], [1.0], [0.05], -5.0, 1.0, 0.0, 10.0, 0.01, 25.0)
    with pytest.raises(ValueError):
        oracle.opacity([1.0], [1.0], [0.05], 300.0, 0.0, 0.0, 10.0, 0.01, 25.0)


def test_points_entry_equals_range_entry():
    wl = workloads.small(seed=12, n_lines=50, nu_max=80.0, cutoff=25.0)
    args = (wl.nu0, wl.S, wl.gamma0, wl.T[0], wl.P_atm[0], wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    k = oracle.opacity(*args)
    js = np.array([0, 17, 4000, 7999, 123, 123])
    assert np.array_equal(oracle.opacity_points(*args, js), k[js])
    with pytest.raises(ValueError):
        oracle.opacity_points(*args, [8000])


def test_pure_doppler_line_gamma_zero_closed_form():
    """gamma0 = 0: y = 0, K(x, 0) = exp(-x^2), so kappa = (S/m) exp(-((nu-nu0)/alpha)^2)/(alpha sqrt(pi)) exactly (PAPER.md:176-183
    with a = 0); pins the oracle where the device path has a special case (floor on y)."""
    nu0 = np.array([50.0]); S = np.array([1e-20]); g0 = np.array([0.0])
    T, P, dnu = 1500.0, 1.0, 1e-4
    k = oracle.opacity(nu0, S, g0, T, P, 0.0, 100.0, dnu, 25.0)
    alpha = 50.0 / 2.99792458e10 * np.sqrt(2 * 1.380649e-16 * T / (18.0 * 1.66053906660e-24))
    nu = np.arange(k.size) * dnu
    ref = 1e-20 / (18.0 * 1.66053906660e-24) * np.exp(-((nu - 50.0) / alpha) ** 2) / (alpha * np.sqrt(np.pi))
    m = ref > 1e-250
    assert np.isfinite(k).all()
    assert np.abs(k[m] / ref[m] - 1.0).max() < 1e-12
    assert k[~m].max() < 1e-240
