"""Pins for the oracle's K(x,y) = Re w(x+iy) (H_V of eq. 19).

None of these call the oracle's own formulas: the expected values are mpmath 50-digit evaluations of the
definition (tests/golden/, written by make_faddeeva_golden.py), brute-force quadrature of the convolution
integral, closed forms, symmetry and asymptotes.
"""
import math
import os

import numpy as np
import pytest

import oracle


def _load(golden_dir, name, cols):
    return np.genfromtxt(os.path.join(golden_dir, name), delimiter=",", comments="#", usecols=cols)


def test_golden_lattice_rings_core(golden_dir):
    d = _load(golden_dir, "faddeeva_golden.csv", (1, 2, 3))
    assert d.shape[0] > 2000
    k = oracle.faddeeva_re(d[:, 0], d[:, 1])
    rel = np.abs(k / d[:, 2] - 1.0)
    assert rel.max() < 1e-13, (rel.max(), d[np.argmax(rel)])


def test_bruteforce_convolution_integral(golden_dir):
    q = _load(golden_dir, "voigt_quad_golden.csv", (0, 1, 2))
    assert q.shape[0] == 100
    k = oracle.faddeeva_re(q[:, 0], q[:, 1])
    assert np.abs(k / q[:, 2] - 1.0).max() < 1e-13


def test_live_mpmath_random_points():
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    rng = np.random.default_rng(7)
    x = np.concatenate([rng.uniform(0, 20, 150), 10 ** rng.uniform(1, 6, 50)])
    y = 10 ** rng.uniform(-10, 3, 200)
    k = oracle.faddeeva_re(x, y)
    for xi, yi, ki in zip(x, y, k):
        z = mp.mpc(xi, yi)
        e = float(mp.re(mp.exp(-z * z) * mp.erfc(-1j * z)))
        assert abs(ki / e - 1.0) < 1e-13, (xi, yi, ki, e)


def test_closed_form_on_imaginary_axis():
    # K(0,y) = exp(y^2) erfc(y);  K(0,1) = e*erfc(1)
    from scipy.special import erfcx
    y = 10 ** np.linspace(-8, 4, 200)
    k = oracle.faddeeva_re(np.zeros_like(y), y)
    assert np.abs(k / erfcx(y) - 1.0).max() < 1e-13
    assert abs(oracle.faddeeva_re(0.0, 1.0)[0] - math.e * math.erfc(1.0)) < 1e-15
    assert abs(oracle.faddeeva_re(0.0, 1.0)[0] - 0.42758357615580700441) < 1e-15


def test_real_axis_limit_is_gaussian():
    # K(x, y->0) = exp(-x^2); at y = 1e-14 the Lorentz wing term y/(sqrt(pi) x^2) is < 1e-14
    x = np.linspace(0, 4, 81)
    y = 1e-14
    k = oracle.faddeeva_re(x, np.full_like(x, y))
    # departure from the Gaussian is the Lorentz term, bounded by 2y/sqrt(pi) * max(1, 1/x^2)
    bound = 2 * y / math.sqrt(math.pi) * np.maximum(1.0, 1.0 / np.maximum(x, 1e-9) ** 2) + 1e-15 * np.exp(-x * x)
    assert np.all(np.abs(k - np.exp(-x * x)) <= bound)
    assert oracle.faddeeva_re(0.0, 1e-300)[0] == pytest.approx(1.0, abs=1e-15)


def test_symmetry_in_x():
    rng = np.random.default_rng(3)
    x = rng.uniform(0, 30, 500)
    y = 10 ** rng.uniform(-6, 2, 500)
    assert np.array_equal(oracle.faddeeva_re(x, y), oracle.faddeeva_re(-x, y))


def test_lorentz_asymptote():
    # K -> y/(sqrt(pi)(x^2+y^2)) with relative correction O(1.5/|z|^2)
    rng = np.random.default_rng(4)
    r = 10 ** rng.uniform(4, 7, 300)
    th = rng.uniform(1e-6, np.pi / 2, 300)
    x, y = r * np.cos(th), r * np.sin(th)
    k = oracle.faddeeva_re(x, y)
    lor = y / (math.sqrt(math.pi) * (x * x + y * y))
    assert np.all(np.abs(k / lor - 1.0) < 2.0 / (r * r))


def test_third_opinion_scipy_wofz():
    from scipy.special import wofz
    rng = np.random.default_rng(5)
    x = 10 ** rng.uniform(-3, 7, 20000)
    y = 10 ** rng.uniform(-8, 4, 20000)
    k = oracle.faddeeva_re(x, y)
    assert np.abs(k / wofz(x + 1j * y).real - 1.0).max() < 5e-13


def test_gauss_legendre_nodes():
    for n in (1, 2, 5, 20, 64):
        g, w = oracle.gauss_legendre(n)
        t, wt = np.polynomial.legendre.leggauss(n)
        assert np.abs(g - 0.5 * (1 + t)).max() < 1e-15
        assert np.abs(w - 0.5 * wt).max() < 1e-14   # numpy leggauss itself is ~1e-13 relative at n=64
        assert abs(w.sum() - 1.0) < 1e-15
    # exact for polynomials up to degree 2n-1 on (0,1)
    g, w = oracle.gauss_legendre(20)
    for p in range(0, 40):
        assert abs(np.sum(w * g ** p) - 1.0 / (p + 1)) < 1e-14
