"""Pins for the oracle's k-distribution (eqs. 14-15; eqs. 1-2)."""
import numpy as np
import pytest

import oracle


def _np_ref(kappa, ppb, n_g):
    t, _ = np.polynomial.legendre.leggauss(n_g)
    g = 0.5 * (1.0 + t)
    yk = (np.arange(ppb) + 0.5) / ppb
    out = []
    for b in range(kappa.size // ppb):
        s = np.sort(kappa[b * ppb:(b + 1) * ppb])
        out.append(np.interp(g, yk, s))                       # library sort + library interp (clamps at the ends)
    return np.array(out)


@pytest.mark.parametrize("ppb,n_g", [(1000, 20), (10000, 20), (37, 5), (2, 3), (1, 4), (64, 64)])
def test_against_numpy_sort_interp(ppb, n_g):
    rng = np.random.default_rng(ppb + n_g)
    kappa = 10 ** rng.uniform(-6, 5, 7 * ppb)
    k = oracle.kdist(kappa, ppb, n_g)
    ref = _np_ref(kappa, ppb, n_g)
    assert np.abs(k / ref - 1.0).max() < 1e-13


def test_permutation_invariance_and_monotone():
    rng = np.random.default_rng(2)
    kappa = 10 ** rng.uniform(-3, 3, 5000)
    k = oracle.kdist(kappa, 1000, 20)
    kp = kappa.reshape(5, 1000).copy()
    for row in kp:
        rng.shuffle(row)
    assert np.array_equal(oracle.kdist(kp.ravel(), 1000, 20), k)
    assert np.all(np.diff(k, axis=1) >= 0.0)


def test_constant_and_linear_bins_are_exact():
    n_g, ppb = 20, 1000
    g, _ = oracle.gauss_legendre(n_g)
    const = np.full(ppb, 3.25)
    assert np.array_equal(oracle.kdist(const, ppb, n_g), np.full((1, n_g), 3.25))
    # kappa linear in x over the bin: kappa_k = a + b (k+1/2)/ppb  =>  kappa(y) = a + b y exactly at every node
    a, b = 2.0, 5.0
    lin = a + b * (np.arange(ppb) + 0.5) / ppb
    k = oracle.kdist(lin[::-1].copy(), ppb, n_g)
    assert np.abs(k[0] - (a + b * g)).max() < 1e-12
    # zeros stay zeros (no logarithm involved)
    assert not oracle.kdist(np.zeros(ppb), ppb, n_g).any()


def test_lebesgue_equals_riemann():
    # eqs. 1-2: int kappa dx = int kappa dy.  With Gauss-Legendre weights sum_q w_q k_q ~ mean(kappa) (quadrature error only)
    rng = np.random.default_rng(3)
    ppb = 1000
    x = (np.arange(ppb) + 0.5) / ppb
    kappa = np.exp(2.0 * np.sin(7 * x) + x)                   # smooth, spans ~1.5 decades
    kappa = kappa[rng.permutation(ppb)]
    _, w = oracle.gauss_legendre(20)
    k = oracle.kdist(kappa, ppb, 20)
    assert abs(np.sum(w * k[0]) / kappa.mean() - 1.0) < 2e-3   # kappa(y) has kinks at local extrema of kappa(x)
    # transmission (eq. 5): mean_x exp(-kappa m) = int exp(-kappa(y) m) dy
    for m in (0.01, 0.3, 2.0):
        assert abs(np.sum(w * np.exp(-k[0] * m)) / np.exp(-kappa * m).mean() - 1.0) < 2e-3


def test_clamping_at_the_ends():
    # n_g large enough that the outer nodes fall below y_0 = 1/(2 ppb) and above y_last
    ppb, n_g = 4, 64
    kappa = np.array([4.0, 1.0, 3.0, 2.0])
    k = oracle.kdist(kappa, ppb, n_g)[0]
    g, _ = oracle.gauss_legendre(n_g)
    assert np.all(k[g <= 0.125] == 1.0) and np.all(k[g >= 0.875] == 4.0)
    assert (g <= 0.125).any() and (g >= 0.875).any()


def test_rejects_ragged_bins():
    with pytest.raises(ValueError):
        oracle.kdist(np.ones(1001), 1000, 20)
