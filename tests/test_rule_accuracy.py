"""Accuracy claim behind the device ladder's far-wing rule (hk_voigt.cuh kR1a/kR1b): the 1-point rule with
the shifted denominator, K ~ (y/sqrt(pi))/(x^2 + y^2 - 3/2), is within 1.5/x^4 + 2 y^2/r^4 of K(x,y), hence within 2.4e-7
from r^2 = max(3600, 4100 y) on (FP64 ladder) and within 2.2e-5 from max(400, 400 y) (FP32 variant).  Checked against the
oracle's Faddeeva routine (itself pinned to mpmath); the formula is restated here in numpy, not imported from the CUDA path."""
import numpy as np

import oracle


def _k1s(x, y):
    return (y / np.sqrt(np.pi)) / (x * x + y * y - 1.5)


def test_error_law_of_the_shifted_one_point_rule():
    y = 10 ** np.linspace(-8, 2.5, 200)
    for r2 in (400.0, 1000.0, 3200.0, 3600.0, 1e4, 1e5, 1e6, 6e6):
        ok = y * y < 0.5 * r2
        x = np.sqrt(r2 - y[ok] ** 2)
        rel = np.abs(_k1s(x, y[ok]) / oracle.faddeeva_re(x, y[ok]) - 1.0)
        law = 1.5 / x ** 4 + 2.0 * y[ok] ** 2 / r2 ** 2
        assert np.all(rel <= 1.15 * law + 5e-13), (r2, (rel / law).max())
        assert rel.max() >= 0.3 * law.min()                       # the law is sharp, not a loose bound


def test_budget_on_the_switch_curves():
    y = 10 ** np.linspace(-8, 3, 300)
    for a, b, budget in ((3600.0, 4100.0, 2.4e-7), (400.0, 400.0, 2.2e-5)):
        for s in (1.0, 1.5, 10.0, 1e3):
            r2 = np.maximum(a, b * y) * s
            ok = r2 > 2 * y * y
            x = np.sqrt(r2[ok] - y[ok] ** 2)
            rel = np.abs(_k1s(x, y[ok]) / oracle.faddeeva_re(x, y[ok]) - 1.0)
            assert rel.max() <= budget, (a, b, s, rel.max())
    # the plain 1-point rule needs r^2 >= 6e6 for the same budget (what the shifted denominator buys)
    x = np.sqrt(3600.0)
    plain = (1e-3 / np.sqrt(np.pi)) / (x * x + 1e-6)
    assert abs(plain / oracle.faddeeva_re(x, 1e-3) - 1.0) > 1e-4
