"""Writes tests/golden/faddeeva_golden.csv and tests/golden/voigt_quad_golden.csv.

Uses ONLY mpmath (50 digits) — neither the oracle nor the CUDA path.  The values are what the
mathematics fixes:
  * faddeeva_golden.csv : K(x,y) = Re[exp(-z^2) erfc(-iz)], z = x+iy   (H_V of eq. 19 as the real part of the
    Faddeeva function), on a log lattice, on rings |z|^2 = R(1 +- 1e-9) around every
    regime switch used by either implementation, and at seeded random points of the core region;
  * voigt_quad_golden.csv : brute-force quadrature of the Voigt convolution integral itself,
    H_V = (a/pi) int exp(-u'^2)/((u-u')^2+a^2) du'   (eq. 19, sign as in DESIGN.md G2).

Run:  python tests/golden/make_faddeeva_golden.py
"""
import os
import random

import mpmath as mp

mp.mp.dps = 50
HERE = os.path.dirname(os.path.abspath(__file__))


def K_mp(x, y):
    z = mp.mpc(x, y)
    return mp.re(mp.exp(-z * z) * mp.erfc(-1j * z))


def K_quad(x, y):
    x, y = mp.mpf(x), mp.mpf(y)
    f = lambda t: mp.exp(-t * t) / ((x - t) ** 2 + y * y)
    pts = sorted({mp.mpf(-40), mp.mpf(-6), mp.mpf(0), x - 10 * y, x - y, x, x + y, x + 10 * y, mp.mpf(6), mp.mpf(40), x + 40})
    pts = [p for p in pts]
    return y / mp.pi * mp.quad(f, pts, maxdegree=10)


def fmt(v):
    return mp.nstr(v, 20, min_fixed=0, max_fixed=0)


def main():
    rnd = random.Random(1503_03806)
    rows = []
    xs = [0.0] + [10.0 ** (e / 2.0) for e in range(-6, 15)]          # 0, 1e-3 .. 1e7
    ys = [10.0 ** (e / 2.0) for e in range(-16, 9)]                   # 1e-8 .. 1e4
    for x in xs:
        for y in ys:
            rows.append(("lattice", x, y))
    rings = [25.0, 36.0, 40.0, 50.0, 64.0, 90.0, 100.0, 200.0, 280.0, 300.0, 1000.0, 3200.0, 1.0e4, 1.0e6, 6.0e6, 1.0e7]
    for R in rings:
        for s in (1.0 - 1e-9, 1.0 + 1e-9):
            r = (R * s) ** 0.5
            for th in [1e-9, 1e-6, 1e-3, 0.05, 0.2, 0.5, 0.9, 1.2, 1.5, mp.pi / 2 - 1e-4]:
                th = float(th)
                rows.append(("ring", float(r * mp.cos(th)), float(r * mp.sin(th))))
    for _ in range(1200):                                             # core region, y down to 1e-12
        r = (rnd.uniform(0.0, 320.0)) ** 0.5
        th = rnd.uniform(0.0, float(mp.pi) / 2) if rnd.random() < 0.5 else 10.0 ** rnd.uniform(-12.0, -0.3)
        rows.append(("core", float(r * mp.cos(th)), float(r * mp.sin(th))))
    for y in (0.25, 0.4999999, 0.5, 0.5000001, 1.0, 2.0):            # oracle's own switch at y = 0.5
        for x in (0.0, 0.3, 1.0, 2.5, 5.0, 7.9):
            rows.append(("switch_y", x, y))
    with open(os.path.join(HERE, "faddeeva_golden.csv"), "w") as f:
        f.write("# K(x,y)=Re w(x+iy), mpmath %d digits; PAPER.md:195 (H_V = real part of Faddeeva function)\n" % mp.mp.dps)
        f.write("# kind,x,y,K\n")
        for kind, x, y in rows:
            if y <= 0.0:
                continue
            f.write("%s,%s,%s,%s\n" % (kind, repr(float(x)), repr(float(y)), fmt(K_mp(x, y))))
    quad_rows = []
    for _ in range(100):
        x = rnd.choice([0.0, rnd.uniform(0, 3), rnd.uniform(0, 12), rnd.uniform(0, 40)])
        y = 10.0 ** rnd.uniform(-3.0, 1.5)
        quad_rows.append((x, y))
    with open(os.path.join(HERE, "voigt_quad_golden.csv"), "w") as f:
        f.write("# H_V(u,a) = (a/pi) int exp(-t^2)/((u-t)^2+a^2) dt by mpmath.quad, eq. 19 (PAPER.md:178)\n")
        f.write("# u,a,H_V\n")
        for x, y in quad_rows:
            f.write("%s,%s,%s\n" % (repr(float(x)), repr(float(y)), fmt(K_quad(x, y))))


if __name__ == "__main__":
    main()
