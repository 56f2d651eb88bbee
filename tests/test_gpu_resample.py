"""Parity of the SURVEY §8(f) rows built on the k-distribution — hk_kdist_cheb / hk_cheb_eval (Chebyshev least-squares
resampling of ln kappa(y)) and hk_transmission / hk_transmission_direct (eq. 5) —
against the oracle on the same seeded inputs.

Tolerances: on IDENTICAL kappa input both sides do the same FP64 arithmetic in a different order: 1e-10 (coefficients,
absolute, relative to max(1, |C|)), 1e-11 (transmission, relative).  End to end from the line list the inputs differ by the
Voigt routine's <= 2.5e-7, i.e. <= 2.5e-7 absolute in ln kappa: coefficients within 2e-6, resampled kappa(y) within 1e-6 x
the sum of |T_n| <= n_c (bar written below)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()


@pytest.mark.parametrize("ppb,n_c,n_bins", [(1000, 20, 7), (10000, 20, 3), (37, 5, 11), (64, 8, 2), (2048, 1, 2), (1, 1, 5)])
def test_cheb_coefficients_on_identical_kappa(ppb, n_c, n_bins):
    rng = np.random.default_rng(ppb + n_c)
    kappa = 10 ** rng.uniform(-8, 4, n_bins * ppb)
    coef = hk.hk_kdist_cheb(_dev(kappa), 0.01, 0.01 * ppb, n_c).cpu().numpy()
    ref = oracle.kdist_cheb(kappa, ppb, n_c)
    tol = 1e-10
    assert np.abs(coef - ref).max() < tol * max(1.0, np.abs(ref).max())


def test_cheb_with_ktable_from_the_same_launch_and_zero_floor():
    import torch
    rng = np.random.default_rng(3)
    kappa = 10 ** rng.uniform(-3, 3, 5000)
    kappa[:1000] = 0.0                                       # a bin of zeros: ln of the 1e-300 floor (reading C1)
    kappa[1000:1010] = 0.0
    d = _dev(kappa)
    coef, ktab = hk.hk_kdist_cheb(d, 0.01, 10.0, 20, n_g=20)
    assert torch.equal(ktab, hk.hk_kdist(d, 0.01, 10.0, 20))
    ref = oracle.kdist_cheb(kappa, 1000, 20)
    assert np.abs(coef.cpu().numpy() - ref).max() < 1e-9 * np.abs(ref).max()
    assert abs(coef[0, 0].item() - np.log(1e-300)) < 1e-9


def test_cheb_eval_matches_oracle_and_reconstructs():
    ppb = 1000
    y = (np.arange(ppb) + 0.5) / ppb
    kappa = np.concatenate([10 ** (-3 + 6 * y ** 3), 10 ** (2 - 4 * y)])
    coef = hk.hk_kdist_cheb(_dev(kappa), 0.01, 10.0, 20)
    yy = np.linspace(0.0, 1.0, 333)
    got = hk.hk_cheb_eval(coef, _dev(yy)).cpu().numpy()
    ref = oracle.cheb_eval(coef.cpu().numpy(), yy)
    assert got.shape == (2, 333) and np.abs(got / ref - 1.0).max() < 1e-12
    rec = hk.hk_cheb_eval(coef, _dev(y)).cpu().numpy()
    assert np.abs(rec[0] / kappa[:ppb] - 1.0).max() < 1e-9   # smooth ln kappa(y): the fit is the function
    assert np.abs(rec[1] / np.sort(kappa[ppb:]) - 1.0).max() < 1e-9


def test_transmission_on_identical_inputs():
    rng = np.random.default_rng(8)
    for ppb, n_bins, n_g, n_m in ((1000, 6, 20, 1000), (10000, 2, 20, 50), (37, 9, 5, 130), (4100, 2, 64, 7)):
        kappa = 10 ** rng.uniform(-4, 3, n_bins * ppb)
        m = np.concatenate(([0.0], 10 ** np.linspace(-5, 3, n_m - 1)))
        d = _dev(kappa)
        ktab = hk.hk_kdist(d, 0.01, 0.01 * ppb, n_g)
        Tk = hk.hk_transmission(ktab, _dev(m)).cpu().numpy()
        Td = hk.hk_transmission_direct(d, 0.01, 0.01 * ppb, _dev(m)).cpu().numpy()
        rk = oracle.transmission_kdist(ktab.cpu().numpy(), m)
        rd = oracle.transmission_direct(kappa, ppb, m)
        assert Tk.shape == Td.shape == (n_bins, n_m)
        for got, ref in ((Tk, rk), (Td, rd)):
            mask = ref > 1e-280
            assert np.abs(got[mask] / ref[mask] - 1.0).max() < 1e-11
            assert np.all(got[~mask] <= 1e-279)
        assert np.all(Td[:, 0] == 1.0) and np.abs(Tk[:, 0] - 1.0).max() < 1e-14


def test_config0_end_to_end_resampling_and_transmission():
    import torch
    wl = workloads.config(0)
    T, P = wl.T[0], wl.P_atm[0]
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    coef, ktab = hk.hk_kdist_cheb(kap, wl.dnu, wl.bin_width, 20, n_g=wl.n_g)
    m = 10 ** np.linspace(-4, 4, 200)
    Tk = hk.hk_transmission(ktab, _dev(m)).cpu().numpy()
    Td = hk.hk_transmission_direct(kap, wl.dnu, wl.bin_width, _dev(m)).cpu().numpy()
    torch.cuda.synchronize()
    ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    ppb = int(round(wl.bin_width / wl.dnu))
    cref = oracle.kdist_cheb(ref, ppb, 20)
    assert np.abs(coef.cpu().numpy() - cref).max() < 2e-6
    y = (np.arange(ppb) + 0.5) / ppb
    rec = hk.hk_cheb_eval(coef, _dev(y)).cpu().numpy()
    assert np.abs(rec / oracle.cheb_eval(cref, y) - 1.0).max() < 20 * 1e-6
    rk = oracle.transmission_kdist(oracle.kdist(ref, ppb, wl.n_g), m)
    rd = oracle.transmission_direct(ref, ppb, m)
    # d ln T = -m dk: a relative error e of kappa moves ln T by at most e |ln T|
    for got, r in ((Tk, rk), (Td, rd)):
        mask = r > 1e-200
        assert np.all(np.abs(got[mask] / r[mask] - 1.0) <= 1.2e-6 * np.maximum(1.0, -np.log(r[mask])))


def test_config1_full_size_1000_column_masses():
    # Fig. 5's "Resampling" and "Transmission" tasks at the size bench.py times: 3000 bins x 1000 points, 20 coefficients,
    # 1000 column masses; the oracle on seeded bins
    import torch
    wl = workloads.config(1)
    T, P = wl.T[0], wl.P_atm[0]
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    m = 10 ** np.linspace(-6, 4, 1000)
    dm = _dev(m)

    ktab = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g)
    coef, ktab2 = hk.hk_kdist_cheb(kap, wl.dnu, wl.bin_width, 20, n_g=wl.n_g)
    Tk = hk.hk_transmission(ktab, dm)
    Td = hk.hk_transmission_direct(kap, wl.dnu, wl.bin_width, dm)
    torch.cuda.synchronize()
    assert torch.equal(ktab, ktab2)
    kh = kap.cpu().numpy()
    rng = np.random.default_rng(6)
    bins = np.sort(rng.choice(3000, 40, replace=False))
    for b in bins:
        seg = kh[b * 1000:(b + 1) * 1000]
        cref = oracle.kdist_cheb(seg, 1000, 20)[0]
        assert np.abs(coef[b].cpu().numpy() - cref).max() < 1e-10 * max(1.0, np.abs(cref).max())
        rd = oracle.transmission_direct(seg, 1000, m)[0]
        rk = oracle.transmission_kdist(ktab[b:b + 1].cpu().numpy(), m)[0]
        for got, r in ((Td[b].cpu().numpy(), rd), (Tk[b].cpu().numpy(), rk)):
            mask = r > 1e-280
            assert np.abs(got[mask] / r[mask] - 1.0).max() < 1e-11


def test_error_codes():
    import torch
    k = torch.ones(1000, dtype=torch.float64, device="cuda")
    m = torch.ones(4, dtype=torch.float64, device="cuda")
    for bad in (lambda: hk.hk_kdist_cheb(k, 0.01, 10.0, 0), lambda: hk.hk_kdist_cheb(k, 0.01, 10.0, 65),
                lambda: hk.hk_kdist_cheb(k, 0.01, 0.1, 20),            # more coefficients than points per bin
                lambda: hk.hk_kdist_cheb(k, 0.01, 3.0, 5),             # 1000 is not a multiple of 300
                lambda: hk.hk_transmission_direct(k, 0.01, 3.0, m),
                lambda: hk.hk_transmission(torch.ones((2, 129), dtype=torch.float64, device="cuda"), m)):
        with pytest.raises(hk.HKError) as e:
            bad()
        assert e.value.code == -1
