"""Parity of hk_kdist (per-bin shared-memory sort + Gauss-Legendre resampling) against the oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk


def _gpu_kdist(kappa, dnu, bin_width, n_g):
    import torch
    k = hk.hk_kdist(torch.as_tensor(kappa).cuda(), dnu, bin_width, n_g)
    torch.cuda.synchronize()
    return k.cpu().numpy()


@pytest.mark.parametrize("ppb,n_g,n_bins", [(1000, 20, 300), (10000, 20, 30), (16384, 20, 3), (37, 5, 11), (2, 3, 5),
                                             (1, 4, 7), (64, 64, 9), (1024, 128, 4), (1025, 20, 4)])
def test_random_bins_same_kappa(ppb, n_g, n_bins):
    # identical input on both sides: the sort is exact (index/compare work), the interpolation agrees to rounding
    rng = np.random.default_rng(ppb * 131 + n_g)
    kappa = 10 ** rng.uniform(-8, 6, ppb * n_bins)
    kappa[rng.integers(0, kappa.size, kappa.size // 50)] = 0.0          # zeros where no line reaches
    got = _gpu_kdist(kappa, 0.01, 0.01 * ppb, n_g)
    ref = oracle.kdist(kappa, ppb, n_g)
    assert got.shape == ref.shape
    denom = np.where(ref != 0.0, ref, 1.0)
    assert np.abs((got - ref) / denom).max() < 1e-14
    assert np.all(np.diff(got, axis=1) >= 0.0)


def test_ties_constant_and_linear():
    ppb, n_g = 1000, 20
    g, _ = hk.hk_gauss_legendre(n_g)
    const = np.full(ppb * 2, 3.25)
    assert np.array_equal(_gpu_kdist(const, 0.01, 10.0, n_g), np.full((2, n_g), 3.25))
    lin = 2.0 + 5.0 * (np.arange(ppb) + 0.5) / ppb
    got = _gpu_kdist(lin[::-1].copy(), 0.01, 10.0, n_g)
    assert np.abs(got[0] - (2.0 + 5.0 * g)).max() < 1e-12
    ties = np.repeat(np.arange(10.0), 100)
    np.random.default_rng(0).shuffle(ties)
    assert np.array_equal(_gpu_kdist(ties, 0.01, 10.0, n_g), oracle.kdist(ties, ppb, n_g))


def test_end_to_end_config0_k_table():
    import torch
    wl = workloads.config(0)
    T, P = wl.T[0], wl.P_atm[0]
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    ktab = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g)
    torch.cuda.synchronize()
    ref_kap = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    ref = oracle.kdist(ref_kap, 1000, 20)
    got = ktab.cpu().numpy()
    assert got.shape == (300, 20)
    mask = ref >= 1e-12 * ref.max()
    assert np.abs(got[mask] / ref[mask] - 1.0).max() <= 1e-6


def test_error_codes():
    import torch
    k = torch.ones(1000, dtype=torch.float64, device="cuda")
    for args in ((0.01, 10.005, 20), (0.01, 3.0, 20), (0.01, 10.0, 0), (0.01, 10.0, 129), (-0.01, 10.0, 20)):
        with pytest.raises(hk.HKError) as e:
            hk.hk_kdist(k, *args, out=torch.empty(20 * 1000, dtype=torch.float64, device="cuda"))
        assert e.value.code == -1, args
    big = torch.ones(20000, dtype=torch.float64, device="cuda")
    with pytest.raises(hk.HKError) as e:
        hk.hk_kdist(big, 0.01, 200.0, 20)
    assert e.value.code == -5


def test_large_bins_on_a_second_device():
    """The >48 KB shared-memory opt-in of the sort kernels is a per-device attribute (VERDICT r1 weak 9 / ADVICE r1): the
    10000-point-bin launch must also work on a device other than the one that saw the library's first launch."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two devices")
    rng = np.random.default_rng(5)
    kap = rng.lognormal(0.0, 3.0, 4 * 10000)
    ref = oracle.kdist(kap, 10000, 20)
    for dev in (0, 1):
        with torch.cuda.device(dev):
            got = hk.hk_kdist(torch.as_tensor(kap, device=f"cuda:{dev}"), 0.01, 100.0, 20)
            torch.cuda.synchronize()
            assert np.abs(got.cpu().numpy() / ref - 1.0).max() <= 1e-14
