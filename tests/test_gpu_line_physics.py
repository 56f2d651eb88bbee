"""Parity of the SURVEY §8(f3) row — full line physics of eqs. 20-21 (natural width, air/self broadening, pressure shift;
PAPER.md:185-189) and species mixing before the sort — and of the "no cutoff" limit of §8(f4)
(every line on every grid point) against the oracle.  Bars as north_star: 1e-6 (FP64), 1e-4 (FP32)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk

BAR, BAR32 = 1.0e-6, 1.0e-4


def _fields(wl, seed):
    rng = np.random.default_rng(seed)
    n = wl.n_lines
    return dict(gamma_self=rng.uniform(0.1, 0.5, n), A21=10 ** rng.uniform(5, 9, n), delta=rng.uniform(-0.02, 0.02, n),
                n_T=rng.uniform(0.3, 0.8, n))


def _check(got, ref, bar):
    mask = ref >= 1e-12 * ref.max()
    assert np.all(np.isfinite(got))
    assert np.abs(got[mask] / ref[mask] - 1.0).max() <= bar
    assert np.all(got[ref == 0.0] == 0.0)


@pytest.mark.parametrize("T,P,f_self", [(1500.0, 1.0, 0.5), (700.0, 30.0, 0.2), (2000.0, 1e-4, 1.0)])
def test_eq20_eq21_against_the_oracle(T, P, f_self):
    import torch
    wl = workloads.small(seed=31, n_lines=1500, nu_max=200.0, cutoff=25.0, with_E=True)
    ex = _fields(wl, 32)
    q = wl.q_ratio(T)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low, **ex)
    ref = oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, E_low=wl.E_low,
                              q_ratio=q, self_fraction=f_self, **ex)
    for prec, bar in ((hk.HK_FP64, BAR), (hk.HK_FP32, BAR32)):
        got = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, self_fraction=f_self,
                            precision=prec)
        torch.cuda.synchronize()
        _check(got.cpu().numpy(), ref, bar)
    if P >= 30.0:
        assert np.any(np.diff(wl.nu0 + ex["delta"] * P) < 0)       # the shift really reorders this list
    # each optional term alone
    for key in ("gamma_self", "A21", "delta"):
        one = {key: ex[key]}
        l1 = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, **one)
        got = hk.hk_opacity(l1, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, self_fraction=f_self).cpu().numpy()
        _check(got, oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                        self_fraction=f_self, **one), BAR)


def test_mixture_is_summed_before_the_sort():
    import torch
    a = workloads.small(seed=41, n_lines=900, nu_max=150.0, cutoff=25.0)
    b = workloads.small(seed=42, n_lines=400, nu_max=150.0, cutoff=25.0)
    T, P, Xa, Xb, mb = 1100.0, 2.0, 0.7, 0.3, 44.0
    la, lb = hk.Lines.from_numpy(a.nu0, a.S, a.gamma0), hk.Lines.from_numpy(b.nu0, b.S, b.gamma0)
    kap = hk.hk_opacity(la, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, abundance=Xa)
    hk.hk_opacity(lb, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, mass_amu=mb, abundance=Xb, accumulate=True, out=kap)
    torch.cuda.synchronize()
    ra = oracle.opacity_full(a.nu0, a.S, a.gamma0, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, abundance=Xa)
    rb = oracle.opacity_full(b.nu0, b.S, b.gamma0, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, abundance=Xb, mass_amu=mb)
    _check(kap.cpu().numpy(), ra + rb, BAR)
    kt = hk.hk_kdist(kap, a.dnu, a.bin_width, a.n_g).cpu().numpy()
    kref = oracle.kdist(ra + rb, int(round(a.bin_width / a.dnu)), a.n_g)
    assert np.abs(kt / kref - 1.0).max() <= BAR
    # no lines + accumulate leaves the sum untouched; the host-buffer form reads the running sum from the host buffer
    empty = hk.Lines(*(torch.empty(0, dtype=torch.float64, device="cuda") for _ in range(3)))
    before = kap.clone()
    hk.hk_opacity(empty, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, accumulate=True, out=kap)
    assert torch.equal(kap, before)
    hk_a, _ = hk.hk_opacity_host(a.nu0, a.S, a.gamma0, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, abundance=Xa)
    hk_ab, _ = hk.hk_opacity_host(b.nu0, b.S, b.gamma0, T, P, a.nu_min, a.nu_max, a.dnu, a.cutoff, mass_amu=mb, abundance=Xb,
                                  accumulate=True, kappa_out=hk_a)
    assert torch.equal(hk_ab, kap.cpu())


def test_no_cutoff_every_line_on_every_point():
    # "full Voigt": a cutoff wider than the grid; N_evals = n_lines * N
    wl = workloads.small(seed=51, n_lines=300, nu_max=80.0, cutoff=25.0)
    T, P, big = 1500.0, 1.0, 1.0e6
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    assert hk.hk_count_evals(wl.nu0, wl.nu_min, wl.n_points, wl.dnu, big) == wl.n_lines * wl.n_points
    ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, big)
    _check(hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, big).cpu().numpy(), ref, BAR)
    _check(hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, big, precision=hk.HK_FP32).cpu().numpy(), ref, BAR32)


def test_large_pressure_shifts_on_a_dense_unsorted_list():
    # eq. 21 without re-ordering: a1 shifts the centres itself and builds its line-range tables from the unshifted ones with a
    # halo of max |delta| P.  Here the shifts (up to 1 cm^-1 = 100 grid steps, several 256-point spans apart at the tile
    # edges) are far larger than the line spacing (0.01 cm^-1) and the list arrives unsorted as well.
    import torch
    wl = workloads.small(seed=71, n_lines=20000, nu_max=200.0, cutoff=10.0, sorted_by_nu0=False)
    delta = np.random.default_rng(72).uniform(-0.02, 0.02, wl.n_lines)
    T, P = 1200.0, 50.0
    assert np.count_nonzero(np.diff(np.sort(wl.nu0) + delta[np.argsort(wl.nu0)] * P) < 0) > 5000
    ref = oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, delta=delta)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, delta=delta)
    for prec, bar in ((hk.HK_FP64, BAR), (hk.HK_FP32, BAR32)):
        got = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, lines_sorted=False, precision=prec)
        torch.cuda.synchronize()
        _check(got.cpu().numpy(), ref, bar)
    ctx = hk.Context(lines, lines_sorted=False)
    for Pc in (50.0, 0.01):
        a = ctx.opacity(T, Pc, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
        assert torch.equal(a, hk.hk_opacity(lines, T, Pc, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, lines_sorted=False))
    ctx.close()


def test_context_with_a_pressure_shift_and_bad_fractions():
    import torch
    wl = workloads.small(seed=61, n_lines=50, nu_max=50.0, cutoff=25.0)
    ex = _fields(wl, 62)
    shifted = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, delta=ex["delta"])
    ctx = hk.Context(shifted)                                       # the shift is applied by a1 at every pressure
    for P in (0.5, 40.0):
        a = ctx.opacity(1200.0, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
        b = hk.hk_opacity(shifted, 1200.0, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
        assert torch.equal(a, b)
        _check(a.cpu().numpy(), oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, 1200.0, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                                    delta=ex["delta"]), BAR)
    ctx.close()
    ls = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, gamma_self=ex["gamma_self"])
    for kw in (dict(self_fraction=1.5), dict(abundance=-1.0)):
        with pytest.raises(hk.HKError) as e:
            hk.hk_opacity(ls, 1000.0, 1.0, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, **kw)
        assert e.value.code == -1
    ctx = hk.Context(ls, self_fraction=0.3)
    got = ctx.opacity(1000.0, 1.0, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff).cpu().numpy()
    ctx.close()
    _check(got, oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, 1000.0, 1.0, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                    gamma_self=ex["gamma_self"], self_fraction=0.3), BAR)


@pytest.mark.parametrize("T,P,W,cap", [(1500.0, 1.0, 500.0, 25.0), (296.0, 1.0, 40.0, 25.0), (1000.0, 30.0, 20.0, 100.0),
                                         (2000.0, 0.01, 500.0, 3.0)])
def test_relative_cutoff_in_lorentz_widths(T, P, W, cap):
    # line i truncated at min(cap, W gamma_i); windows are no longer ordered like the centres
    import torch
    wl = workloads.small(seed=71, n_lines=2500, nu_max=300.0, cutoff=cap)
    ex = _fields(wl, 72)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, gamma_self=ex["gamma_self"])
    ref = oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, cap, gamma_self=ex["gamma_self"],
                              cutoff_widths=W)
    ref_abs = oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, cap, gamma_self=ex["gamma_self"])
    for prec, bar in ((hk.HK_FP64, BAR), (hk.HK_FP32, BAR32)):
        got = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, cap, cutoff_widths=W, precision=prec)
        torch.cuda.synchronize()
        _check(got.cpu().numpy(), ref, bar)
    if W * 0.02 * P * (296.0 / T) ** 0.5 < cap:
        assert not np.array_equal(ref, ref_abs)                      # the relative cutoff binds for some line
    # single line: bit-exact support (index work in FP64 on both sides)
    one = hk.Lines.from_numpy(wl.nu0[100:101], wl.S[100:101], wl.gamma0[100:101])
    got1 = hk.hk_opacity(one, 296.0, 1.0, wl.nu_min, wl.nu_max, wl.dnu, cap, cutoff_widths=W).cpu().numpy()
    ref1 = oracle.opacity_full(wl.nu0[100:101], wl.S[100:101], wl.gamma0[100:101], 296.0, 1.0, wl.nu_min, wl.nu_max, wl.dnu, cap,
                               cutoff_widths=W)
    assert np.array_equal(got1 != 0.0, ref1 != 0.0)
    with pytest.raises(hk.HKError):
        hk.hk_opacity(one, 296.0, 1.0, wl.nu_min, wl.nu_max, wl.dnu, cap, cutoff_widths=-1.0)


def test_host_buffer_form_with_every_optional_field():
    import torch
    wl = workloads.small(seed=81, n_lines=1200, nu_max=120.0, cutoff=25.0, with_E=True)
    ex = _fields(wl, 82)
    T, P, q = 900.0, 20.0, wl.q_ratio(900.0)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low, **ex)
    for prec in (hk.HK_FP64, hk.HK_FP32):
        dev = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, self_fraction=0.4, abundance=0.6,
                            cutoff_widths=300.0, precision=prec)
        kt = hk.hk_kdist(dev, wl.dnu, wl.bin_width, wl.n_g)
        hk_kap, hk_k = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, E_low=wl.E_low,
                                          q_ratio=q, self_fraction=0.4, abundance=0.6, cutoff_widths=300.0, precision=prec,
                                          bin_width=wl.bin_width, n_g=wl.n_g, **ex)
        assert torch.equal(hk_kap, dev.cpu()) and torch.equal(hk_k, kt.cpu())
    ref = oracle.opacity_full(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, E_low=wl.E_low, q_ratio=q,
                              self_fraction=0.4, abundance=0.6, cutoff_widths=300.0, **ex)
    _check(hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, self_fraction=0.4, abundance=0.6,
                         cutoff_widths=300.0).cpu().numpy(), ref, BAR)
