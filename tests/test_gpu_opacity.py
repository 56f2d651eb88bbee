"""Parity of hk_opacity (C ABI, CUDA) against the oracle on the same seeded inputs.

Bar (BASELINE.json north_star): max relative error <= 1e-6 at grid points with kappa >= 1e-12 * max(kappa).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk

BAR = 1.0e-6
BAR32 = 1.0e-4      # north_star: "<= 1e-4 (optional FP32 path)"


def _gpu_kappa(wl, T, P, q_ratio=1.0, **kw):
    import torch
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low)
    k = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu, q_ratio=q_ratio, **kw)
    torch.cuda.synchronize()
    return k.cpu().numpy()


def _check(got, ref, ref_max=None, bar=BAR):
    ref_max = ref.max() if ref_max is None else ref_max
    mask = ref >= 1e-12 * ref_max
    assert np.all(np.isfinite(got))
    rel = np.abs(got[mask] / ref[mask] - 1.0)
    assert rel.max() <= bar, (rel.max(), np.flatnonzero(mask)[np.argmax(rel)])
    assert np.all(got[ref == 0.0] == 0.0)
    return rel.max()


def test_config0_full_grid():
    wl = workloads.config(0)
    T, P = wl.T[0], wl.P_atm[0]
    got = _gpu_kappa(wl, T, P)
    ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    assert got.shape == ref.shape == (300000,)
    _check(got, ref)
    got32 = _gpu_kappa(wl, T, P, precision=hk.HK_FP32)
    e32 = _check(got32, ref, bar=BAR32)
    assert e32 > 1e-9                      # it is a different arithmetic, not the FP64 path under another name


@pytest.mark.parametrize("n_lines,nu_max,cutoff,T,P", [
    (1, 40.0, 25.0, 1500.0, 1.0),
    (50, 33.33, 7.0, 300.0, 1e-3),        # ragged: N = 3333 is not a multiple of the tile or the warp span
    (400, 123.45, 25.0, 2500.0, 10.0),
    (2000, 250.0, 100.0, 1000.0, 1e-5),   # Doppler-dominated: tiny y, series region
    (300, 60.0, 25.0, 800.0, 100.0),      # Lorentz-dominated: y >> 1
])
def test_small_cases_full_grid(n_lines, nu_max, cutoff, T, P):
    wl = workloads.small(seed=n_lines, n_lines=n_lines, nu_max=nu_max, cutoff=cutoff, T=T, P_atm=P)
    got = _gpu_kappa(wl, T, P)
    ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    _check(got, ref)
    _check(_gpu_kappa(wl, T, P, precision=hk.HK_FP32), ref, bar=BAR32)


@pytest.mark.parametrize("P", [1e-10, 1e-13])                    # y = gamma/alpha ~ 1e-9 and ~ 1e-12: far below the 1e-8 switch
@pytest.mark.parametrize("dnu", [0.1, 0.02, 0.0065, 0.001])       # alpha/dnu ~ 0.2, 1, 3, 20 at nu0 = 5000 cm^-1, T = 1500 K
def test_tiny_damping_on_coarse_and_fine_grids(P, dnu):
    # with y < 1e-8 the 6-point rule adds the Gaussian term exp(-x^2) out to x^2 ~ 41...50; on a grid coarser
    # than the line (alpha/dnu < 3) those points reach x^2 > 709, where an unclamped exp_fast wrapped its exponent field
    rng = np.random.default_rng(7)
    n = 60
    nu0 = np.sort(rng.uniform(4990.0, 5010.0, n))
    S = 10.0 ** rng.uniform(-24.0, -19.0, n)
    g0 = rng.uniform(0.02, 0.1, n)
    T, nu_min, nu_max, cutoff = 1500.0, 4980.0, 5020.0, 5.0
    lines = hk.Lines.from_numpy(nu0, S, g0)
    ref = oracle.opacity(nu0, S, g0, T, P, nu_min, nu_max, dnu, cutoff)
    for prec, bar in ((hk.HK_FP64, BAR), (hk.HK_FP32, BAR32)):
        got = hk.hk_opacity(lines, T, P, nu_min, nu_max, dnu, cutoff, precision=prec).cpu().numpy()
        assert np.all(got >= 0.0)
        _check(got, ref, bar=bar)


def test_pure_doppler_lines_gamma_zero():
    # gamma0 = 0 and no natural width gives y = 0, K(x, 0) = exp(-x^2): the profile is finite everywhere
    # (1/y used to be inf) and matches the oracle; mixed with ordinary lines, on a fine and on a coarse grid
    rng = np.random.default_rng(11)
    n = 40
    nu0 = np.sort(rng.uniform(2990.0, 3010.0, n))
    S = 10.0 ** rng.uniform(-24.0, -19.0, n)
    g0 = rng.uniform(0.02, 0.1, n)
    g0[::2] = 0.0
    T, P, nu_min, nu_max, cutoff = 1500.0, 1.0, 2980.0, 3020.0, 5.0
    lines = hk.Lines.from_numpy(nu0, S, g0)
    for dnu in (0.001, 0.01, 0.05):
        ref = oracle.opacity(nu0, S, g0, T, P, nu_min, nu_max, dnu, cutoff)
        for prec, bar in ((hk.HK_FP64, BAR), (hk.HK_FP32, BAR32)):
            got = hk.hk_opacity(lines, T, P, nu_min, nu_max, dnu, cutoff, precision=prec).cpu().numpy()
            _check(got, ref, bar=bar)
    # all lines without damping: kappa is a sum of Gaussians, zero (to underflow) between them
    only = hk.Lines.from_numpy(nu0, S, np.zeros(n))
    ref = oracle.opacity(nu0, S, np.zeros(n), T, P, nu_min, nu_max, 0.002, cutoff)
    got = hk.hk_opacity(only, T, P, nu_min, nu_max, 0.002, cutoff).cpu().numpy()
    assert np.all(np.isfinite(got)) and np.all(got >= 0.0)
    mask = ref >= 1e-12 * ref.max()
    assert np.abs(got[mask] / ref[mask] - 1.0).max() <= BAR


def test_lines_far_up_the_spectrum_small_alpha_to_large_alpha():
    # same draw shifted to 20000-20100 cm^-1: alpha ~ 0.08, several regimes per tile
    wl = workloads.small(seed=77, n_lines=500, nu_max=100.0, cutoff=25.0)
    wl.nu0 = wl.nu0 + 20000.0
    wl.nu_min, wl.nu_max = 20000.0, 20100.0
    T, P = 1500.0, 1.0
    got = _gpu_kappa(wl, T, P)
    ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    _check(got, ref)
    _check(_gpu_kappa(wl, T, P, precision=hk.HK_FP32), ref, bar=BAR32)


def test_window_semantics_bit_exact_support():
    import torch
    # a line exactly on a grid node with cutoff an exact multiple of dnu; one outside the grid within the cutoff;
    # one beyond the cutoff; one at nu0 = 0 (alpha = 0: Lorentzian)
    nu0 = np.array([-10.0, 0.0, 50.0, 130.0])
    S = np.full(4, 1e-20)
    g0 = np.full(4, 0.05)
    lines = hk.Lines.from_numpy(nu0, S, g0)
    for sel in ([2], [0], [3], [1], [0, 1, 2, 3]):
        sub = hk.Lines.from_numpy(nu0[sel], S[sel], g0[sel])
        ref = oracle.opacity(nu0[sel], S[sel], g0[sel], 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0)
        for prec, bar in ((hk.HK_FP64, BAR), (hk.HK_FP32, BAR32)):
            got = hk.hk_opacity(sub, 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0, precision=prec).cpu().numpy()
            assert np.array_equal(got != 0.0, ref != 0.0), sel      # support: index work is bit-exact (FP64 in both variants)
            if ref.any():
                _check(got, ref, bar=bar)
    got = hk.hk_opacity(hk.Lines.from_numpy(nu0[[2]], S[[2]], g0[[2]]), 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0).cpu().numpy()
    nz = np.flatnonzero(got)
    assert nz[0] == 2500 and nz[-1] == 7500 and nz.size == 5001
    torch.cuda.synchronize()


def test_no_lines_gives_zero():
    import torch
    empty = hk.Lines(torch.empty(0, dtype=torch.float64, device="cuda"), torch.empty(0, dtype=torch.float64, device="cuda"),
                     torch.empty(0, dtype=torch.float64, device="cuda"))
    out = torch.full((1000,), 7.0, dtype=torch.float64, device="cuda")
    hk.hk_opacity(empty, 1000.0, 1.0, 0.0, 10.0, 0.01, 25.0, out=out)
    assert not out.cpu().numpy().any()


def test_deterministic_bitwise():
    wl = workloads.small(seed=3, n_lines=3000, nu_max=200.0, cutoff=25.0)
    for prec in (hk.HK_FP64, hk.HK_FP32):
        a = _gpu_kappa(wl, 1500.0, 1.0, precision=prec)
        b = _gpu_kappa(wl, 1500.0, 1.0, precision=prec)
        assert np.array_equal(a, b)


def test_line_strength_scaling_path():
    wl = workloads.small(seed=9, n_lines=600, nu_max=120.0, cutoff=25.0, with_E=True, T=900.0)
    for T in (500.0, 900.0, 3000.0):
        q = wl.q_ratio(T)
        got = _gpu_kappa(wl, T, 1.0, q_ratio=q)
        ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, 1.0, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, E_low=wl.E_low, q_ratio=q)
        _check(got, ref)
        _check(_gpu_kappa(wl, T, 1.0, q_ratio=q, precision=hk.HK_FP32), ref, bar=BAR32)


def test_context_form_matches_one_shot():
    import torch
    wl = workloads.small(seed=4, n_lines=800, nu_max=150.0, cutoff=25.0, with_E=True)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low)
    ctx = hk.Context(lines, mass_amu=18.0)
    for T, P in ((700.0, 0.1), (2000.0, 5.0)):
        q = wl.q_ratio(T)
        a = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q)
        b = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q)
        torch.cuda.synchronize()
        assert torch.equal(a, b)
    ctx.close()


def test_error_codes():
    import torch
    lines = hk.Lines.from_numpy([1.0, 2.0], [1e-20, 1e-20], [0.05, 0.05])
    bad = [dict(T=-1.0), dict(P_atm=0.0), dict(dnu=0.0), dict(cutoff=-5.0), dict(mass_amu=0.0), dict(T=float("nan"))]
    base = dict(T=1000.0, P_atm=1.0, nu_min=0.0, nu_max=10.0, dnu=0.01, cutoff=25.0, mass_amu=18.0)
    for b in bad:
        kw = dict(base)
        kw.update(b)
        with pytest.raises(hk.HKError) as e:
            hk.hk_opacity(lines, kw["T"], kw["P_atm"], kw["nu_min"], kw["nu_max"], kw["dnu"], kw["cutoff"],
                          mass_amu=kw["mass_amu"], out=torch.empty(1000, dtype=torch.float64, device="cuda"))
        assert e.value.code == -1
    with pytest.raises(hk.HKError) as e:
        hk.hk_opacity(lines, 1000.0, 1.0, 0.0, 10.0, 0.01, 25.0, precision=7)
    assert e.value.code == -1
    with pytest.raises(hk.HKError):
        hk.hk_opacity(lines, 1000.0, 1.0, 10.0, 0.0, 0.01, 25.0, out=torch.empty(1, dtype=torch.float64, device="cuda"))
    assert hk.hk_lines_check_sorted(lines.nu0)
    assert not hk.hk_lines_check_sorted(torch.tensor([2.0, 1.0], dtype=torch.float64, device="cuda"))


def test_config1_full_size_full_grid():
    # the configuration bench.py times: 1e5 lines, 3e6 points, cutoff 100 — the oracle on EVERY grid point (2e9 line-point
    # evaluations, ~15 s of the host cores) and on every k-table row; the mask threshold is the oracle's own maximum (A11)
    wl = workloads.config(1)
    T, P = wl.T[0], wl.P_atm[0]
    got = _gpu_kappa(wl, T, P)
    assert got.shape == (3_000_000,)
    ref = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    _check(got, ref)
    assert got.min() > 0.0
    got32 = _gpu_kappa(wl, T, P, precision=hk.HK_FP32)
    _check(got32, ref, bar=BAR32)
    import torch
    kref = oracle.kdist(ref, 1000, wl.n_g)
    for g, bar in ((got, BAR), (got32, BAR32)):
        kt = hk.hk_kdist(torch.as_tensor(g).cuda(), wl.dnu, wl.bin_width, wl.n_g).cpu().numpy()
        assert kt.shape == kref.shape == (3000, 20)
        m = kref >= 1e-12 * kref.max()
        assert np.abs(kt[m] / kref[m] - 1.0).max() <= bar


def test_config2_pressure_sweep_whole_bins_and_sampled_points():
    # 1e6 lines, six pressures from Doppler- to Lorentz-dominated; per pressure the oracle on 8 whole 1000-point bins (both
    # ends of the grid among them) and at 1500 seeded points; mask threshold from the oracle's values of the compared set
    wl = workloads.config(2)
    T = wl.T[0]
    rng = np.random.default_rng(2)
    js = np.sort(rng.choice(wl.n_points, 1500, replace=False))
    bins = np.sort(np.concatenate(([0, 2999], rng.choice(np.arange(1, 2999), 6, replace=False))))
    jb = (bins[:, None] * 1000 + np.arange(1000)[None, :]).ravel()
    import torch
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    ctx = hk.Context(lines)
    ctx32 = hk.Context(lines, precision=hk.HK_FP32)
    for P in wl.P_atm:
        got = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
        got32 = ctx32.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
        torch.cuda.synchronize()
        got, got32 = got.cpu().numpy(), got32.cpu().numpy()
        for idx in (js, jb):
            ref = oracle.opacity_points(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, idx)
            _check(got[idx], ref)
            _check(got32[idx], ref, bar=BAR32)
    ctx.close()
    ctx32.close()


def test_unsorted_input_is_sorted_on_a_copy():
    import torch
    wl = workloads.small(seed=21, n_lines=5000, nu_max=150.0, cutoff=25.0, with_E=True, sorted_by_nu0=False)
    assert np.any(np.diff(wl.nu0) < 0)
    T, P, q = 1200.0, 0.5, wl.q_ratio(1200.0)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low)
    before = [t.clone() for t in (lines.nu0, lines.S, lines.gamma0, lines.E_low)]
    got = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, lines_sorted=False)
    ctx = hk.Context(lines, lines_sorted=False)
    got_ctx = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q)
    torch.cuda.synchronize()
    ctx.close()
    for a, b in zip(before, (lines.nu0, lines.S, lines.gamma0, lines.E_low)):
        assert torch.equal(a, b)                                     # inputs are never modified
    idx = np.argsort(wl.nu0, kind="stable")
    ref = oracle.opacity(wl.nu0[idx], wl.S[idx], wl.gamma0[idx], T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                         E_low=wl.E_low[idx], q_ratio=q)
    _check(got.cpu().numpy(), ref)
    assert torch.equal(got, got_ctx)
    # an ordered list passed with lines_sorted=False takes the no-copy path and gives the same bits as lines_sorted=True
    s = hk.Lines.from_numpy(wl.nu0[idx], wl.S[idx], wl.gamma0[idx], E_low=wl.E_low[idx])
    a = hk.hk_opacity(s, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, lines_sorted=False)
    b = hk.hk_opacity(s, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, lines_sorted=True)
    assert torch.equal(a, b) and torch.equal(a, got)


def test_host_buffer_form_matches_device_form():
    import torch
    wl = workloads.small(seed=5, n_lines=1500, nu_max=200.0, cutoff=25.0)
    T, P = 1500.0, 1.0
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    ktab = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g)
    pin = lambda a: torch.as_tensor(a).pin_memory()
    hk_kap, hk_k = hk.hk_opacity_host(pin(wl.nu0), pin(wl.S), pin(wl.gamma0), T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                      bin_width=wl.bin_width, n_g=wl.n_g)
    assert torch.equal(hk_kap, kap.cpu()) and torch.equal(hk_k, ktab.cpu())
    # pageable numpy buffers, k-table only
    none_kap, k2 = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                      bin_width=wl.bin_width, n_g=wl.n_g, want_kappa=False)
    assert none_kap is None and torch.equal(k2, ktab.cpu())
    with pytest.raises(hk.HKError):
        hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, want_kappa=False)


@pytest.mark.parametrize("precision", [hk.HK_FP64, hk.HK_FP32])
def test_host_buffer_form_on_a_grid_wide_enough_for_the_ranged_path(precision):
    # with >= 48 far-kernel tiles hk_opacity_host runs a3 as six tapered (far, near) launch pairs on
    # streams of their own and copies each range of kappa back as it becomes final; the other host-form tests stay below
    # that size.  N = 100 003 (prime: ragged last tile, last plan block and last range) is 98 tiles of 1024 points (FP64)
    # or 391 of 256 (FP32 variant).  The result must be the bits of the device form.
    import torch
    wl = workloads.small(seed=33, n_lines=6000, nu_max=1000.03, cutoff=25.0, bin_width=None)
    assert wl.n_points == 100003
    T, P = 1100.0, 0.3
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, precision=precision)
    pin = lambda a: torch.as_tensor(a).pin_memory()
    h = [pin(wl.nu0), pin(wl.S), pin(wl.gamma0)]
    for _ in range(3):                                       # the streams and events of the ranges are reused between calls
        got, none_k = hk.hk_opacity_host(*h, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, precision=precision)
        assert none_k is None and torch.equal(got, kap.cpu())
    # a mixture: the running sum goes up with the call, every range adds to its own part and comes back
    run = torch.full((wl.n_points,), 3.0, dtype=torch.float64).pin_memory()
    dev = torch.full((wl.n_points,), 3.0, dtype=torch.float64, device="cuda")
    hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=dev, accumulate=True, abundance=0.25,
                  precision=precision)
    hk.hk_opacity_host(*h, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, kappa_out=run, accumulate=True, abundance=0.25,
                       precision=precision)
    assert torch.equal(run, dev.cpu())


@pytest.mark.parametrize("precision", [hk.HK_FP64, hk.HK_FP32])
def test_host_buffer_form_ranged_path_with_the_k_table(precision):
    # the same path with the k-distribution behind it (what bench.py's e2e leg times at config 1): kappa and k-table, and
    # the k-table alone (one range: nothing to copy early)
    import torch
    wl = workloads.small(seed=34, n_lines=4000, nu_max=800.0, cutoff=100.0, bin_width=10.0)
    assert wl.n_points == 80000
    T, P = 1500.0, 1.0
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, precision=precision)
    ktab = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g)
    hk_kap, hk_k = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                      bin_width=wl.bin_width, n_g=wl.n_g, precision=precision)
    assert torch.equal(hk_kap, kap.cpu()) and torch.equal(hk_k, ktab.cpu())
    none_kap, k2 = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                      bin_width=wl.bin_width, n_g=wl.n_g, want_kappa=False, precision=precision)
    assert none_kap is None and torch.equal(k2, ktab.cpu())


def test_fp32_variant_stays_inside_the_float_range():
    # the float 1-/2-point rules invert ~d^8.  (1) Lines 7e4 - 1.2e5 cm^-1 away from the grid under a
    # cutoff that admits them (d^8 > 3.4e38: the product overflowed and the wing was dropped without notice); (2) a grid of
    # 2e-6 cm^-1 with lines narrow enough that the 1-point rule starts three grid points from the centre (d^8 denormal:
    # NaN); (3) a strong line that does not reach a span must not flush a weak one of its batch that does
    rng = np.random.default_rng(77)
    T, P = 1500.0, 1.0
    far0 = np.sort(rng.uniform(7.0e4, 1.2e5, 30))
    near0 = np.sort(rng.uniform(0.0, 80.0, 5))
    nu0 = np.concatenate((near0, far0))
    S = np.concatenate((np.full(5, 1e-27), 10.0 ** rng.uniform(-20.0, -19.0, 30)))
    g0 = rng.uniform(0.02, 0.1, 35)
    lines = hk.Lines.from_numpy(nu0, S, g0)
    ref = oracle.opacity(nu0, S, g0, T, P, 0.0, 80.0, 0.01, 1.0e6)
    only_near = oracle.opacity(near0, S[:5], g0[:5], T, P, 0.0, 80.0, 0.01, 1.0e6)
    assert np.median(ref / np.maximum(only_near, 1e-300)) > 2.0           # the distant lines matter on this grid
    _check(hk.hk_opacity(lines, T, P, 0.0, 80.0, 0.01, 1.0e6, precision=hk.HK_FP32).cpu().numpy(), ref, bar=BAR32)
    _check(hk.hk_opacity(lines, T, P, 0.0, 80.0, 0.01, 1.0e6).cpu().numpy(), ref)
    with pytest.raises(hk.HKError) as e:
        hk.hk_opacity(lines, T, P, 0.0, 80.0, 0.01, 3.0e6, precision=hk.HK_FP32)
    assert e.value.code == -5
    # (2)
    nu0 = np.sort(rng.uniform(0.008, 0.032, 40))
    S = 10.0 ** rng.uniform(-24.0, -20.0, 40)
    g0 = rng.uniform(0.02, 0.1, 40)
    T, P, dnu = 300.0, 2.0e-4, 2.0e-6
    lines = hk.Lines.from_numpy(nu0, S, g0)
    ref = oracle.opacity(nu0, S, g0, T, P, 0.0, 0.04, dnu, 0.01)
    assert ref.shape == (20000,)
    got32 = hk.hk_opacity(lines, T, P, 0.0, 0.04, dnu, 0.01, precision=hk.HK_FP32).cpu().numpy()
    _check(got32, ref, bar=BAR32)
    _check(hk.hk_opacity(lines, T, P, 0.0, 0.04, dnu, 0.01).cpu().numpy(), ref)
    # (3) one batch of 32 lines under a relative cutoff of 100 Lorentz widths (windows of +-2.2 cm^-1): the line at 10 cm^-1,
    # 2^150 stronger, is in the batch of every span up to 35 cm^-1 (the tables know the absolute cutoff) and reaches none
    # of the spans of the weak lines at 20 - 30 cm^-1
    nu0 = np.concatenate(([10.0], np.linspace(20.0, 30.0, 31)))
    S = np.concatenate(([1.0e-10], np.full(31, 1.0e-56)))
    g0 = np.full(32, 0.05)
    lines = hk.Lines.from_numpy(nu0, S, g0)
    ref = oracle.opacity_full(nu0, S, g0, 1500.0, 1.0, 0.0, 100.0, 0.01, 25.0, cutoff_widths=100.0)
    got32 = hk.hk_opacity(lines, 1500.0, 1.0, 0.0, 100.0, 0.01, 25.0, precision=hk.HK_FP32, cutoff_widths=100.0).cpu().numpy()
    weak = np.arange(1500, 10000)                                         # beyond the strong line's own window
    assert ref[weak].max() > 0.0 and ref[:1500].max() > 1e40 * ref[weak].max()
    _check(got32[weak], ref[weak], bar=BAR32)


@pytest.mark.parametrize("precision", [hk.HK_FP64, hk.HK_FP32])
def test_host_buffer_form_on_a_long_grid_with_the_k_table(precision):
    # 1.6e6 grid points with 1000-point bins: long enough for the library to cut its six ranges at multiples of lcm(tile, bin)
    # (128 000 points for the FP64 tile of 1024, 32 000 for the FP32 variant's 256) and sort each range's bins on the range's
    # own stream — the path a build with -DHK_HOST_KDIST_BY_RANGE takes (off by default: it measured slower); either way the
    # result is the bits of the device form.  Twice, so that the per-thread streams and events are reused
    import torch
    wl = workloads.small(seed=35, n_lines=5000, nu_max=16000.0, cutoff=25.0, bin_width=10.0)
    assert wl.n_points == 1_600_000
    T, P = 1500.0, 1.0
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, precision=precision)
    ktab = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g)
    for _ in range(2):
        hk_kap, hk_k = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                          bin_width=wl.bin_width, n_g=wl.n_g, precision=precision)
        assert torch.equal(hk_kap, kap.cpu()) and torch.equal(hk_k, ktab.cpu())
    # a bin width that shares no useful multiple with the tile (1250 points: lcm 160 000, ten units)
    k2 = hk.hk_kdist(kap, wl.dnu, 12.5, wl.n_g)
    _, hk_k2 = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, bin_width=12.5,
                                  n_g=wl.n_g, precision=precision)
    assert torch.equal(hk_k2, k2.cpu())
