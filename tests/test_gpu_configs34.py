"""Parity at BASELINE.json's full sizes for config 3 (1e8 lines, ramped density, 300 bins x 10000 points) and
config 4 (T-P table: 1e6 lines with eq.-18 line strengths, 20 T x 10 P), in the launch configuration bench.py uses
(hk.Context / hk_opacity + hk_kdist on the whole grid).  The oracle cannot cover these grids in test time
(5e11 / 4e12 line-point evaluations), so it is called on seeded samples: single points and whole bins, every line that
can reach them included.  Bar: max relative error <= 1e-6 where the oracle value >= 1e-12 * max (north_star).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk

BAR = 1.0e-6
BAR32 = 1.0e-4      # the optional FP32 variant (north_star)


def _reach(wl, j_lo, j_hi):
    """Slice of the (ordered) line list that can reach grid points j_lo..j_hi: a superset, the oracle windows exactly."""
    lo = np.searchsorted(wl.nu0, wl.nu_min + j_lo * wl.dnu - wl.cutoff - 1.0, "left")
    hi = np.searchsorted(wl.nu0, wl.nu_min + j_hi * wl.dnu + wl.cutoff + 1.0, "right")
    return slice(int(lo), int(hi))


def _oracle_points(wl, T, P, js, q_ratio=1.0):
    sl = _reach(wl, int(js.min()), int(js.max()))
    E = None if wl.E_low is None else wl.E_low[sl]
    return oracle.opacity_points(wl.nu0[sl], wl.S[sl], wl.gamma0[sl], T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, js,
                                 E_low=E, q_ratio=q_ratio)


def _check(got, ref, bar=BAR):
    mask = ref >= 1e-12 * ref.max()          # the oracle's maximum over the compared set (A11)
    assert np.all(np.isfinite(got))
    rel = np.abs(got[mask] / ref[mask] - 1.0)
    assert rel.max() <= bar, (rel.max(), int(np.argmax(rel)))
    return float(rel.max())


def test_config3_hot_line_list_scale_full_size():
    import torch
    wl = workloads.config(3)                                      # 1e8 lines, 2.4 GB of float64 on the host
    assert wl.n_lines == 100_000_000 and wl.n_points == 3_000_000
    T, P = wl.T[0], wl.P_atm[0]
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    ctx = hk.Context(lines)
    kap = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)          # warm-up (allocates scratch)
    ktab = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g)
    got = kap.cpu().numpy()
    gk = ktab.cpu().numpy()
    ctx.close()
    # the optional FP32 variant of this config (BASELINE.json configs[3]: "FP64 with an optional FP32 variant")
    ctx32 = hk.Context(lines, precision=hk.HK_FP32)
    kap = ctx32.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=kap)
    got32 = kap.cpu().numpy()
    gk32 = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g).cpu().numpy()
    ctx32.close()
    assert np.abs(got32 / got - 1.0).max() <= 1.5 * BAR32             # every grid point, against the FP64 variant
    assert got.shape == (3_000_000,) and gk.shape == (300, 20)
    # (1) short runs of consecutive points across the density ramp, including both ends of the grid
    rng = np.random.default_rng(3)
    starts = np.concatenate(([0, wl.n_points - 40], rng.integers(0, wl.n_points - 40, 6)))
    for s in starts:
        js = np.arange(s, s + 40, dtype=np.int64)
        ref = _oracle_points(wl, T, P, js)
        _check(got[js], ref)
        _check(got32[js], ref, BAR32)
    # (2) whole k-distribution bins (10000 points each): kappa and the k-table row.  Bin 0 is the dense end of the ramp:
    # 3.3e5 lines per point (the longest accumulations, the FP32 variant's hardest case) and the alpha -> 0 lines near
    # nu0 = 0, ~3e9 line-point evaluations of the oracle; the others lie where it finishes in seconds
    for b in (0, 299, 262, 231):
        js = np.arange(b * 10000, (b + 1) * 10000, dtype=np.int64)
        ref = _oracle_points(wl, T, P, js)
        _check(got[js], ref)
        _check(got32[js], ref, BAR32)
        kref = oracle.kdist(ref, 10000, wl.n_g)[0]
        assert np.abs(gk[b] / kref - 1.0).max() <= BAR
        assert np.abs(gk32[b] / kref - 1.0).max() <= BAR32
    assert np.all(np.diff(gk, axis=1) >= 0.0)


def test_config4_tp_table_full_size():
    import torch
    wl = workloads.config(4)
    assert wl.n_lines == 1_000_000 and len(wl.T) == 20 and len(wl.P_atm) == 10
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low)
    ctx = hk.Context(lines)
    N, ppb = wl.n_points, 1000
    kap = torch.empty(N, dtype=torch.float64, device="cuda")
    ktab = torch.empty((N // ppb, wl.n_g), dtype=torch.float64, device="cuda")
    rng = np.random.default_rng(4)
    pairs = [(it, ip) for it in range(20) for ip in range(10)]
    checked = {(0, 0), (0, 9), (19, 0), (19, 9)} | {pairs[i] for i in rng.choice(200, 12, replace=False)}
    ctx.opacity(wl.T[0], wl.P_atm[0], wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=wl.q_ratio(wl.T[0]), out=kap)
    worst = 0.0
    for it, ip in pairs:                                          # the whole table: 200 opacity functions + k-tables
        T, P = wl.T[it], wl.P_atm[ip]
        q = wl.q_ratio(T)

        def step():
            ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, out=kap)
            hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g, out=ktab)
        step()
        if (it, ip) not in checked:
            continue
        got, gk = kap.cpu().numpy(), ktab.cpu().numpy()
        for b in rng.choice(N // ppb, 2, replace=False):         # two whole bins: kappa and the k-table row
            js = np.arange(b * ppb, (b + 1) * ppb, dtype=np.int64)
            ref = _oracle_points(wl, T, P, js, q_ratio=q)
            worst = max(worst, _check(got[js], ref))
            kref = oracle.kdist(ref, ppb, wl.n_g)[0]
            m = kref >= 1e-12 * kref.max()
            assert np.abs(gk[b][m] / kref[m] - 1.0).max() <= BAR
        js = np.sort(rng.choice(N, 200, replace=False)).astype(np.int64)     # scattered points over the whole grid
        sl_ref = oracle.opacity_points(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, js,
                                       E_low=wl.E_low, q_ratio=q)
        worst = max(worst, _check(got[js], sl_ref))
    ctx.close()
    assert worst <= BAR
