"""Parity at BASELINE.json's full sizes for config 3 (1e8 lines, ramped density, 300 bins x 10000 points) and
config 4 (T-P table: 1e6 lines with eq.-18 line strengths, 20 T x 10 P), in the launch configuration bench.py uses
(hk.Context / hk_opacity + hk_kdist on the whole grid).  The oracle cannot cover these grids in test time
(5e11 / 4e12 line-point evaluations), so it is called on seeded samples: single points and whole bins, every line that
can reach them included.  Bar: max relative error <= 1e-6 where the oracle value >= 1e-12 * max (north_star).
"""
import json
import os
import time

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import workloads
import paper_1503_03806_b200 as hk

BAR = 1.0e-6
BAR32 = 1.0e-4      # the optional FP32 variant (north_star)
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _note(key, value):
    """Best-effort record of device timings for DESIGN.md / profiles (never read back by any test)."""
    try:
        d = os.path.join(ROOT, "gpurun_out")
        os.makedirs(d, exist_ok=True)
        path = os.path.join(d, "config_timings.json")
        cur = json.load(open(path)) if os.path.exists(path) else {}
        cur[key] = value
        json.dump(cur, open(path, "w"), indent=1)
    except OSError:
        pass


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


def _check(got, ref, ref_max, bar=BAR):
    mask = ref >= 1e-12 * ref_max
    assert np.all(np.isfinite(got))
    rel = np.abs(got[mask] / ref[mask] - 1.0)
    assert rel.max() <= bar, (rel.max(), int(np.argmax(rel)))
    return float(rel.max())


def _timed(fn):
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    out = fn()
    e1.record()
    torch.cuda.synchronize()
    return out, e0.elapsed_time(e1)


def test_config3_hot_line_list_scale_full_size():
    import torch
    t0 = time.time()
    wl = workloads.config(3)                                      # 1e8 lines, 2.4 GB of float64 on the host
    gen_s = time.time() - t0
    assert wl.n_lines == 100_000_000 and wl.n_points == 3_000_000
    T, P = wl.T[0], wl.P_atm[0]
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    ctx = hk.Context(lines)
    kap = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)          # warm-up (allocates scratch)
    kap, ms = _timed(lambda: ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=kap))
    ktab, ms_k = _timed(lambda: hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g))
    got = kap.cpu().numpy()
    gk = ktab.cpu().numpy()
    ctx.close()
    # the optional FP32 variant of this config (BASELINE.json configs[3]: "FP64 with an optional FP32 variant")
    ctx32 = hk.Context(lines, precision=hk.HK_FP32)
    kap = ctx32.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=kap)
    kap, ms32 = _timed(lambda: ctx32.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=kap))
    got32 = kap.cpu().numpy()
    gk32 = hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g).cpu().numpy()
    ctx32.close()
    n_evals = hk.hk_count_evals(wl.nu0, wl.nu_min, wl.n_points, wl.dnu, wl.cutoff)
    _note("config3", {"n_lines": wl.n_lines, "line_point_evals": n_evals, "opacity_ms": ms, "kdist_ms": ms_k,
                      "evals_per_s": n_evals / (ms * 1e-3), "host_generation_s": gen_s,
                      "fp32_variant_opacity_ms": ms32, "fp32_variant_evals_per_s": n_evals / (ms32 * 1e-3),
                      "fp32_vs_fp64_max_rel_diff_whole_grid": float(np.abs(got32 / got - 1.0).max())})
    assert np.abs(got32 / got - 1.0).max() <= 1.5 * BAR32             # every grid point, against the FP64 variant
    assert got.shape == (3_000_000,) and gk.shape == (300, 20)
    gmax = float(got.max())
    # (1) short runs of consecutive points across the density ramp, including both ends of the grid
    rng = np.random.default_rng(3)
    starts = np.concatenate(([0, wl.n_points - 40], rng.integers(0, wl.n_points - 40, 6)))
    for s in starts:
        js = np.arange(s, s + 40, dtype=np.int64)
        ref = _oracle_points(wl, T, P, js)
        _check(got[js], ref, gmax)
        _check(got32[js], ref, gmax, BAR32)
    # (2) whole k-distribution bins (10000 points each) where the oracle finishes in seconds: kappa and the k-table row
    for b in (299, 262, 231):
        js = np.arange(b * 10000, (b + 1) * 10000, dtype=np.int64)
        ref = _oracle_points(wl, T, P, js)
        _check(got[js], ref, gmax)
        _check(got32[js], ref, gmax, BAR32)
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
    total_ms, worst = 0.0, 0.0
    for it, ip in pairs:                                          # the whole table: 200 opacity functions + k-tables
        T, P = wl.T[it], wl.P_atm[ip]
        q = wl.q_ratio(T)

        def step():
            ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=q, out=kap)
            hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g, out=ktab)
        _, ms = _timed(step)
        total_ms += ms
        if (it, ip) not in checked:
            continue
        got, gk = kap.cpu().numpy(), ktab.cpu().numpy()
        gmax = float(got.max())
        for b in rng.choice(N // ppb, 2, replace=False):         # two whole bins: kappa and the k-table row
            js = np.arange(b * ppb, (b + 1) * ppb, dtype=np.int64)
            ref = _oracle_points(wl, T, P, js, q_ratio=q)
            worst = max(worst, _check(got[js], ref, gmax))
            kref = oracle.kdist(ref, ppb, wl.n_g)[0]
            m = kref >= 1e-12 * gmax
            assert np.abs(gk[b][m] / kref[m] - 1.0).max() <= BAR
        js = np.sort(rng.choice(N, 200, replace=False)).astype(np.int64)     # scattered points over the whole grid
        sl_ref = oracle.opacity_points(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, js,
                                       E_low=wl.E_low, q_ratio=q)
        worst = max(worst, _check(got[js], sl_ref, gmax))
    ctx.close()
    n_evals = hk.hk_count_evals(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff)
    _note("config4", {"pairs": 200, "line_point_evals_per_pair": n_evals, "table_ms": total_ms,
                      "evals_per_s": 200 * n_evals / (total_ms * 1e-3), "worst_rel_err_checked": worst})
