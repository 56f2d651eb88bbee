#!/usr/bin/env python
"""bench.py — the hot path of HELIOS-K on BASELINE.json's workloads.

One "step" = one whole opacity function plus its k-distribution through the C ABI:
    hk_opacity (a1 line prep, a2 tile plan, a3 Voigt accumulation, a4 kappa store)  +  hk_kdist (a5 per-bin sort, a6 resample)
The headline (`value`, `e2e`, `roofline`, `cpu_baseline`) is BASELINE.json configs[1] — the configuration the metric "...at
1e5 lines" is quoted on: 1e5 lines, 3e6 grid points, cutoff 100 cm^-1, 3000 bins x 1000 points, 20 Gauss-Legendre g-points, FP64.

    python bench.py [--gpus N] [--steps K] [--warmup W]                  our arm (CUDA, sm_100a)
    python bench.py --impl reference [...]                                the oracle, as it stands, on the host cores
    python bench.py --config k                                            one line for config k alone (same code as the `configs` key)
    python bench.py --stage-times                                         per-stage times of configs 1-3, both precisions

At N = 1 the default line also carries `parity` (the oracle's kappa and k-table rows of the cpu_baseline sample compared with
the GPU's of the same run: the run fails above 1e-6) and `configs`: configs 0, 2, 3, 4 at BASELINE size (config 2 all six
pressures, config 3 the full 1e8 lines, config 4 all 200 (T,P) pairs through hk.Context), each with CUDA-event times, line-point
evaluations/s, the regime census, the a3 roofline fraction, parity on seeded 1000-point units and the oracle's time on those
units extrapolated to the whole config by N_evals (SURVEY.md:386-391).  `--no-configs` leaves them out.

N > 1 (torchrun, one rank per GPU): the path shards with NO collective — rank r computes the opacity function of the r-th
(T, P) pair of a small T-P table over the same line list ("repeat this calculation for multiple combinations of
temperature and pressure"); rank 0 keeps config 1's (1500 K, 1 atm).  Per-GPU work is fixed: weak scaling.  NCCL is used only
for the barrier and the max-over-ranks of the device time.  `--shard grid` instead splits ONE opacity function of config 3 along
the wavenumber grid (shard.shard_grid: bin-aligned ranges balanced by line-point evaluations; strong scaling).

Prints ONE JSON line (rank 0).  `value` = line-point Voigt evaluations per second, whole job, inputs resident in HBM, device time
by CUDA events around each step (L2 flushed between steps, outside the events).  `e2e` = the same metric through
hk.hk_opacity_host(): pinned host line arrays -> device, both calls, kappa and the k-table -> pinned host, wall clock.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "voigt_line_point_evals_per_s"
UNIT = "line-point evals/s"
WORKLOAD = "BASELINE.json configs[1]: 1e5 lines, 3e6 grid points, cutoff 100 cm^-1, T=1500 K, P=1 atm, 3000 bins x 1000 pts, 20 g-points"
PARITY_BAR = 1.0e-6          # north_star, FP64 path
PARITY_BAR32 = 1.0e-4

# FP64-pipe thread-instructions the method needs per line-point evaluation, by regime.  The wing rules are
# counted from the formulas of hk_voigt.cuh with the Newton reciprocal; the series is counted from the kernel as built: the
# SASS of the near kernel's two-item series loop holds 136 DFMA + 16 DMUL + 14 DADD = 166 FP64 instructions for two
# evaluations.  These are per POINT, for the cheapest valid rule (hk_regime_census), not the rule a whole group happened to get.
FP64_INST_PER_EVAL = {"gh1": 5.0, "gh2": 7.0, "gh3": 11.0, "gh6": 22.0, "series": 83.0}
FAR_REGIMES, NEAR_REGIMES = ("gh1", "gh2", "gh3"), ("gh6", "series")
# --precision fp32: FP32-pipe thread-instructions per evaluation of the rules the far kernel runs in float (hk_voigt.cuh
# gh1_acc2f / gh2_acc2f: 8 and 13 per pair of points, + 1 MUFU.RCP per pair; gh3_accf: 10 + 1 MUFU.RCP per point)
FP32_INST_PER_EVAL = {"gh1": 4.0, "gh2": 6.5, "gh3": 10.0}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the roofline kernels, read from the committed `ncu --set full`
# summaries named here (not live: ncu cannot run inside a timed bench).  Not memory-bound: context only.
def _ncu_dram(*files):
    """Sum of the DRAM bytes (read + written) of one launch of each kernel, from profiles/<file>; None if a file is missing."""
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    total = 0.0
    for f in files:
        try:
            rows = [l.split() for l in open(os.path.join(ROOT, "profiles", f)) if l.startswith(("dram__bytes_read.sum ", "dram__bytes_write.sum "))]
        except OSError:
            return None
        if len(rows) != 2:
            return None
        total += sum(float(r[2]) * scale[r[1]] for r in rows)
    return total


NCU_DRAM = {"fp64": {"bytes": _ncu_dram("r03_voigt_far_kernel_ncu_full.txt", "r03_voigt_near_kernel_ncu_full.txt"),
                     "source": "profiles/r03_voigt_far_kernel_ncu_full.txt + r03_voigt_near_kernel_ncu_full.txt (ncu flushes the "
                               "caches before each kernel: the near kernel's 36.9 MB are the 24 MB of kappa the far kernel wrote, "
                               "L2-resident in a real step, plus line records)"},
            "fp32": {"bytes": _ncu_dram("r03_voigt_far32_kernel_ncu_full.txt"), "source": "profiles/r03_voigt_far32_kernel_ncu_full.txt"}}
NOMINAL_FP64_LANES = 148 * 64   # DFMA lanes of a B200 (B200_PROFILING.md): nominal peak = lanes x SM clock


def tp_table(wl, world):
    """(T, P_atm) of each rank: rank 0 is config 1's own pair; further ranks walk a small seeded-free T-P ladder."""
    pairs = [(wl.T[0], wl.P_atm[0])]
    for r in range(1, world):
        pairs.append((wl.T[0] * (1.0 + 0.1 * ((r + 1) // 2) * (1 if r % 2 else -1) / 2.0), wl.P_atm[0] * (2.0 ** ((r % 4) - 1))))
    return pairs


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the two timed regions (device-timed steps, then the
    e2e steps) run (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,"
         "utilization.gpu")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, load, pw, reasons = [], [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
                pw.append(float(r[3]))
            except ValueError:
                continue
            try:
                load.append(float(r[9]) >= 50.0)
            except (ValueError, IndexError):
                load.append(True)
            for k, nm in enumerate(names):
                if r[5 + k].lower().startswith("active"):
                    reasons.add(nm)
        # the GPU idles (and clocks down) while the host times the oracle between the legs: the median is over the samples
        # taken under load (utilization.gpu >= 50 %) when there are any
        busy = [v for v, b in zip(sm, load) if b] or sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "samples_under_load": int(sum(load)),
                "sm_mhz_min_under_load": min(busy) if busy else None, "power_w_max": max(pw) if pw else None}


def host_cores():
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def _reach(wl, j_lo, j_hi):
    """Slice of the (ordered) line list that can reach grid points j_lo..j_hi: a superset; the oracle windows exactly."""
    lo = np.searchsorted(wl.nu0, wl.nu_min + j_lo * wl.dnu - wl.cutoff - 1.0, "left")
    hi = np.searchsorted(wl.nu0, wl.nu_min + j_hi * wl.dnu + wl.cutoff + 1.0, "right")
    return slice(int(lo), int(hi))


def oracle_units(wl, T, P, target_s, unit, seed, q_ratio=1.0, with_kdist=False, max_units=None, include=(), min_units=2):
    """Times the oracle, as it stands, on seeded whole units of `unit` consecutive grid points (a k-distribution bin where the
    config has 1000-point bins): kappa of every point of the unit (+ the unit's k-distribution row when `with_kdist`).  A
    2-unit pilot sizes the sample for about `target_s` seconds.  Returns a dict with the timing, the sampled indices and the
    oracle's values (for the parity check of the same run)."""
    import oracle
    n_units = wl.n_points // unit
    order = np.random.default_rng(seed).permutation(n_units)
    if len(include):     # units that must be in the sample (e.g. unit 0, the dense end of config 3's ramp), after the pilot pair
        inc = np.asarray(include, dtype=order.dtype)
        rest = order[~np.isin(order, inc)]
        order = np.concatenate((rest[:2], inc, rest[2:]))
    ar = np.arange(unit, dtype=np.int64)

    def run(units):
        us = np.sort(units)
        t0 = time.perf_counter()
        kap = np.empty(us.size * unit)
        ne = 0
        for n, u in enumerate(us):           # unit by unit: each call sees only the lines that can reach its unit
            js = u * unit + ar
            sl = _reach(wl, int(js[0]), int(js[-1]))
            E = None if wl.E_low is None else wl.E_low[sl]
            kap[n * unit:(n + 1) * unit] = oracle.opacity_points(wl.nu0[sl], wl.S[sl], wl.gamma0[sl], T, P, wl.nu_min, wl.nu_max,
                                                                 wl.dnu, wl.cutoff, js, mass_amu=wl.mass_amu, E_low=E,
                                                                 q_ratio=q_ratio)
        ktab = oracle.kdist(kap, unit, wl.n_g) if with_kdist else None
        dt = time.perf_counter() - t0
        for u in us:
            nu = wl.nu_min + (u * unit + ar) * wl.dnu
            ne += int(np.sum(np.searchsorted(wl.nu0, nu + wl.cutoff, "right") - np.searchsorted(wl.nu0, nu - wl.cutoff, "left")))
        return dt, ne, us, kap, ktab

    dt, ne, us, kap, ktab = run(order[:2])
    nu_ = int(min(n_units, max(2, min_units, 2 + len(include), round(2 * target_s / max(dt, 1e-3)))))
    if max_units:
        nu_ = min(nu_, max_units)
    if nu_ > 2:
        dt, ne, us, kap, ktab = run(order[:nu_])
    return {"evals_per_s": ne / dt, "seconds": dt, "evals": ne, "units": us, "unit": unit, "kappa": kap, "ktab": ktab,
            "cores": host_cores(),
            "sample": f"{us.size} seeded whole units of {unit} consecutive grid points ({us.size * unit} points, {ne} "
                      f"line-point evals, {dt:.1f} s) of the {n_units}-unit grid" + (", with their k-distribution rows" if with_kdist else "")}


def parity_of(got, ref, bar):
    """max relative error where the oracle value >= 1e-12 x the largest oracle value of the compared set (A11)."""
    mask = ref >= 1e-12 * ref.max()
    if not np.all(np.isfinite(got)):
        return float("inf")
    err = float(np.abs(got[mask] / ref[mask] - 1.0).max()) if mask.any() else 0.0
    if np.any(got[ref == 0.0] != 0.0):
        return float("inf")
    return err


def unit_indices(units, unit):
    return (np.asarray(units)[:, None] * unit + np.arange(unit)[None, :]).ravel()


def roofline_fp64(census, ms_far, ms_near, fp64_peak, sm_mhz):
    """a3 = far + near kernel: FMA-equivalent TFLOP/s (1 FP64 instruction = 2 flop) of the algorithmic work against the
    live-measured DFMA peak, per kernel and as a whole, and against the nominal peak at the sampled SM clock."""
    far = sum(FP64_INST_PER_EVAL[k] * census[k] for k in FAR_REGIMES)
    near = sum(FP64_INST_PER_EVAL[k] * census[k] for k in NEAR_REGIMES)
    peak = 2.0 * fp64_peak / 1e12
    ach = 2.0 * (far + near) / ((ms_far + ms_near) * 1e-3) / 1e12
    out = {"achieved": ach, "peak": peak, "frac": ach / peak,
           "frac_far": 2.0 * far / (ms_far * 1e-3) / 1e12 / peak if ms_far > 0 else None,
           "frac_near": 2.0 * near / (ms_near * 1e-3) / 1e12 / peak if ms_near > 0 else None,
           "algorithmic_fp64_instructions": far + near}
    if sm_mhz:
        nominal = 2.0 * NOMINAL_FP64_LANES * sm_mhz * 1e6 / 1e12
        out["nominal_peak"] = nominal
        out["frac_vs_nominal"] = ach / nominal
    return out


def hbm_peak():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (6.65 TB/s, B200_PROFILING.md)"


def line_prep_hbm(n_lines, n_inputs, ms, f32=False):
    """a1 (line_prep_kernel) against the HBM roofline (an HBM-bound step; "Line"): per line it reads
    8 B of each input array given and writes the packed records (144 B; + 32 B in the FP32 variant); the line-range tables
    (12 B per 256 grid points) are left out."""
    hbm, src = hbm_peak()
    per_line = 8 * n_inputs + 144 + (32 if f32 else 0)
    gbs = per_line * n_lines / (ms * 1e-3) / 1e9 if ms > 0 else None
    return {"kernel": "line_prep_kernel (a1+a2)", "bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s",
            "frac": gbs / hbm if gbs else None, "algorithmic_bytes_per_line": per_line, "ms": ms, "peak_source": src}


def kdist_hbm(n_points, n_bins, n_g, ms, extra_bytes=0.0, kernel="kdist_kernel (a5+a6)"):
    """a5+a6 against the HBM roofline: 8 B/point read + 8 n_g B/bin written (+ extra_bytes for the Chebyshev variant)."""
    hbm, src = hbm_peak()
    b = 8.0 * n_points + 8.0 * n_bins * n_g + extra_bytes
    gbs = b / (ms * 1e-3) / 1e9 if ms > 0 else None
    return {"kernel": kernel, "bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm if gbs else None,
            "algorithmic_bytes": b, "ms": ms, "points_per_bin": n_points // n_bins, "peak_source": src}


def fp32_variant_leg(hk, wl, lines, T, P, flush, fp32_peak, steps=20):
    """The optional FP32 variant (north_star; BASELINE.json configs[3] names it) on the headline workload, timed like the
    headline: CUDA events around each step, L2 flushed between steps, per-stage times from the library's own events."""
    import torch
    N = wl.n_points
    ppb = int(round(wl.bin_width / wl.dnu))
    kap = torch.empty(N, dtype=torch.float64, device="cuda")
    ktab = torch.empty((N // ppb, wl.n_g), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(3):
        hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu, out=kap, precision=hk.HK_FP32)
    hk.hk_set_timing(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    stage = np.zeros(3)
    for i in range(steps):
        flush.zero_()
        ev[i][0].record(stream)
        hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu, out=kap, precision=hk.HK_FP32)
        hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g, out=ktab)
        ev[i][1].record(stream)
        stage += np.array(hk.hk_last_stage_ms())
    torch.cuda.synchronize()
    hk.hk_set_timing(False)
    stage /= steps
    ms = sum(a.elapsed_time(b) for a, b in ev) / steps
    census = hk.hk_regime_census(wl.nu0, wl.gamma0, T, P, wl.mass_amu, wl.nu_min, N, wl.dnu, wl.cutoff, precision=hk.HK_FP32)
    alg = sum(FP32_INST_PER_EVAL[k] * census[k] for k in FP32_INST_PER_EVAL)
    ach = 2.0 * alg / (stage[1] * 1e-3) / 1e12
    peak = 2.0 * fp32_peak / 1e12
    leg = {"workload": WORKLOAD + " [optional FP32 variant, bar 1e-4]", "steps": steps, "ms_per_step": ms,
           "stage_ms": {"line_prep": float(stage[0]), "voigt_far": float(stage[1]), "voigt_near": float(stage[2])},
           "roofline": {"kernel": "voigt_far_kernel<FP32>", "bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                        "frac": ach / peak, "ms": float(stage[1]), "regime_census": census,
                        "note": "FP32-pipe thread-instructions x2 of the float 1-/2-/3-point rules (4 / 6.5 / 10 per evaluation) "
                                "against the FFMA microbenchmark of this run; the near kernel stays FP64"},
           "line_prep_hbm": line_prep_hbm(wl.n_lines, 3, float(stage[0]), f32=True)}
    return leg, kap.cpu().numpy(), ktab.cpu().numpy()


def f_rows_leg(hk, wl, kappa, ktab, fp64_peak, n_c=20, n_m=1000, reps=20):
    """SURVEY.md 8(f1)/(f2) at the headline size (Fig. 5: "Resampling", "Transmission"): device times by CUDA
    events around `reps` back-to-back calls, each against its roofline; the outputs are returned for the parity check."""
    import torch
    N = wl.n_points
    ppb = int(round(wl.bin_width / wl.dnu))
    nb = N // ppb
    mcol = 10 ** np.linspace(-6, 4, n_m)
    dm = torch.as_tensor(mcol).cuda()

    def timed(fn):
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            out = fn()
        e1.record()
        torch.cuda.synchronize()
        return out, e0.elapsed_time(e1) / reps

    (coef, kt2), ms_c = timed(lambda: hk.hk_kdist_cheb(kappa, wl.dnu, wl.bin_width, n_c, n_g=wl.n_g))
    t_k, ms_tk = timed(lambda: hk.hk_transmission(ktab, dm))
    t_d, ms_td = timed(lambda: hk.hk_transmission_direct(kappa, wl.dnu, wl.bin_width, dm))
    inst = 19.0   # FP64-pipe instructions per exp term: product, clamp, exp_fast (16), accumulate
    peak = 2.0 * fp64_peak / 1e12

    def alu(terms, ms, kernel):
        a = 2.0 * inst * terms / (ms * 1e-3) / 1e12
        return {"kernel": kernel, "bound": "alu", "achieved": a, "peak": peak, "unit": "TFLOP/s", "frac": a / peak, "ms": ms,
                "exp_per_s": terms / (ms * 1e-3), "fp64_inst_per_term": inst}

    leg = {"workload": f"headline size: {nb} bins x {ppb} points, n_c = {n_c}, n_g = {wl.n_g}, {n_m} column masses",
           "timing": f"CUDA events around {reps} back-to-back calls",
           "kdist_cheb_with_ktable": kdist_hbm(N, nb, wl.n_g, ms_c, extra_bytes=8.0 * nb * n_c + 16.0 * N,
                                               kernel="kdist_kernel<ln> + cheb_project_kernel (f1; ln of the sorted bins "
                                                      "written and read once: + 16 B/point)"),
           "transmission_ktable": alu(float(nb) * wl.n_g * n_m, ms_tk, "transmission_kernel (f2, Lebesgue side)"),
           "transmission_direct": alu(float(N) * n_m, ms_td, "transmission_direct_kernel (f2, Riemann side)")}
    got = {"coef": coef.cpu().numpy(), "ktab": kt2.cpu().numpy(), "t_k": t_k.cpu().numpy(), "t_d": t_d.cpu().numpy(),
           "mcol": mcol, "n_c": n_c}
    return leg, got


def f_rows_parity(got, o, ppb):
    """The f-rows against the oracle on the cpu_baseline sample's bins.  The oracle works from ITS OWN kappa of those bins (no
    oracle input comes from the CUDA path), so each figure includes the <= 1e-6 relative difference of the two kappa: bars
    1e-5 on the coefficients of ln kappa(y) (absolute, relative to max(1, |C|)), 1e-6 on the transmission (absolute, T <= 1)."""
    import oracle
    us = o["units"]
    C = oracle.kdist_cheb(o["kappa"], ppb, got["n_c"])
    ce = float((np.abs(got["coef"][us] - C) / np.maximum(1.0, np.abs(C))).max())
    tk = float(np.abs(got["t_k"][us] - oracle.transmission_kdist(o["ktab"], got["mcol"])).max())
    td = float(np.abs(got["t_d"][us] - oracle.transmission_direct(o["kappa"], ppb, got["mcol"])).max())
    kt = parity_of(got["ktab"][us].ravel(), o["ktab"].ravel(), PARITY_BAR)
    ok = ce <= 1e-5 and tk <= 1e-6 and td <= 1e-6 and kt <= PARITY_BAR
    return {"bins": int(us.size), "cheb_coef_max_err": ce, "cheb_ktable_max_rel": kt, "transmission_ktable_max_abs": tk,
            "transmission_direct_max_abs": td, "bars": {"cheb_coef": 1e-5, "ktable": PARITY_BAR, "transmission": 1e-6}}, ok


# ---------------------------------------------------------------------------------------------------------------------------
# one config at BASELINE size: device times, census, roofline, parity and oracle time on seeded units
# ---------------------------------------------------------------------------------------------------------------------------
def config_leg(hk, k, fp64_peak, flush, oracle_s=6.0, sm_mhz=None, precision=None):
    import torch
    prec = hk.HK_FP64 if precision is None else precision
    bar = PARITY_BAR if prec == hk.HK_FP64 else PARITY_BAR32
    t_gen = time.perf_counter()
    wl = workloads.config(k)
    t_gen = time.perf_counter() - t_gen
    N = wl.n_points
    ppb = int(round(wl.bin_width / wl.dnu)) if wl.bin_width else None
    unit = 1000
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low)
    n_evals = hk.hk_count_evals(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff)
    pairs = [(T, P) for T in wl.T for P in wl.P_atm]
    qr = (lambda T: wl.q_ratio(T)) if wl.q_ratio else (lambda T: 1.0)
    ctx = hk.Context(lines, precision=prec)
    kap = torch.empty(N, dtype=torch.float64, device="cuda")
    ktab = torch.empty((N // ppb, wl.n_g), dtype=torch.float64, device="cuda") if ppb else None
    stream = torch.cuda.current_stream()
    big = wl.n_lines >= 10_000_000                 # records >> L2: nothing to flush, and one repetition is 0.3 s
    reps = 1 if (big or len(pairs) > 6) else 5

    def step(T, P):
        ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=qr(T), out=kap)
        if ppb:
            hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g, out=ktab)

    step(*pairs[0])                                # warm-up: allocates scratch, loads the kernels
    step(*pairs[-1])
    torch.cuda.synchronize()
    # parity sample: seeded pairs of the config's (T,P) list; oracle units on each (sized for ~oracle_s seconds in all)
    rng = np.random.default_rng(100 + k)
    if len(pairs) == 1:
        chk = [0]
    elif len(pairs) <= 6:
        chk = list(range(len(pairs)))
    else:
        chk = sorted({0, len(pairs) - 1} | set(int(i) for i in rng.choice(len(pairs), 4, replace=False)))
    hk.hk_set_timing(True)
    ms_op = ms_kd = 0.0
    stage = np.zeros(3)
    per_pair, got_kappa, got_ktab = [], {}, {}
    for ip, (T, P) in enumerate(pairs):
        best = None
        for _ in range(reps):
            if not big:
                flush.zero_()
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            e[0].record(stream)
            ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=qr(T), out=kap)
            e[1].record(stream)
            if ppb:
                hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g, out=ktab)
            e[2].record(stream)
            st = np.array(hk.hk_last_stage_ms())
            torch.cuda.synchronize()
            t = (e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2]), st)
            if best is None or t[0] + t[1] < best[0] + best[1]:
                best = t
        ms_op += best[0]
        ms_kd += best[1]
        stage += best[2]
        per_pair.append({"T_K": T, "P_atm": P, "opacity_ms": best[0], "far_ms": float(best[2][1]), "near_ms": float(best[2][2])})
        if ip in chk:
            got_kappa[ip] = kap.cpu().numpy()
            if ppb:
                got_ktab[ip] = ktab.cpu().numpy()
    hk.hk_set_timing(False)
    ctx.close()
    # census + roofline on the checked pairs (all pairs when there are at most six)
    cen_tot = {r: 0 for r in FP64_INST_PER_EVAL}
    far_ms = near_ms = 0.0
    for ip in chk:
        T, P = pairs[ip]
        c = hk.hk_regime_census(wl.nu0, wl.gamma0, T, P, wl.mass_amu, wl.nu_min, N, wl.dnu, wl.cutoff, precision=prec)
        for r in cen_tot:
            cen_tot[r] += c[r]
        far_ms += per_pair[ip]["far_ms"]
        near_ms += per_pair[ip]["near_ms"]
    roof = roofline_fp64(cen_tot, far_ms, near_ms, fp64_peak, sm_mhz) if prec == hk.HK_FP64 else None
    # oracle on seeded units of the checked pairs: parity of this run's kappa (and k-table rows), and the CPU time
    worst_k, worst_t, o_ev, o_s, n_pts, samples = 0.0, 0.0, 0, 0.0, 0, []
    for ip in chk:
        T, P = pairs[ip]
        o = oracle_units(wl, T, P, oracle_s / len(chk), unit, seed=1000 * k + ip, q_ratio=qr(T),
                         with_kdist=(ppb == unit), max_units=64, include=(0,) if k == 3 else (), min_units=10 if k == 3 else 2)
        js = unit_indices(o["units"], unit)
        worst_k = max(worst_k, parity_of(got_kappa[ip][js], o["kappa"], bar))
        if ppb == unit:
            gk, rk = got_ktab[ip][o["units"]].ravel(), o["ktab"].ravel()
            worst_t = max(worst_t, parity_of(gk, rk, bar))
        o_ev += o["evals"]
        o_s += o["seconds"]
        n_pts += js.size
        samples.append(o["sample"])
    n_tot = n_evals * len(pairs)
    leg = {
        "workload": f"BASELINE.json configs[{k}] at full size", "n_lines": wl.n_lines, "n_points": N, "pairs": len(pairs),
        "precision": "fp32" if prec == hk.HK_FP32 else "fp64",
        "line_point_evals": n_tot, "opacity_ms": ms_op, "kdist_ms": ms_kd if ppb else None,
        "s_per_opacity_function": ms_op / len(pairs) * 1e-3,
        "evals_per_s": n_tot / ((ms_op + ms_kd) * 1e-3),
        "evals_per_s_opacity_only": n_tot / (ms_op * 1e-3),
        "stage_ms": {"line_prep": float(stage[0]), "voigt_far": float(stage[1]), "voigt_near": float(stage[2])},
        "timing": f"CUDA events on the launching stream, best of {reps} per (T,P) pair, "
                  + ("line records (14 GB) >> L2" if big else "L2 flushed before each repetition"),
        "regime_census": cen_tot, "census_pairs": len(chk),
        "roofline": roof,
        "parity": {"kappa_max_rel": worst_k, "ktable_max_rel": worst_t if ppb == unit else None, "points": n_pts,
                   "pairs_checked": len(chk), "bar": bar},
        "cpu_baseline": {"value": o_ev / o_s, "unit": UNIT, "cores": host_cores(), "kind": "oracle",
                         "sample": samples[0] + (f" (+ {len(samples) - 1} more (T,P) pairs, same size)" if len(samples) > 1 else ""),
                         "seconds_full_config_extrapolated_by_n_evals": n_tot / (o_ev / o_s)},
        "host_generation_s": t_gen,
        "line_prep_hbm": line_prep_hbm(wl.n_lines, 3 + (wl.E_low is not None), float(stage[0]) / len(pairs), f32=prec == hk.HK_FP32),
        "kdist_hbm": kdist_hbm(N, N // ppb, wl.n_g, ms_kd / len(pairs)) if ppb else None,
    }
    if k == 3 and roof is not None:
        # wasted re-reads of the dense far shape (one-warp CTAs, each streaming its own +-cutoff window of records): DRAM bytes of
        # one far-kernel launch at 1e7 lines from the committed ncu capture against the 96 B/line the ring copies once per line
        t = _ncu_dram("r02_config3_1e7_voigt_far_kernel_ncu_full.txt")
        roof["traffic"] = t
        roof["traffic_algorithmic"] = 96.0e7 + 8.0 * N
        roof["traffic_ratio"] = t / roof["traffic_algorithmic"] if t else None
        roof["traffic_source"] = ("profiles/r02_config3_1e7_voigt_far_kernel_ncu_full.txt: one launch at 1e7 lines (the far kernel "
                                  "is unchanged since); algorithmic = 96 B of ring records per line + the kappa store; 662 GB/s, "
                                  "10 % of the HBM rate: not the limiter")
    if len(pairs) > 1 and len(pairs) <= 6:
        leg["per_pair"] = per_pair
    ok = worst_k <= bar and (worst_t <= bar)
    return leg, ok


def run_config(args):
    import torch
    import paper_1503_03806_b200 as hk
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --config: no CUDA device — the hot path has no CPU fallback")
    hk.load_library()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    prec = hk.HK_FP32 if args.precision == "fp32" else hk.HK_FP64
    leg, ok = config_leg(hk, args.config, hk.hk_fp64_peak(), flush, oracle_s=args.oracle_seconds, sm_mhz=None, precision=prec)
    print(json.dumps(leg))
    if not ok:
        raise SystemExit(f"bench.py --config {args.config}: parity above the bar")


def run_reference(args):
    """--impl reference: the oracle on the host cores (this tier's reference arm).  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    wl = workloads.config(1)
    T, P = wl.T[0], wl.P_atm[0]
    import oracle
    oracle.build()
    per_step_s = max(2.0, min(20.0, 90.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_units(wl, T, P, per_step_s, 1000, seed=1, with_kdist=True)
    tot_e, tot_t, desc, cores = 0, 0.0, "", 1
    for _ in range(args.steps):
        o = oracle_units(wl, T, P, per_step_s, 1000, seed=1, with_kdist=True)
        tot_e += o["evals"]
        tot_t += o["seconds"]
        desc, cores = o["sample"], o["cores"]
    v = tot_e / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": "each step: " + desc},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": "each step: " + desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1503_03806_b200 as hk

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the hot path has no CPU fallback (use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    hk.load_library()
    wl = workloads.config(1)
    T, P = tp_table(wl, world)[rank]
    N = wl.n_points
    ppb = int(round(wl.bin_width / wl.dnu))
    n_evals = hk.hk_count_evals(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kappa = torch.empty(N, dtype=torch.float64, device="cuda")
    ktab = torch.empty((N // ppb, wl.n_g), dtype=torch.float64, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    stream = torch.cuda.current_stream()

    prec = hk.HK_FP32 if args.precision == "fp32" else hk.HK_FP64
    bar = PARITY_BAR32 if prec == hk.HK_FP32 else PARITY_BAR

    def step():
        hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu, out=kappa, precision=prec)
        hk.hk_kdist(kappa, wl.dnu, wl.bin_width, wl.n_g, out=ktab)

    fp64_peak = hk.hk_fp64_peak()                                        # DFMA thread-instructions/s, measured live
    fp32_peak = hk.hk_fp32_peak()                                        # FFMA, likewise
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    # ---- timed region: K steps, device time by CUDA events around each step, L2 flushed between steps ----------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    hk.hk_set_timing(True)                                               # per-stage events inside hk_opacity (same stream)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    stage = np.zeros(3)
    barrier()
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.zero_()
        ev[i][0].record(stream)
        hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu, out=kappa, precision=prec)
        ev[i][1].record(stream)
        hk.hk_kdist(kappa, wl.dnu, wl.bin_width, wl.n_g, out=ktab)
        ev[i][2].record(stream)
        stage += np.array(hk.hk_last_stage_ms())
    barrier()
    t_wall = time.perf_counter() - t_wall0
    hk.hk_set_timing(False)
    ms_opacity = sum(e[0].elapsed_time(e[1]) for e in ev)
    ms_kdist = sum(e[1].elapsed_time(e[2]) for e in ev)
    ms_total = ms_opacity + ms_kdist
    stage /= args.steps
    got_kappa = kappa.cpu().numpy() if rank == 0 else None              # this run's result, for the parity check below
    got_ktab = ktab.cpu().numpy() if rank == 0 else None
    # ---- e2e: host buffers in, host buffers out, through the public API -----------------------------------------------
    pin = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).pin_memory()
    h_nu0, h_S, h_g0 = pin(wl.nu0), pin(wl.S), pin(wl.gamma0)
    h_kappa = torch.empty(N, dtype=torch.float64, pin_memory=True)
    h_ktab = torch.empty((N // ppb, wl.n_g), dtype=torch.float64, pin_memory=True)
    for _ in range(2):
        hk.hk_opacity_host(h_nu0, h_S, h_g0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu,
                           bin_width=wl.bin_width, n_g=wl.n_g, kappa_out=h_kappa, k_out=h_ktab, precision=prec)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        hk.hk_opacity_host(h_nu0, h_S, h_g0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu,
                           bin_width=wl.bin_width, n_g=wl.n_g, kappa_out=h_kappa, k_out=h_ktab, precision=prec)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    clocks = None
    h2d = 3 * 8 * wl.n_lines
    d2h = 8 * N + 8 * (N // ppb) * wl.n_g

    # ---- max over ranks ------------------------------------------------------------------------------------------------
    red = torch.tensor([ms_total, ms_opacity, ms_kdist, e2e_s * 1e3, stage[1] + stage[2], stage[1], stage[2]], dtype=torch.float64,
                       device="cuda")
    if world > 1:
        dist.all_reduce(red, op=dist.ReduceOp.MAX)
    ms_total, ms_opacity, ms_kdist, e2e_ms, ms_voigt, ms_far, ms_near = [float(v) for v in red.cpu()]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    K = args.steps
    value = world * n_evals * K / (ms_total * 1e-3)
    run_legs = world == 1 and not args.no_configs and prec == hk.HK_FP64
    ok = True
    legs = {}
    fp32_leg = frows = None
    if run_legs:   # the optional FP32 variant and the 8(f) rows on the headline workload (a few tens of ms of GPU time)
        fp32_leg, got32_kappa, got32_ktab = fp32_variant_leg(hk, wl, lines, T, P, flush, fp32_peak)
        frows, frows_got = f_rows_leg(hk, wl, kappa, ktab, fp64_peak)
    if run_legs:   # configs 0, 2, 3, 4 at BASELINE size; the clock sampler keeps running (config 4 is 2 s of continuous load)
        del kappa, ktab, lines
        torch.cuda.empty_cache()
        for k in (0, 2, 3, 4):
            leg, lok = config_leg(hk, k, fp64_peak, flush, oracle_s=args.oracle_seconds, sm_mhz=None)
            legs[str(k)] = leg
            ok = ok and lok
            hk.hk_trim()
            torch.cuda.empty_cache()
    clocks = sampler.stop()
    sm_mhz = clocks.get("sm_mhz") if clocks else None
    for leg in legs.values():      # nominal-peak fraction at the clock sampled under load
        r = leg.get("roofline")
        if r and sm_mhz:
            r["nominal_peak"] = 2.0 * NOMINAL_FP64_LANES * sm_mhz * 1e6 / 1e12
            r["frac_vs_nominal"] = r["achieved"] / r["nominal_peak"]
    # roofline of the dominant kernels (a3+a4): ALU-bound on the FP64 pipe
    census = hk.hk_regime_census(wl.nu0, wl.gamma0, T, P, wl.mass_amu, wl.nu_min, N, wl.dnu, wl.cutoff, precision=prec)
    if prec == hk.HK_FP32:
        # the FP32 variant's dominant kernel is the far kernel alone (1-/2-/3-point rules in float, FP32 pipe)
        alg_inst = sum(FP32_INST_PER_EVAL[k] * census[k] for k in FP32_INST_PER_EVAL)
        achieved = 2.0 * alg_inst / (ms_far * 1e-3) / 1e12
        peak = 2.0 * fp32_peak / 1e12
        roof = {"kernel": "voigt_far_kernel<FP32> (a3 far wings + a4)", "bound": "alu", "achieved": achieved, "peak": peak,
                "unit": "TFLOP/s", "frac": achieved / peak, "ms": ms_far,
                "note": "FP32-pipe thread-instructions x2 of the 1-/2-/3-point rules (regime census x per-eval figure); peak = "
                        "hk_fp32_peak FFMA microbenchmark measured live in this run; the near kernel (6-point rule, series) "
                        "stays FP64 and is reported in stage_ms"}
    else:
        r = roofline_fp64(census, ms_far, ms_near, fp64_peak, sm_mhz)
        roof = {"kernel": "voigt_far_kernel + voigt_near_kernel (a3+a4)", "bound": "alu", "achieved": r["achieved"],
                "peak": r["peak"], "unit": "TFLOP/s", "frac": r["frac"], "frac_far": r["frac_far"], "frac_near": r["frac_near"],
                "frac_vs_nominal": r.get("frac_vs_nominal"), "nominal_peak": r.get("nominal_peak"), "ms": ms_voigt,
                "note": "FP64-pipe thread-instructions x2; algorithmic instructions = regime census x per-evaluation figure "
                        "(DESIGN.md §4: 5 / 7 / 11 / 22 for the 1-/2-/3-/6-point rules, 83 for the series, counted from the "
                        "kernel's SASS); peak = hk_fp64_peak DFMA microbenchmark measured live in this run; nominal_peak = "
                        "148 SMs x 64 lanes x the SM clock sampled under load x 2"}
    roof.update({"traffic": NCU_DRAM[args.precision]["bytes"], "traffic_source": NCU_DRAM[args.precision]["source"],
                 "regime_census": census, "fp64_peak_tflops": 2.0 * fp64_peak / 1e12, "fp32_peak_tflops": 2.0 * fp32_peak / 1e12,
                 "fp64_inst_per_eval": FP64_INST_PER_EVAL})

    # HBM-bound steps: a5+a6 reads kappa once and writes the k-table; a4 is the kappa store inside the far kernel
    hbm, hbm_src = hbm_peak()
    kdist_bytes = 8.0 * N + 8.0 * (N // ppb) * wl.n_g
    kdist_gbs = kdist_bytes / (ms_kdist / K * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == hk.HK_FP32 else "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD + (" [optional FP32 variant, bar 1e-4]" if prec == hk.HK_FP32 else ""), "n_lines": wl.n_lines, "n_points": N, "line_point_evals": n_evals,
                   "parallelism": f"tp-pairs x{world} (no collective)", "api": "hk_opacity + hk_kdist (C ABI, one-shot form)",
                   "l2": "flushed between steps by a 512 MiB memset outside the per-step CUDA events",
                   "T_K": T, "P_atm": P},
        "s_per_opacity_function": ms_opacity / K * 1e-3, "s_per_kdist": ms_kdist / K * 1e-3,
        "stage_ms": {"line_prep": stage[0], "voigt_far": ms_far, "voigt_near": ms_near, "voigt_accumulate_store": ms_voigt,
                     "kdist": ms_kdist / K},
        "wall_s_timed_region": t_wall,
        "e2e": {"value": world * n_evals * K / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / K},
        "gpu_launches": 4 * K,   # line_prep, voigt_far, voigt_near, kdist
        "roofline": roof,
        "kdist_hbm": {"kernel": "kdist_kernel (a5+a6)", "bound": "hbm", "achieved": kdist_gbs, "peak": hbm, "unit": "GB/s",
                      "frac": kdist_gbs / hbm, "algorithmic_bytes": kdist_bytes, "peak_source": hbm_src,
                      "note": "8 B/point read + 8 n_g B/bin written; the kernel is bound by the bitonic network's "
                              "compare-exchange count, not by HBM (profiles/)"},
        "line_prep_hbm": line_prep_hbm(wl.n_lines, 3, float(stage[0]), f32=prec == hk.HK_FP32),
        "clocks": clocks,
    }
    if world == 1:
        # the oracle, as it stands, on seeded whole bins: the CPU baseline AND the parity check of this run's kappa / k-table
        o = oracle_units(wl, T, P, args.oracle_seconds_headline, ppb, seed=1, with_kdist=True)
        line["cpu_baseline"] = {"value": o["evals_per_s"], "unit": UNIT, "cores": o["cores"], "kind": "oracle", "sample": o["sample"],
                                "seconds_full_config_extrapolated_by_n_evals": n_evals / o["evals_per_s"]}
        js = unit_indices(o["units"], ppb)
        pk = parity_of(got_kappa[js], o["kappa"], bar)
        pt = parity_of(got_ktab[o["units"]].ravel(), o["ktab"].ravel(), bar)
        line["parity"] = {"kappa_max_rel": pk, "ktable_max_rel": pt, "points": int(js.size), "bins": int(o["units"].size), "bar": bar,
                          "note": "GPU kappa and k-table of this run's last timed step against the oracle on the cpu_baseline "
                                  "sample; mask: oracle value >= 1e-12 x the oracle's max over the compared set"}
        ok = ok and pk <= bar and pt <= bar
        # the host-buffer call's own outputs (last e2e step; the ranged path of hk_opacity_host), against the same oracle sample
        e_k, e_t = h_kappa.numpy(), h_ktab.numpy()
        pke = parity_of(e_k[js], o["kappa"], bar)
        pte = parity_of(e_t[o["units"]].ravel(), o["ktab"].ravel(), bar)
        same = bool(np.array_equal(e_k, got_kappa) and np.array_equal(e_t, got_ktab))
        line["e2e"]["parity"] = {"kappa_max_rel": pke, "ktable_max_rel": pte, "bitwise_equal_to_device_form": same, "bar": bar}
        ok = ok and pke <= bar and pte <= bar and same
        if fp32_leg is not None:
            p32k = parity_of(got32_kappa[js], o["kappa"], PARITY_BAR32)
            p32t = parity_of(got32_ktab[o["units"]].ravel(), o["ktab"].ravel(), PARITY_BAR32)
            fp32_leg["parity"] = {"kappa_max_rel": p32k, "ktable_max_rel": p32t, "points": int(js.size), "bar": PARITY_BAR32}
            line["fp32_variant"] = fp32_leg
            fpar, fok = f_rows_parity(frows_got, o, ppb)
            frows["parity"] = fpar
            line["f_rows"] = frows
            ok = ok and p32k <= PARITY_BAR32 and p32t <= PARITY_BAR32 and fok
        if legs:
            line["configs"] = legs
    line["paper_context"] = "~1 s per opacity function of ~1e5 lines on a Tesla K20 (PAPER.md:9, 267); other hardware, not a target"
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    if not ok:
        raise SystemExit("bench.py: parity against the oracle above the bar (see the `parity` keys of the line)")


def run_grid_shard(args):
    """--shard grid (with --gpus N under torchrun): ONE opacity function + k-distribution of config 3 split along the
    wavenumber grid by shard.shard_grid — contiguous, bin-aligned ranges balanced by line-point evaluations, each rank with the
    slice of the line list whose windows reach its range (a read-only halo, no collective on the data path).
    Strong scaling: the total work is fixed.  NCCL carries the barrier and the max-over-ranks of the device time only."""
    import torch
    import torch.distributed as dist
    import paper_1503_03806_b200 as hk
    from paper_1503_03806_b200 import shard
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --shard grid: no CUDA device")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    wl = workloads.config(3, n_lines=args.shard_lines)
    T, P = wl.T[0], wl.P_atm[0]
    N = wl.n_points
    ppb = int(round(wl.bin_width / wl.dnu))
    sh = shard.shard_grid(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff, ppb, world)[rank]
    sl = slice(sh.line_lo, sh.line_hi)
    lines = hk.Lines.from_numpy(wl.nu0[sl], wl.S[sl], wl.gamma0[sl])
    n_own = sh.j_hi - sh.j_lo
    kap = torch.empty(n_own, dtype=torch.float64, device="cuda")
    ktab = torch.empty((n_own // ppb, wl.n_g), dtype=torch.float64, device="cuda")
    ctx = hk.Context(lines)
    stream = torch.cuda.current_stream()

    def step():
        ctx.opacity(T, P, sh.nu_min, sh.nu_max, wl.dnu, wl.cutoff, out=kap)
        hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g, out=ktab)

    for _ in range(max(args.warmup, 3)):
        step()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for i in range(args.steps):
        ev[i][0].record(stream)
        step()
        ev[i][1].record(stream)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    red = torch.tensor([sum(a.elapsed_time(b) for a, b in ev)], dtype=torch.float64, device="cuda")
    tot = torch.tensor([float(sh.evals)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(red, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    ctx.close()
    if rank == 0:
        ms = float(red.item())
        print(json.dumps({
            "metric": METRIC, "value": float(tot.item()) * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[3] with {wl.n_lines} lines: one opacity function + k-distribution, grid "
                                   f"split into {world} bin-aligned ranges balanced by line-point evaluations (shard.shard_grid)",
                       "parallelism": f"grid-range x{world} (no collective)", "line_point_evals": int(tot.item()),
                       "l2": "line records (144 B/line) >> L2: no flush"},
            "gpu_launches": 4 * args.steps}))
    if world > 1:
        dist.destroy_process_group()


def run_stage_times(args):
    """--stage-times: per-stage device times (hk_set_timing) of hk_opacity on configs 1, 2 (its highest pressure) and 3 cut to
    1e7 lines, in both precisions — the figures profiles/ and DESIGN.md quote beside the bench line.  One GPU; not a bench line."""
    import torch
    import paper_1503_03806_b200 as hk
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --stage-times: no CUDA device")
    for cfg, n_lines, reps in ((1, None, 10), (2, None, 5), (3, 10_000_000, 3)):
        wl = workloads.config(cfg) if n_lines is None else workloads.config(cfg, n_lines=n_lines)
        T, P = wl.T[0], (wl.P_atm[-1] if cfg == 2 else wl.P_atm[0])
        lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
        ne = hk.hk_count_evals(wl.nu0, wl.nu_min, wl.n_points, wl.dnu, wl.cutoff)
        for prec, name in ((hk.HK_FP64, "fp64"), (hk.HK_FP32, "fp32")):
            ctx = hk.Context(lines, precision=prec)
            out = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
            hk.hk_set_timing(True)
            st = np.zeros(3)
            for _ in range(reps):
                ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=out)
                st += np.array(hk.hk_last_stage_ms())
            hk.hk_set_timing(False)
            st /= reps
            ctx.close()
            print(json.dumps({"config": cfg, "n_lines": wl.n_lines, "T_K": T, "P_atm": P, "precision": name,
                              "line_prep_ms": st[0], "voigt_far_ms": st[1], "voigt_near_ms": st[2],
                              "opacity_ms": float(st.sum()), "evals_per_s": ne / (st.sum() * 1e-3)}), flush=True)


def run_f_rows(args):
    """--f-rows: device times of the SURVEY §8(f) rows at config 1's size (3000 bins x 1000 points, 20 Chebyshev coefficients,
    1000 column masses): CUDA events around `reps` back-to-back calls.  One GPU; not a bench line."""
    import torch
    import paper_1503_03806_b200 as hk
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --f-rows: no CUDA device")
    wl = workloads.config(1)
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    kap = hk.hk_opacity(lines, wl.T[0], wl.P_atm[0], wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
    dm = torch.as_tensor(10 ** np.linspace(-6, 4, 1000)).cuda()

    def timed(fn, reps=20):
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            out = fn()
        e1.record()
        torch.cuda.synchronize()
        return out, e0.elapsed_time(e1) / reps

    ktab, ms_k = timed(lambda: hk.hk_kdist(kap, wl.dnu, wl.bin_width, wl.n_g))
    _, ms_c = timed(lambda: hk.hk_kdist_cheb(kap, wl.dnu, wl.bin_width, 20, n_g=wl.n_g))
    _, ms_tk = timed(lambda: hk.hk_transmission(ktab, dm))
    _, ms_td = timed(lambda: hk.hk_transmission_direct(kap, wl.dnu, wl.bin_width, dm))
    print(json.dumps({"workload": "config 1 size: 3000 bins x 1000 points, n_c = 20, n_g = 20, 1000 column masses",
                      "kdist_ms": ms_k, "kdist_cheb_with_ktable_ms": ms_c, "transmission_ktable_ms": ms_tk,
                      "transmission_direct_ms": ms_td, "direct_exp_per_s": 3.0e9 / (ms_td * 1e-3),
                      "timing": "CUDA events around 20 back-to-back calls (host launch overhead included)"}))


def run_shift_sweep(args):
    """--shift-sweep: config 4's 200 (T,P) pairs through hk.Context with and without a pressure-shift field (eq. 21,
    PAPER.md:189): what the shifted copy, its order check / re-ordering and the per-call scratch cost per opacity function.
    delta ~ U[-0.02, 0.02] cm^-1/atm (seeded; HITRAN's air-induced shifts are of this size).  One GPU; not a bench line."""
    import torch
    import paper_1503_03806_b200 as hk
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --shift-sweep: no CUDA device")
    wl = workloads.config(4)
    delta = np.random.default_rng(44).uniform(-0.02, 0.02, wl.n_lines)
    N = wl.n_points
    kap = torch.empty(N, dtype=torch.float64, device="cuda")
    out = {}
    for name, d in (("no_shift", None), ("with_shift", delta)):
        lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0, E_low=wl.E_low, delta=d)
        ctx = hk.Context(lines)
        ctx.opacity(wl.T[0], wl.P_atm[0], wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=wl.q_ratio(wl.T[0]), out=kap)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for T in wl.T:
            for P in wl.P_atm:
                ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, q_ratio=wl.q_ratio(T), out=kap)
        e1.record()
        torch.cuda.synchronize()
        out[name] = {"device_ms_200_pairs": e0.elapsed_time(e1), "wall_ms_200_pairs": 1e3 * (time.perf_counter() - t0)}
        ctx.close()
    out["overhead_frac_device"] = out["with_shift"]["device_ms_200_pairs"] / out["no_shift"]["device_ms_200_pairs"] - 1.0
    out["overhead_frac_wall"] = out["with_shift"]["wall_ms_200_pairs"] / out["no_shift"]["wall_ms_200_pairs"] - 1.0
    out["workload"] = "config 4 (1e6 lines, 200 (T,P) pairs, opacity functions only), delta ~ U[-0.02, 0.02] cm^-1/atm, seed 44"
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--precision", choices=["fp64", "fp32"], default="fp64",
                    help="fp64 (BASELINE.json config 1, the default) or the optional FP32 variant (bar 1e-4)")
    ap.add_argument("--config", type=int, choices=[0, 1, 2, 3, 4], default=None,
                    help="print the per-config leg of config k alone (BASELINE size) and exit")
    ap.add_argument("--no-configs", action="store_true", help="default line without the `configs` key (configs 0, 2, 3, 4)")
    ap.add_argument("--oracle-seconds", type=float, default=6.0, help="CPU seconds of oracle per config leg (parity + cpu_baseline)")
    ap.add_argument("--oracle-seconds-headline", type=float, default=15.0, help="likewise for the headline config 1")
    ap.add_argument("--stage-times", action="store_true",
                    help="print per-stage device times of configs 1, 2, 3 (1e7 lines) in both precisions and exit")
    ap.add_argument("--f-rows", action="store_true",
                    help="print device times of the SURVEY 8(f) rows (Chebyshev resampling, transmission) at config 1's size and exit")
    ap.add_argument("--shard", choices=["pairs", "grid"], default="pairs",
                    help="N > 1: 'pairs' (default) gives rank r the r-th (T,P) pair of config 1, weak scaling; 'grid' splits ONE "
                         "opacity function of config 3 along the grid (shard.shard_grid), strong scaling")
    ap.add_argument("--shard-lines", type=int, default=100_000_000, help="--shard grid: lines of config 3 (default: all 1e8)")
    ap.add_argument("--shift-sweep", action="store_true",
                    help="time config 4's T-P sweep with and without a pressure-shift field (eq. 21) and exit")
    args = ap.parse_args()
    if args.shift_sweep:
        run_shift_sweep(args)
    elif args.f_rows:
        run_f_rows(args)
    elif args.stage_times:
        run_stage_times(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.config is not None:
        run_config(args)
    elif args.shard == "grid":
        run_grid_shard(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
