#!/usr/bin/env python
"""bench.py — the hot path of HELIOS-K on BASELINE.json config 1.

One "step" = one whole opacity function plus its k-distribution through the C ABI:
    hk_opacity (a1 line prep, a2 tile plan, a3 Voigt accumulation, a4 kappa store)  +  hk_kdist (a5 per-bin sort, a6 resample)
on the seeded synthetic 1e5-line workload (workloads.config(1): 3e6 grid points, cutoff 100 cm^-1, 3000 bins x 1000 points,
20 Gauss-Legendre g-points), FP64.

    python bench.py [--gpus N] [--steps K] [--warmup W]                  our arm (CUDA, sm_100a)
    python bench.py --impl reference [...]                                the oracle, as it stands, on the host cores

N > 1 (torchrun, one rank per GPU): the path shards with NO collective — rank r computes the opacity function of the r-th
(T, P) pair of a small T-P table over the same line list ("repeat this calculation for multiple combinations of
temperature and pressure"); rank 0 keeps config 1's (1500 K, 1 atm).  Per-GPU work is fixed: weak scaling.  NCCL is used only
for the barrier and the max-over-ranks of the device time.

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

# FP64-pipe thread-instructions the method needs per line-point evaluation, by regime (counted from
# the formulas of hk_voigt.cuh with the Newton reciprocal; these are the algorithmic figures, not the executed SASS).
# gh1 = the 1-point rule with the shifted denominator (from r^2 >= max(3600, 4100 y)), gh2 the shell between 3200 and that.
FP64_INST_PER_EVAL = {"gh1": 5.0, "gh2": 7.0, "gh3": 11.0, "gh6": 22.0, "series": 150.0}
# --precision fp32: FP32-pipe thread-instructions per evaluation of the two rules the far kernel runs in float, two points per
# reciprocal (hk_voigt.cuh gh1_acc2f / gh2_acc2f: 8 and 13 per pair, + 1 MUFU.RCP per pair)
FP32_INST_PER_EVAL = {"gh1": 4.0, "gh2": 6.5}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the roofline kernel(s), from the committed `ncu --set full` captures
# of this command (profiles/r01c_voigt_{far,near,far32}_kernel_ncu_full.txt): far 9.76 MB + near 36.90 MB read, ~0 written
# (kappa, 24 MB, stays in the 126 MB L2 between the two kernels); FP32 far kernel 6.52 MB.  Not memory-bound: context only.
NCU_DRAM_BYTES = {"fp64": 9.719e6 + 36.894e6 + 0.020e6, "fp32": 6.518e6}


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
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

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
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if r[5 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(wl, T, P, target_s, seed=1):
    """Times the oracle, as it stands, on whole seeded bins of the workload (kappa of every point of the bin + the bin's
    k-distribution).  A 4-bin pilot sizes the sample for about `target_s` seconds.  Returns (evals/s, description, cores)."""
    import oracle
    ppb = int(round(wl.bin_width / wl.dnu))
    n_bins = wl.n_points // ppb
    rng = np.random.default_rng(seed)
    order = rng.permutation(n_bins)

    def run(bins):
        js = (np.sort(bins)[:, None] * ppb + np.arange(ppb)[None, :]).ravel()
        t0 = time.perf_counter()
        kap = oracle.opacity_points(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, js,
                                    mass_amu=wl.mass_amu)
        oracle.kdist(kap, ppb, wl.n_g)
        dt = time.perf_counter() - t0
        nu = wl.nu_min + js * wl.dnu
        ne = int(np.sum(np.searchsorted(wl.nu0, nu + wl.cutoff, "right") - np.searchsorted(wl.nu0, nu - wl.cutoff, "left")))
        return dt, ne

    dt, ne = run(order[:4])
    nb = int(min(n_bins, max(4, round(4 * target_s / max(dt, 1e-3)))))
    dt, ne = run(order[:nb])
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    return ne / dt, dt, ne, f"{nb} seeded whole bins ({nb * ppb} grid points, {ne} line-point evals, {dt:.1f} s) of the {n_bins}-bin workload", cores


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
        oracle_sample(wl, T, P, per_step_s)
    tot_e, tot_t, desc, cores = 0, 0.0, "", 1
    for _ in range(args.steps):
        _, dt, ne, desc, cores = oracle_sample(wl, T, P, per_step_s)
        tot_e += ne
        tot_t += dt
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
    clocks = sampler.stop() if rank == 0 else None
    h2d = 3 * 8 * wl.n_lines
    d2h = 8 * N + 8 * (N // ppb) * wl.n_g

    # ---- max over ranks ------------------------------------------------------------------------------------------------
    red = torch.tensor([ms_total, ms_opacity, ms_kdist, e2e_s * 1e3, stage[1] + stage[2], stage[1]], dtype=torch.float64,
                       device="cuda")
    if world > 1:
        dist.all_reduce(red, op=dist.ReduceOp.MAX)
    ms_total, ms_opacity, ms_kdist, e2e_ms, ms_voigt, ms_far = [float(v) for v in red.cpu()]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    K = args.steps
    value = world * n_evals * K / (ms_total * 1e-3)
    # roofline of the dominant kernel (voigt_kernel, a3+a4): ALU-bound on the FP64 pipe
    census = hk.hk_regime_census(wl.nu0, wl.gamma0, T, P, wl.mass_amu, wl.nu_min, N, wl.dnu, wl.cutoff, precision=prec)
    if prec == hk.HK_FP32:
        # the FP32 variant's dominant kernel is the far kernel alone (1-/2-point rules in float, FP32 pipe)
        alg_inst = sum(FP32_INST_PER_EVAL[k] * census[k] for k in FP32_INST_PER_EVAL)
        achieved = 2.0 * alg_inst / (ms_far * 1e-3) / 1e12
        peak = 2.0 * fp32_peak / 1e12
        roof_kernel, roof_ms = "voigt_far_kernel<FP32> (a3 far wings + a4)", ms_far
        roof_note = ("FP32-pipe thread-instructions x2 of the 1-/2-point rules (regime census x per-eval figure, two points per "
                     "MUFU.RCP); peak = hk_fp32_peak FFMA microbenchmark measured live in this run; the near kernel "
                     "(3-/6-point rules, series) stays FP64 and is reported in stage_ms")
    else:
        alg_inst = sum(FP64_INST_PER_EVAL[k] * census[k] for k in FP64_INST_PER_EVAL)
        achieved = 2.0 * alg_inst / (ms_voigt * 1e-3) / 1e12            # FMA-equivalent TFLOP/s (1 FP64 instruction = 2 flop)
        peak = 2.0 * fp64_peak / 1e12
        roof_kernel, roof_ms = "voigt_far_kernel + voigt_near_kernel (a3+a4)", ms_voigt
        roof_note = ("FP64-pipe thread-instructions x2; algorithmic instructions = regime census x per-eval figure "
                     "(DESIGN.md); peak = hk_fp64_peak DFMA microbenchmark measured live in this run")
    cpu_v, cpu_dt, cpu_ne, cpu_desc, cores = oracle_sample(wl, T, P, 15.0) if world == 1 else (None, 0, 0, "", 0)

    # HBM-bound steps: a5+a6 reads kappa once and writes the k-table; a4 is the kappa store inside the far kernel
    hbm_peak, hbm_src = 6650.0, "of fallback (6.65 TB/s, B200_PROFILING.md)"
    try:
        hbm_peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
        hbm_src = "of measured (MEASURED_PEAKS.json hbm_gbs)"
    except (OSError, KeyError, ValueError):
        pass
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
        "stage_ms": {"line_prep": stage[0], "voigt_far": stage[1], "voigt_near": stage[2], "voigt_accumulate_store": ms_voigt,
                     "kdist": ms_kdist / K},
        "wall_s_timed_region": t_wall,
        "e2e": {"value": world * n_evals * K / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / K},
        "gpu_launches": 4 * K,   # line_prep, voigt_far, voigt_near, kdist
        "roofline": {"kernel": roof_kernel, "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak, "traffic": NCU_DRAM_BYTES[args.precision],
                     "traffic_note": "DRAM bytes per launch from the committed ncu --set full capture (profiles/r01c_*), not live",
                     "note": roof_note, "regime_census": census, "ms": roof_ms,
                     "fp64_peak_tflops": 2.0 * fp64_peak / 1e12, "fp32_peak_tflops": 2.0 * fp32_peak / 1e12},
        "kdist_hbm": {"kernel": "kdist_kernel (a5+a6)", "bound": "hbm", "achieved": kdist_gbs, "peak": hbm_peak, "unit": "GB/s",
                      "frac": kdist_gbs / hbm_peak, "algorithmic_bytes": kdist_bytes, "peak_source": hbm_src,
                      "note": "8 B/point read + 8 n_g B/bin written; the kernel is bound by the bitonic network's "
                              "compare-exchange count, not by HBM (profiles/r01b_kdist_kernel_ncu_full.txt)"},
        "clocks": clocks,
    }
    if cpu_v is not None:
        line["cpu_baseline"] = {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": cpu_desc}
    line["paper_context"] = "~1 s per opacity function of ~1e5 lines on a Tesla K20 (PAPER.md:9, 267); other hardware, not a target"
    print(json.dumps(line))
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--precision", choices=["fp64", "fp32"], default="fp64",
                    help="fp64 (BASELINE.json config 1, the default) or the optional FP32 variant (bar 1e-4)")
    ap.add_argument("--stage-times", action="store_true",
                    help="print per-stage device times of configs 1, 2, 3 (1e7 lines) in both precisions and exit")
    args = ap.parse_args()
    if args.stage_times:
        run_stage_times(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
