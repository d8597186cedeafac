#!/usr/bin/env python
"""bench.py -- power-Doppler ensembles/s of the localized EVD clutter filter (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A step = one pass of the whole hot path (Gram -> EVD -> weights -> projection -> combine, SURVEY.md
section 8a) over one synthetic ensemble of BASELINE.json config 2 (256x256x128, 8x8 windows,
sigma 24, 3-sigma boxes, soft energy-rule weights), through the C ABI.

  value     K ensembles through one `lcf_filter_batch` call (the plan's three lanes overlap the kernels of
            consecutive ensembles), inputs resident in HBM: a ring of 4 distinct ensembles (268 MB > the
            126 MB L2), CUDA events on the caller's stream, max over ranks.
  latency   single `lcf_filter` calls with the L2 flushed between them; the per-kernel stage times of
            these calls feed the rooflines (a kernel timed alone).
  e2e       `lcf_filter_host_batch` from pinned host memory (copies inside the timed region, wall clock).
  per_config / paper_shaped_context   latency of the other BASELINE.json configs and of the paper's
            shapes (context for PAPER.md:184-238).
Prints ONE JSON line on rank 0.

N > 1 (torchrun): the path shards by ensemble with no data-path collective (DESIGN.md
"Multi-GPU"); every rank filters its own ensembles, weak scaling, time = max over ranks.

--impl reference: there is no reference implementation (the paper ships no code); this arm times
the float64 CPU oracle (oracle/) on the host cores: every step is all windows of one ensemble.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2405_11105_b200 import synth  # noqa: E402

METRIC = "power-Doppler ensembles/sec at 256x256x128, 64 windows"
UNIT = "ensembles/s"
# FP32 roofline denominator derived from unit counts and clocks:
# 148 SMs x 128 FP32 lanes x 2 flop/FMA x 1.965 GHz (clocks.max.sm)
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (metric: 2)")
    ap.add_argument("--thresh-mode", type=int, default=None,
                    help="override the threshold mode of the chosen config (include/lcf.h lcf_thresh_mode; e.g. 16 = "
                         "LCF_HARD_ENERGY_TOP); the workload string says so.  For profiling the other kernels.")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-streaming", action="store_true", help="skip the config 4 streaming section")
    ap.add_argument("--no-context", action="store_true", help="skip the per-config latencies and the paper-shaped context runs")
    return ap.parse_args()


def workload_name(cfg) -> str:
    d, f = cfg.data, cfg.filt
    mode = {0: "hard_fixed", 1: "hard_energy", 2: "soft_fixed", 3: "soft_energy", 4: "hard_median", 5: "soft_median", 6: "hard_curvature", 7: "soft_curvature", 8: "soft_adaptive", 9: "hard_slope", 10: "soft_slope", 11: "hard_slope_db", 12: "soft_slope_db", 13: "hard_ncc", 14: "soft_ncc", 15: "hard_fixed_top", 16: "hard_energy_top"}[f.mode]
    return (f"{cfg.name}: IQ {d.Nz}x{d.Nx}x{d.N} complex64, {f.Kz}x{f.Kx} windows sigma={f.sigma_z:g} "
            f"trunc={f.trunc:g}, {mode}, precision={f.precision}")


# ------------------------------------------------------------------------------ clocks sampling
class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.t.join(timeout=2)

    def summary(self) -> dict:
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------ CPU oracle timing
def oracle_sample(cfg, iq, n_windows: int):
    """Times the float64 oracle (as it stands) on a sample of whole windows of this workload, one
    window per host thread, plus Eq. 13 over the sampled windows.  Returns (seconds, fraction of
    the ensemble's sum_k P_k the sample covers, threads used, description)."""
    from oracle import lcf_oracle as orc
    from concurrent.futures import ThreadPoolExecutor
    orc.build()
    d, f = cfg.data, cfg.filt
    K = f.Kz * f.Kx
    gz = orc.axis_windows(d.Nz, f.Kz, f.sigma_z, f.trunc)
    gx = orc.axis_windows(d.Nx, f.Kx, f.sigma_x, f.trunc)
    n = min(n_windows, K)
    ks = sorted({int(round(i * (K - 1) / max(n - 1, 1))) for i in range(n)})      # spread over the grid
    Pk = lambda k: int((gz[k % f.Kz] != 0).sum()) * int((gx[k // f.Kz] != 0).sum())
    frac = sum(Pk(k) for k in ks) / float(sum(Pk(k) for k in range(K)))
    threads = min(len(ks), os.cpu_count() or 1)

    def one(k):
        return orc.window(iq, gz[k % f.Kz], gx[k // f.Kz], f.mode, f.k_fixed, f.energy_frac, f.beta, f.cut_scale)["PDk"]

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=threads) as ex:           # ctypes releases the GIL
        tiles = list(ex.map(one, ks))
    orc.combine(np.stack(tiles))
    dt = time.perf_counter() - t0
    what = (f"float64 oracle (oracle/lcf_oracle.c, gcc -O2) on {len(ks)} of {K} windows "
            f"({100 * frac:.1f}% of sum_k P_k) of one ensemble, one window per thread, "
            f"scaled by that fraction")
    return dt, frac, threads, what


def oracle_single_thread(cfg, iq):
    """Single-thread oracle time of one ensemble, extrapolated from two whole windows (first and central)."""
    from oracle import lcf_oracle as orc
    d, f = cfg.data, cfg.filt
    K = f.Kz * f.Kx
    gz = orc.axis_windows(d.Nz, f.Kz, f.sigma_z, f.trunc)
    gx = orc.axis_windows(d.Nx, f.Kx, f.sigma_x, f.trunc)
    Pk = lambda k: int((gz[k % f.Kz] != 0).sum()) * int((gx[k // f.Kz] != 0).sum())
    ks = sorted({0, K // 2})
    t0 = time.perf_counter()
    for k in ks:
        orc.window(iq, gz[k % f.Kz], gx[k // f.Kz], f.mode, f.k_fixed, f.energy_frac, f.beta, f.cut_scale)
    dt = time.perf_counter() - t0
    frac = sum(Pk(k) for k in ks) / float(sum(Pk(k) for k in range(K)))
    return dt / frac, f"{len(ks)} of {K} windows ({100 * frac:.1f}% of sum_k P_k) on one thread, scaled by that fraction"


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores (rank 0 only).  There is no reference code (the
    paper ships none); each step is the float64 oracle on ALL windows of one ensemble, one window per
    host thread -- the same measurement as the `cpu_baseline` of the CUDA arm."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    iq = np.ascontiguousarray(synth.ensemble(synth.generate(cfg), cfg, 0))
    K = cfg.filt.Kz * cfg.filt.Kx
    times, frac, thr, what = [], 1.0, 1, ""
    for i in range(args.warmup + args.steps):
        dt, frac, thr, what = oracle_sample(cfg, iq, K)
        if i >= args.warmup:
            times.append(dt)
    t_step = float(np.mean(times)) if times else float("nan")
    value = frac / t_step
    t1, what1 = oracle_single_thread(cfg, iq)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "note": "no reference code exists (paper only); this arm is "
                   "the float64 CPU oracle on all windows of one ensemble per step, one window per host thread"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": what,
                         "single_thread": {"value": 1.0 / t1, "unit": UNIT, "seconds_per_ensemble": t1, "sample": what1}},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------ the CUDA arm
def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text())
        except ValueError:
            pass
    return {}


def profiled_traffic(kernel_substr: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the named kernel, parsed from the newest
    profiles/*_ncu_full_summary.txt (text of `ncu --page raw`); (None, None) if no committed capture has it."""
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    files = sorted((ROOT / "profiles").glob("*_ncu_full_summary.txt"), key=lambda f: f.name, reverse=True)
    for f in files:
        cur, tot, found = None, {}, None
        for ln in f.read_text().splitlines():
            t = ln.split()
            if ln.startswith("  ") and not ln.startswith("    ") and "(" in ln and "Device" in ln:    # "  kernel(args) (grid)x(block), Context ..., Device ..."
                cur = ln.strip()
            elif cur and len(t) >= 3 and t[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and t[1] in unit:
                try:
                    tot.setdefault(cur, {})[t[0]] = float(t[2].replace(",", "")) * unit[t[1]]
                except ValueError:
                    pass
        for name, v in tot.items():
            if kernel_substr in name and len(v) == 2:
                found = sum(v.values())
                break
        if found is not None:
            return found, f"profiles/{f.name}"
    return None, None


def quick_latency(lcf, torch, cfg, iq, steps=5, warmup=2):
    """ms per lcf_filter call (median of CUDA-event times, inputs resident) and the plan's stage times."""
    d = cfg.data
    iq_d = torch.from_numpy(np.ascontiguousarray(iq)).cuda()
    pd_d = torch.empty((d.Nx, d.Nz), dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream()
    with lcf.Plan.from_spec(d.Nz, d.Nx, d.N, cfg.filt) as plan:
        w = plan.work()
        for _ in range(warmup):
            plan.filter(iq_d, pd_d, st)
        plan.set_timing(True)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            a.record(st); plan.filter(iq_d, pd_d, st); b.record(st)
        torch.cuda.synchronize()
        ms = float(np.median([a.elapsed_time(b) for a, b in ev]))
        stages = plan.stage_ms()
        unconv = plan.unconverged()
    return {"ms": ms, "stages_ms": {k: round(v, 4) for k, v in stages.items()},
            "kernels": {"gram_tc": w["gram_tc"], "evd_chol": w["evd_chol"], "proj_tc": w["proj_tc"]}, "unconverged_windows": unconv}


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2405_11105_b200 import lcf            # raises if liblcf.so is missing: no fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    lcf.load()

    d = cfg.data
    # every rank filters its own ensembles (same recipe, different seeds): weak scaling, no collective.
    # A ring of RING distinct resident ensembles (4 x 67 MB = 268 MB at config 2) is larger than the 126 MB L2,
    # so consecutive steps never find their input cached; no flush is needed in the throughput loop.
    RING = 4
    def ens(i):
        dspec = type(d)(**{**d.__dict__, "seed": d.seed + 1000 * rank + 7 * i})
        return np.ascontiguousarray(synth.ensemble(synth.generate_sequence(dspec), cfg, 0))
    iq_h = torch.from_numpy(ens(0)).pin_memory()
    pd_h = torch.empty((d.Nx, d.Nz), dtype=torch.float32).pin_memory()
    ring = [iq_h.cuda()] + [torch.from_numpy(ens(i)).cuda() for i in range(1, RING)]
    iq_d = ring[0]
    pd_d = torch.empty((d.Nx, d.Nz), dtype=torch.float32, device="cuda")
    pd_ring = [pd_d, torch.empty_like(pd_d), torch.empty_like(pd_d)]      # one image buffer per lane
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2, for the latency loop
    stream = torch.cuda.current_stream()
    plan = lcf.Plan.from_spec(d.Nz, d.Nx, d.N, cfg.filt)
    work = plan.work()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- throughput (`value`): K steps = one lcf_filter_batch call over the ring (three lanes inside the plan:
    # the kernels of consecutive ensembles overlap), CUDA events on the caller's stream around it
    def batch(n):
        plan.filter_batch([ring[i % RING] for i in range(n)], [pd_ring[i % 3] for i in range(n)], stream)
    if args.warmup > 0:
        batch(max(args.warmup, 4))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        e0.record(stream)
        batch(args.steps)
        e1.record(stream)
        barrier()
        t_wall = time.perf_counter() - t_wall0
    total_ms = float(e0.elapsed_time(e1))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / max(args.steps, 1)
    value = world * args.steps / (total_ms * 1e-3)

    # ---- latency and per-kernel times: single lcf_filter calls, one CUDA-event pair per call, L2 flushed
    # between calls, stage events between the launches (a kernel timed alone: the rooflines use these)
    nlat = max(min(args.steps, 50), 1)
    for _ in range(3):
        flush.zero_()
        plan.filter(iq_d, pd_d, stream)
    plan.set_timing(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nlat)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        plan.filter(iq_d, pd_d, stream)
        b.record(stream)
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    stages = plan.stage_ms()
    plan.set_timing(False)

    # ---- end to end through the host API: every step copies its ensemble from pinned host memory
    # and reads its image back.  lcf_filter_host_batch pipelines the copy of step i+1 under the
    # kernels of step i; the serial lcf_filter_host figure is reported next to it.
    for _ in range(min(3, max(args.warmup, 1))):
        plan.filter_host(iq_h, pd_h, stream)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        plan.filter_host(iq_h, pd_h, stream)            # synchronises the stream before returning
    barrier()
    e2e_serial_s = time.perf_counter() - t0
    plan.filter_host_batch([iq_h] * 2, [pd_h] * 2, stream)      # creates the second staging set
    barrier()
    t0 = time.perf_counter()
    plan.filter_host_batch([iq_h] * args.steps, [pd_h] * args.steps, stream)
    barrier()
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = world * args.steps / e2e_s
    pd_sum = float(pd_h.double().sum())

    if rank != 0:
        plan.destroy()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines (live stage times from CUDA events recorded between the launches)
    peaks = measured_peaks()
    try:
        live = {"ffma": lcf.measure_peak(0), "ffma2": lcf.measure_peak(1), "dfma": lcf.measure_peak(2), "tcgen05_f16": lcf.measure_peak(3)}
    except Exception:                                        # measurement helper only
        live = {}
    unconverged = plan.unconverged()                         # over every lcf_filter call of the timed loops
    if unconverged:
        raise SystemExit(f"bench.py: {unconverged} window EVDs hit the sweep cap on the timed input: the number would be invalid")
    sweeps = plan.sweeps()
    N = d.N
    # EVD algorithmic flops: one-sided Jacobi = 36 flops per row per column pair (three dot products,
    # two rotated columns), N rows, N(N-1)/2 pairs per sweep; two-sided = 30 N^3 per sweep
    # (DESIGN.md "Rooflines"); sweeps as measured on this input
    if work["evd_chol"] == 2:
        # leading-eigenpair modes: a round of the block iteration on M = 16 vectors is the product R Q (8 N^2 M), the
        # small Gram H (8 N M^2), classical Gram-Schmidt twice (16 N M^2 / 2 x 2) and the rotation of Q and Y
        # (16 N M^2): 8 N M (N + 5 M) flops in double; rounds as measured on this input
        Mb = 16
        evd_flops = float(sweeps.sum()) * 8.0 * N * Mb * (N + 5 * Mb)
    else:
        evd_flops = float(sweeps.sum()) * (36.0 * N * N * (N - 1) / 2 if work["evd_chol"] else 30.0 * N ** 3)
    # the contractions run on the FP16 tensor path (.kind::f16, fp32 accumulate).  Denominator: the bare
    # tcgen05 kind::f16 loop measured in this run (lcf_measure_peak(3)); MEASURED_PEAKS.json's bf16 matmul
    # figure (same nominal rate) is carried beside it
    if live.get("tcgen05_f16"):
        tensor_peak, tensor_src = live["tcgen05_f16"], "lcf_measure_peak(3): bare tcgen05.mma.kind::f16 128x256x16 loop, this run"
    elif peaks.get("bf16_tflops"):
        tensor_peak, tensor_src = peaks["bf16_tflops"], "MEASURED_PEAKS.json bf16_tflops (burst); fp16 has the same nominal rate"
    else:
        tensor_peak, tensor_src = 1590.0, "fallback 1590 TFLOP/s bf16 (B200_PROFILING.md); fp16 has the same nominal rate"
    if live.get("ffma2"):
        fp32_peak, fp32_src = live["ffma2"], "lcf_measure_peak(1): FFMA2 register loop, this run (derived 148 x 128 x 2 x 1.965 GHz = %.1f)" % NOMINAL_FP32_TFLOPS
    else:
        fp32_peak, fp32_src = NOMINAL_FP32_TFLOPS, "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md Rooflines)"
    fp64_peak = live.get("dfma") or NOMINAL_FP32_TFLOPS / 2
    kern = {
        "gram": {"kernel": "gram_tc_kernel" if work["gram_tc"] else "gram_kernel", "flops": work["gram_flops"],
                 "bound": "tensor" if work["gram_tc"] else "alu", "executed_flops": work["gram_tensor_flops"] or None},
        "evd": {"kernel": "evd_top_kernel (block subspace iteration, fp64)" if work["evd_chol"] == 2 else ("evd_chol_kernel (Cholesky) + jacobi_cluster_*_kernel | evd_chol_kernel" if work["evd_chol"] else "jacobi_kernel + vbuild_kernel"), "flops": evd_flops, "bound": "alu",
                "executed_flops": None},
        "projection": {"kernel": "project_tc_kernel" if work["proj_tc"] else ("project_dd_kernel" if cfg.filt.precision == 1 else "project_kernel"), "flops": work["proj_flops"],
                       "bound": "tensor" if work["proj_tc"] else "alu", "executed_flops": work["proj_tensor_flops"] or None},
    }
    per_kernel = {}
    for sname, kd in kern.items():
        ms = stages.get(sname)
        if not ms:
            continue
        dbl = cfg.filt.precision == 1 or (sname == "evd" and work["evd_chol"] == 2)       # kernels on the FP64 pipe
        peak = tensor_peak if kd["bound"] == "tensor" else (fp64_peak if dbl else fp32_peak)
        ach = kd["flops"] / (ms * 1e-3) / 1e12
        per_kernel[sname] = {"kernel": kd["kernel"], "ms": ms, "bound": kd["bound"], "achieved": ach, "peak": peak,
                             "unit": "TFLOP/s", "frac": ach / peak, "algorithmic_flops_per_launch": kd["flops"],
                             "peak_source": tensor_src if kd["bound"] == "tensor" else ("lcf_measure_peak(2): DFMA register loop, this run" if dbl else fp32_src)}
        if kd["executed_flops"]:
            ex = kd["executed_flops"] / (ms * 1e-3) / 1e12
            per_kernel[sname].update({"executed_tflops": ex, "executed_frac": ex / peak,
                                      "executed_note": "3 fp16 products of hi/lo splits per fp32 product, padded tiles: flops the MMAs execute (pipe occupancy, not a roofline fraction of the method's work; with the x3 split the algorithmic ceiling is 1/3)"})
        if kd["bound"] == "tensor" and peaks.get("bf16_tflops"):
            per_kernel[sname]["frac_vs_measured_peaks_bf16"] = ach / peaks["bf16_tflops"]
    dom = max(per_kernel, key=lambda s_: per_kernel[s_]["ms"]) if per_kernel else None
    roofline = dict(per_kernel[dom]) if dom else {"bound": "alu", "achieved": None, "peak": fp32_peak, "unit": "TFLOP/s", "frac": None}
    roofline.update({
        "traffic": None, "kernel_ms": roofline.get("ms"), "stages_ms": stages, "per_kernel": per_kernel,
        "stage_times_from": "single lcf_filter calls with the L2 flushed (kernels timed alone; in the three-lane throughput loop they overlap)",
        "live_pipe_peaks_tflops": live,
        "evd_sweeps": {"mean": float(sweeps.mean()), "max": int(sweeps.max())},
        "hbm": {"algorithmic_bytes": work["hbm_bytes"], "peak_gbs": peaks.get("hbm_gbs"),
                "peak_source": "MEASURED_PEAKS.json" if peaks else "absent"},
    })
    if dom == "evd":
        roofline["note"] = ("the EVD is bound by instruction issue and dependency latency, not by a memory system: the cluster "
                            "Jacobi keeps the columns in registers (16 warps per SM); the flops counted here are the rotations' "
                            "36 per row and pair x the sweeps measured on this input")
    # DRAM bytes per launch of the dominant kernel from the newest committed ncu --set full summary (static, not measured in this run)
    dom_kernel = {"gram": "gram_tc", "evd": "jacobi_cluster", "projection": "project_tc"}.get(dom, "")
    if args.config == 2 and dom_kernel:
        roofline["traffic"], roofline["traffic_source"] = profiled_traffic(dom_kernel)

    # ---- BASELINE.json config 4: 16 ensembles of 100 frames at stride 50 over one resident
    # 900-frame sequence (pointer offsets, no copies): sustained power-Doppler frames/s, latency
    streaming = None
    if not args.no_streaming and args.config == 2:
        try:
            cfg4 = synth.baseline_configs()[4]
            d4 = cfg4.data
            seq_d = torch.from_numpy(synth.generate(cfg4)).cuda()
            pd4 = torch.empty((d4.Nx, d4.Nz), dtype=torch.float32, device="cuda")
            with lcf.Plan.from_spec(d4.Nz, d4.Nx, d4.N, cfg4.filt) as plan4:
                views = [seq_d[e * cfg4.stride:e * cfg4.stride + d4.N] for e in range(cfg4.n_ensembles)]
                for v in views[:3]:
                    plan4.filter(v, pd4, stream)
                evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                       for _ in range(3 * len(views))]
                torch.cuda.synchronize()
                for i, (a4, b4) in enumerate(evs):
                    a4.record(stream)
                    plan4.filter(views[i % len(views)], pd4, stream)
                    b4.record(stream)
                torch.cuda.synchronize()
                lat = np.array([a4.elapsed_time(b4) for a4, b4 in evs])
                tot = evs[0][0].elapsed_time(evs[-1][1])
                # sustained rate through the two-lane batch entry point (3 passes over the 16 ensembles)
                pd4b = [pd4, torch.empty_like(pd4), torch.empty_like(pd4)]
                n4 = 3 * len(views)
                plan4.filter_batch(views[:4], [pd4b[i % 3] for i in range(4)], stream)
                torch.cuda.synchronize()
                s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                s0.record(stream)
                plan4.filter_batch([views[i % len(views)] for i in range(n4)], [pd4b[i % 3] for i in range(n4)], stream)
                s1.record(stream)
                torch.cuda.synchronize()
                tot_b = s0.elapsed_time(s1)
                assert plan4.unconverged() == 0
                # sliding-window reuse (lcf_filter_stream): only the 50 new frames' Gram columns per call; single lane
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                plan4.set_timing(True)
                plan4.filter_stream(views[0], pd4, cfg4.stride, stream)
                g0.record(stream)
                for i in range(1, len(views)):
                    plan4.filter_stream(views[i], pd4, cfg4.stride, stream)
                g1.record(stream)
                torch.cuda.synchronize()
                reuse_ms = g0.elapsed_time(g1) / (len(views) - 1)
                reuse_gram_ms = plan4.stage_ms()["gram"]
                plan4.set_timing(False)
                assert plan4.unconverged() == 0
            streaming = {"workload": workload_name(cfg4) + f", {cfg4.n_ensembles} ensembles at stride {cfg4.stride} of a "
                         f"resident {d4.n_frames}-frame sequence, 3 passes, L2 not flushed (472 MB sequence > L2)",
                         "pd_frames_per_s": n4 / (tot_b * 1e-3), "how": "lcf_filter_batch (three lanes), CUDA events around the call",
                         "pd_frames_per_s_single_lane": len(evs) / (tot * 1e-3),
                         "latency_ms": {"median": float(np.median(lat)), "p95": float(np.percentile(lat, 95))},
                         "sliding_window_reuse": {"api": "lcf_filter_stream(stride=50): Gram columns of the new frames only, the rest shifted from the previous call",
                                                  "ms_per_ensemble": reuse_ms, "gram_stage_ms": reuse_gram_ms,
                                                  "note": "single lane; compare latency_ms.median (full Gram every call)"}}
            del seq_d
        except Exception as ex:                                  # reported, never fatal for the headline
            streaming = {"error": repr(ex)}

    # ---- the other BASELINE.json configs (parity cases, not the metric): latency per ensemble, resident inputs
    per_config = None
    context = None
    if args.config == 2 and not args.no_context:
        per_config = {}
        for ci in (0, 1, 3, 4):
            try:
                c = synth.baseline_configs()[ci]
                seq = synth.generate(c)
                r = quick_latency(lcf, torch, c, synth.ensemble(seq, c, 0))
                r["workload"] = workload_name(c)
                per_config[f"config{ci}"] = r
                del seq
            except Exception as ex:
                per_config[f"config{ci}"] = {"error": repr(ex)}
        from dataclasses import replace as _rep
        # the hard energy cut from the leading eigenpairs only (LCF_HARD_ENERGY_TOP): config 3 as
        # BASELINE.json states it is 'config3' above (full-spectrum EVD); the same filter by subspace iteration here,
        # and the metric workload's shape under the same hard rule both ways
        for name, ci, mode in (("config3_hard_energy_top", 3, synth.HARD_ENERGY_TOP), ("config2_hard_energy", 2, synth.HARD_ENERGY),
                               ("config2_hard_energy_top", 2, synth.HARD_ENERGY_TOP)):
            try:
                c0 = synth.baseline_configs()[ci]
                c = _rep(c0, filt=_rep(c0.filt, mode=mode))
                r = quick_latency(lcf, torch, c, synth.ensemble(synth.generate(c0), c0, 0))
                r["workload"] = workload_name(c)
                per_config[name] = r
            except Exception as ex:
                per_config[name] = {"error": repr(ex)}
        try:                                                 # the metric workload with method 4 + 5 (NCC cut-off): one more pass over the data
            c = _rep(cfg, filt=_rep(cfg.filt, mode=synth.SOFT_NCC))
            r = quick_latency(lcf, torch, c, iq_h.numpy())
            r["workload"] = workload_name(c)
            per_config["config2_method4_ncc"] = r
        except Exception as ex:
            per_config["config2_method4_ncc"] = {"error": repr(ex)}
        # ---- paper-shaped context runs (phantom 196x180, kidney 180x180, liver 177x173; packets
        # 50/70/90; global, 2x2, 3x3 un-truncated Gaussian subsets, fixed cut): ms per packet next to the paper's
        # 2.4 / 16.6 / 39.8 ms (RTX A6000 + Xeon, MATLAB).  Synthetic data of that shape; context, not the target.
        context = {"note": "synthetic IQ of the paper's shapes, hard fixed cut k = 5, windows over the full field of view (trunc = 0), "
                           "sigma = 0.75 x window spacing; paper (RTX A6000 + Xeon W-2265, MATLAB, PAPER.md:198,212,224): "
                           "global 2.4-2.6 ms, 2x2 15.6-16.6 ms, 3x3 35.2-39.8 ms per packet of 50",
                   "ms_per_packet": {}}
        base = synth.baseline_configs()[1]
        for (name, Nz, Nx) in (("phantom_196x180", 196, 180), ("kidney_180x180", 180, 180), ("liver_177x173", 177, 173)):
            for Np_ in (50, 70, 90):
                try:
                    dsp = type(base.data)(**{**base.data.__dict__, "Nz": Nz, "Nx": Nx, "N": Np_, "n_frames": Np_, "seed": 50 + Np_})
                    seq = synth.generate_sequence(dsp)
                    for Kg in (1, 2, 3):
                        if Kg == 1:
                            f = synth.FilterSpec(1, 1, 0.0, 0.0, 0.0, synth.HARD_FIXED, k_fixed=5, precision=0)
                        else:
                            f = synth.FilterSpec(Kg, Kg, 0.75 * Nz / Kg, 0.75 * Nx / Kg, 0.0, synth.HARD_FIXED, k_fixed=5, precision=0)
                        c = synth.Config(f"{name}_N{Np_}_K{Kg}x{Kg}", dsp, f)
                        r = quick_latency(lcf, torch, c, seq, steps=5, warmup=2)
                        context["ms_per_packet"][c.name] = round(r["ms"], 4)
                except Exception as ex:
                    context["ms_per_packet"][f"{name}_N{Np_}"] = repr(ex)

    # ---- the paper's own sliding regime (packet 50, 5-frame interval = 90 % overlap), 180x180, 3x3 windows
    paper_stream = None
    if args.config == 2 and not args.no_context:
        try:
            base = synth.baseline_configs()[4]
            dsp = type(base.data)(**{**base.data.__dict__, "Nz": 180, "Nx": 180, "N": 50, "n_frames": 150, "seed": 77})
            fs = synth.FilterSpec(3, 3, 45.0, 45.0, 3.0, synth.SOFT_ENERGY, precision=0)
            seqp = torch.from_numpy(synth.generate_sequence(dsp)).cuda()
            pdp = torch.empty((180, 180), dtype=torch.float32, device="cuda")
            res = {}
            with lcf.Plan.from_spec(180, 180, 50, fs) as pp:
                for name in ("reuse", "full"):
                    pp.set_timing(True)
                    for rep in range(2):
                        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        if name == "reuse":
                            pp.filter_stream(seqp[0:50], pdp, 5, stream)
                        q0.record(stream)
                        for e in range(1, 21):
                            v = seqp[5 * e:5 * e + 50]
                            (pp.filter_stream(v, pdp, 5, stream) if name == "reuse" else pp.filter(v, pdp, stream))
                        q1.record(stream)
                        torch.cuda.synchronize()
                    res[name] = {"ms_per_packet": q0.elapsed_time(q1) / 20, "stages_ms": {k_: round(v_, 4) for k_, v_ in pp.stage_ms().items()}}
                    pp.set_timing(False)
            paper_stream = {"workload": "180x180x50 packets at a 5-frame interval, 3x3 windows sigma=45 trunc=3, soft_energy", **res}
            del seqp
        except Exception as ex:
            paper_stream = {"error": repr(ex)}

    cpu = None
    if not args.no_cpu_baseline:
        dt, frac, thr, what = oracle_sample(cfg, iq_h.numpy(), cfg.filt.Kz * cfg.filt.Kx)
        t1, what1 = oracle_single_thread(cfg, iq_h.numpy())
        cpu = {"value": frac / dt, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": what,
               "seconds": dt, "single_thread": {"value": 1.0 / t1, "unit": UNIT, "seconds_per_ensemble": t1, "sample": what1}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "data": "synthetic",
        "dtype": ("f16x2-split/f32-acc (contractions), f32 (EVD)" if (work["gram_tc"] or work["proj_tc"]) else "f32") if cfg.filt.precision == 0 else "f64 (Gram, EVD), f16x2-split/f32-acc (projection)",
        "config": {"workload": workload_name(cfg),
                   "l2": f"ring of {RING} distinct resident ensembles ({RING * iq_h.numel() * 8 / 1e6:.0f} MB) > 126 MB L2, no flush needed",
                   "parallelism": f"ensemble-sharded x{world}, no collective",
                   "timing": "CUDA events on the caller's stream around one lcf_filter_batch call of K ensembles (three lanes inside the plan)"},
        "latency_ms": {"median": float(np.median(step_ms)), "min": float(np.min(step_ms)),
                       "p95": float(np.percentile(step_ms, 95)), "calls": nlat,
                       "how": "single lcf_filter calls, CUDA events per call, 512 MiB buffer overwritten between calls (L2 flushed)"},
        "single_lane_ensembles_per_s": 1e3 / float(np.mean(step_ms)),
        "pd_frames_per_s": value,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(iq_h.numel() * 8),
                "d2h_bytes_per_step": int(pd_h.numel() * 4), "api": "lcf_filter_host_batch (copies pipelined under the kernels)",
                "serial_lcf_filter_host": world * args.steps / e2e_serial_s, "pd_checksum": pd_sum},
        "gpu_launches": int(work["launches"]) * args.steps,
        "clocks": clk.summary(), "wall_s_timed_region": t_wall,
        "roofline": roofline, "cpu_baseline": cpu, "streaming_config4": streaming,
        "per_config": per_config, "paper_shaped_context": context, "paper_sliding_packets": paper_stream,
    }
    print(json.dumps(line), flush=True)
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    cfg = synth.baseline_configs()[args.config]
    if args.thresh_mode is not None:
        from dataclasses import replace as _rep
        cfg = _rep(cfg, filt=_rep(cfg.filt, mode=args.thresh_mode))
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
