#!/usr/bin/env python
"""bench.py -- power-Doppler ensembles/s of the localized EVD clutter filter (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A step = one pass of the whole hot path (Gram -> EVD -> weights -> projection -> combine, SURVEY.md
section 8a) over one synthetic ensemble of BASELINE.json config 2 (256x256x128, 8x8 windows,
sigma 24, 3-sigma boxes, soft energy-rule weights), through the C ABI (`lcf_filter`).  Inputs are
resident in HBM for `value`; `e2e` times `lcf_filter_host` (pinned host in, host out).  Between
timed steps a 512 MiB buffer is overwritten to flush the 126 MB L2 (the 67 MB cube would otherwise
stay resident).  Prints ONE JSON line on rank 0.

N > 1 (torchrun): the path shards by ensemble with no data-path collective (DESIGN.md
"Multi-GPU"); every rank filters its own ensemble, weak scaling, time = max over ranks.

--impl reference: there is no reference implementation (the paper ships no code); this arm times
the float64 CPU oracle (oracle/) on the host cores, on a bounded sample of the same workload.
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-streaming", action="store_true", help="skip the config 4 streaming section")
    return ap.parse_args()


def workload_name(cfg) -> str:
    d, f = cfg.data, cfg.filt
    mode = {0: "hard_fixed", 1: "hard_energy", 2: "soft_fixed", 3: "soft_energy", 4: "hard_median", 5: "soft_median", 6: "hard_curvature", 7: "soft_curvature", 8: "soft_adaptive", 9: "hard_slope", 10: "soft_slope", 11: "hard_slope_db", 12: "soft_slope_db"}[f.mode]
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


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    iq = np.ascontiguousarray(synth.ensemble(synth.generate(cfg), cfg, 0))
    ncores = os.cpu_count() or 1
    nwin = min(8, ncores)
    times, frac, thr, what = [], 1.0, 1, ""
    for i in range(args.warmup + args.steps):
        dt, frac, thr, what = oracle_sample(cfg, iq, nwin)
        if i >= args.warmup:
            times.append(dt)
    t_step = float(np.mean(times)) if times else float("nan")
    value = frac / t_step                                    # ensembles/s extrapolated from the sample
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "note": "no reference code exists (paper only); this arm is "
                   "the float64 CPU oracle, each step a bounded sample of the workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": what},
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
    # every rank filters its own ensemble (same recipe, different seed): weak scaling, no collective
    dspec = d if rank == 0 else type(d)(**{**d.__dict__, "seed": d.seed + 1000 * rank})
    iq_h = torch.from_numpy(np.ascontiguousarray(synth.ensemble(synth.generate_sequence(dspec), cfg, 0))).pin_memory()
    pd_h = torch.empty((d.Nx, d.Nz), dtype=torch.float32).pin_memory()
    iq_d = iq_h.cuda()
    pd_d = torch.empty((d.Nx, d.Nz), dtype=torch.float32, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    stream = torch.cuda.current_stream()
    plan = lcf.Plan.from_spec(d.Nz, d.Nx, d.N, cfg.filt)
    work = plan.work()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps, one CUDA-event pair per step, L2 flushed between steps
    for _ in range(max(args.warmup, 0)):
        flush.zero_()
        plan.filter(iq_d, pd_d, stream)
    plan.set_timing(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            plan.filter(iq_d, pd_d, stream)
            b.record(stream)
        barrier()
        t_wall = time.perf_counter() - t_wall0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    stages = plan.stage_ms() if args.steps > 0 else {}
    plan.set_timing(False)
    total_ms = float(np.sum(step_ms))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / max(args.steps, 1)
    value = world * args.steps / (total_ms * 1e-3)

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
        live = {"ffma": lcf.measure_peak(0), "ffma2": lcf.measure_peak(1), "dfma": lcf.measure_peak(2)}
    except Exception:                                        # measurement helper only
        live = {}
    sweeps = plan.sweeps(allow_unconverged=True)
    N = d.N
    # EVD algorithmic flops: one-sided Jacobi = 36 flops per row per column pair (three dot products,
    # two rotated columns), N rows, N(N-1)/2 pairs per sweep; two-sided = 30 N^3 per sweep
    # (DESIGN.md "Rooflines"); sweeps as measured on this input
    evd_flops = float(sweeps.sum()) * (36.0 * N * N * (N - 1) / 2 if work["evd_chol"] else 30.0 * N ** 3)
    # the contractions run on the FP16 tensor path (.kind::f16, fp32 accumulate): same nominal rate as bf16
    tensor_peak = (peaks.get("bf16_tflops") or 1590.0)
    tensor_src = ("MEASURED_PEAKS.json bf16_tflops (burst); fp16 has the same nominal rate" if peaks.get("bf16_tflops")
                else "fallback 1590 TFLOP/s bf16; fp16 has the same nominal rate")
    fp32_src = "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md Rooflines)"
    kern = {
        "gram": {"kernel": "gram_tc_kernel" if work["gram_tc"] else "gram_kernel", "flops": work["gram_flops"],
                 "bound": "tensor" if work["gram_tc"] else "alu", "executed_flops": work["gram_tensor_flops"] or None},
        "evd": {"kernel": "evd_chol_kernel (Cholesky) + jacobi_cluster_*_kernel | evd_chol_kernel" if work["evd_chol"] else "jacobi_kernel + vbuild_kernel", "flops": evd_flops, "bound": "alu",
                "executed_flops": None},
        "projection": {"kernel": "project_tc_kernel" if work["proj_tc"] else "project_kernel", "flops": work["proj_flops"],
                       "bound": "tensor" if work["proj_tc"] else "alu", "executed_flops": work["proj_tensor_flops"] or None},
    }
    per_kernel = {}
    for sname, kd in kern.items():
        ms = stages.get(sname)
        if not ms:
            continue
        peak = tensor_peak if kd["bound"] == "tensor" else (NOMINAL_FP32_TFLOPS / 2 if cfg.filt.precision == 1 and sname != "projection" else NOMINAL_FP32_TFLOPS)
        ach = kd["flops"] / (ms * 1e-3) / 1e12
        per_kernel[sname] = {"kernel": kd["kernel"], "ms": ms, "bound": kd["bound"], "achieved": ach, "peak": peak,
                             "unit": "TFLOP/s", "frac": ach / peak, "algorithmic_flops_per_launch": kd["flops"],
                             "peak_source": tensor_src if kd["bound"] == "tensor" else fp32_src}
        if kd["executed_flops"]:
            ex = kd["executed_flops"] / (ms * 1e-3) / 1e12
            per_kernel[sname].update({"executed_tflops": ex, "executed_frac": ex / peak,
                                      "executed_note": "3 fp16 products of hi/lo splits per fp32 product, padded tiles: flops the MMAs execute"})
    dom = max(per_kernel, key=lambda s_: per_kernel[s_]["ms"]) if per_kernel else None
    roofline = dict(per_kernel[dom]) if dom else {"bound": "alu", "achieved": None, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s", "frac": None}
    roofline.update({
        "traffic": None, "kernel_ms": roofline.get("ms"), "stages_ms": stages, "per_kernel": per_kernel,
        "live_pipe_peaks_tflops": live,
        "evd_sweeps": {"mean": float(sweeps.mean()), "max": int(sweeps.max())},
        "hbm": {"algorithmic_bytes": work["hbm_bytes"], "peak_gbs": peaks.get("hbm_gbs"),
                "peak_source": "MEASURED_PEAKS.json" if peaks else "absent"},
    })
    if dom == "evd":
        roofline["note"] = ("the EVD is bound by instruction issue and dependency latency, not by a memory system: the "
                            "cluster Jacobi keeps the columns in registers (16 warps per SM, issue slots 63 % busy, FMA pipe "
                            "49 %, profiles/r1g) and the flops counted here are the rotations' 36 per row and pair only")
        # DRAM bytes of one Cholesky + one cluster-Jacobi launch, from the ncu --set full capture
        # profiles/r1g_ncu_full_summary.txt (dram__bytes_read.sum + dram__bytes_write.sum), config 2
        if args.config == 2 and "jacobi_cluster" in roofline.get("kernel", ""):
            roofline["traffic"] = 8.4544e6 + 8.7168e6
            roofline["traffic_source"] = "profiles/r1g_ncu_full_summary.txt"

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
            streaming = {"workload": workload_name(cfg4) + f", {cfg4.n_ensembles} ensembles at stride {cfg4.stride} of a "
                         f"resident {d4.n_frames}-frame sequence, 3 passes, L2 not flushed (472 MB sequence > L2)",
                         "pd_frames_per_s": len(evs) / (tot * 1e-3), "latency_ms": {"median": float(np.median(lat)),
                         "p95": float(np.percentile(lat, 95))}}
            del seq_d
        except Exception as ex:                                  # reported, never fatal for the headline
            streaming = {"error": repr(ex)}

    cpu = None
    if not args.no_cpu_baseline:
        dt, frac, thr, what = oracle_sample(cfg, iq_h.numpy(), 4 * (os.cpu_count() or 1))
        cpu = {"value": frac / dt, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": what,
               "seconds": dt}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if cfg.filt.precision == 0 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "l2": "512 MiB buffer overwritten between timed steps",
                   "parallelism": f"ensemble-sharded x{world}, no collective", "timing": "CUDA events per step"},
        "latency_ms": {"median": float(np.median(step_ms)), "min": float(np.min(step_ms)),
                       "p95": float(np.percentile(step_ms, 95))},
        "pd_frames_per_s": value,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(iq_h.numel() * 8),
                "d2h_bytes_per_step": int(pd_h.numel() * 4), "api": "lcf_filter_host_batch (copies pipelined under the kernels)",
                "serial_lcf_filter_host": world * args.steps / e2e_serial_s, "pd_checksum": pd_sum},
        "gpu_launches": int(work["launches"]) * args.steps,
        "clocks": clk.summary(), "wall_s_timed_region": t_wall,
        "roofline": roofline, "cpu_baseline": cpu, "streaming_config4": streaming,
    }
    print(json.dumps(line), flush=True)
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    cfg = synth.baseline_configs()[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
