#!/usr/bin/env python
"""bench.py — headline measurement of the averaged-RQA hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--series all|0,4]

Metric (BASELINE.json): recurrence cells x thresholds per second at N = 1e5, K = 20 recurrence rates.
Workload at N=1 GPU: BASELINE.json configs[3] ("config4"): five series of N = 1e5 (logistic and Lorenz x at
SNR 1 and 0.1, white noise), m = 3, tau = 1, max norm, K = 20 log-spaced RRs 0.001..0.2, l_min = 2.
A step = one pass of the whole hot path (rqa_eps_for_rr -> rqa_line_hist -> rqa_det_avg; the embedding is a
strided view) over the batch of five series, 5 x 9.9995e10 = 5.0e11 cells x thresholds.

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2208_09136_b200 import shard, workloads as wl  # noqa: E402

METRIC = "recurrence cells x thresholds / s at N=1e5, K=20 RRs"
UNIT = "cells*thresholds/s"

# ALU issue roofline: 148 SMs x 4 schedulers x 32 lanes = 18 944 lane-instructions per clock,
# at the maximum SM clock of 1965 MHz (B200_PROFILING.md; MEASURED_PEAKS.json sm_max_mhz).
SM_COUNT, LANES_PER_SM_CLK = 148, 128
# algorithmic lane-instructions per cell of the line-scan kernel: distance 2m-1 = 5, plus one
# threshold test and one run update per threshold = 2K.
def line_scan_lane_instr_per_cell(m: int, K: int) -> int:
    return (2 * m - 1) + 2 * K


# DRAM bytes of ONE line_scan_kernel launch over one N=1e5, K=20 series (dram__bytes_read.sum + dram__bytes_write.sum of
# the ncu --set full capture in profiles/r1k_ncu_line_scan.md); the bench launch covers `batch` series.
NCU_LINE_SCAN_DRAM_BYTES_PER_SERIES = 341.5e6


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        return json.loads(p.read_text()), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([f.strip() for f in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------- reference arm
def oracle_sample_run(series, m, tau, rr, norm, l_min, n_sample, threads):
    """The oracle as it stands on a bounded sample (the first n_sample points of one series)."""
    from oracle import rqa_oracle
    y = np.ascontiguousarray(series[:n_sample])
    t0 = time.perf_counter()
    rqa_oracle.sweep(y, m, tau, rr, norm, l_min, threads=threads)
    dt = time.perf_counter() - t0
    units = rqa_oracle.n_pairs(len(y), m, tau) * len(rr)
    return units, dt


def run_reference(args):
    rank, world, _ = shard.env_rank_world()
    if rank != 0:
        return 0
    from oracle import rqa_oracle
    rqa_oracle.build()
    w = wl.config4(which=[4])
    cores = rqa_oracle.max_threads()
    n_sample = args.ref_sample
    for _ in range(args.warmup):
        oracle_sample_run(w.series[0], w.m, w.tau, w.rr, w.norm, 2, min(n_sample, 2000), 0)
    total_units, total_t = 0, 0.0
    for _ in range(args.steps):
        u, dt = oracle_sample_run(w.series[0], w.m, w.tau, w.rr, w.norm, 2, n_sample, 0)
        total_units += u
        total_t += dt
    value = total_units / total_t
    sample = f"first {n_sample} points of the config4 white-noise series, K={w.K}, whole path per step"
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": "config4_long_N100000 (bounded sample)", "N": n_sample, "m": w.m, "tau": w.tau, "K": w.K,
                      "norm": "max", "l_min": 2},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch

    import paper_2208_09136_b200 as rqa

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    rank, world, local = shard.env_rank_world()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    shard.init_process_group("nccl")
    rqa.load_library()

    which = None if args.series == "all" else [int(s) for s in args.series.split(",")]
    real = shard.realisations_for_rank(rank, world)[0]
    w = wl.config4(N=args.N, which=which, realisation=real)
    K, n, P = w.K, w.n_points, w.n_pairs
    units_per_step = w.units

    series = torch.as_tensor(w.series).to(dev)
    buf = rqa.SweepBuffers.allocate(series, w.m, w.tau, K)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        rqa.rqa_eps_for_rr(buf.view, w.norm, w.rr, buf.eps, buf.count, buf.rr, buf.ws)
        if ev:
            ev[1].record(stream)
        rqa.rqa_line_hist(buf.view, w.norm, buf.eps, buf.hist, buf.ws)
        if ev:
            ev[2].record(stream)
        rqa.rqa_det_avg(buf.hist, 2, buf.det, buf.det_mean)
        if ev:
            ev[3].record(stream)

    for _ in range(args.warmup):
        step()
        flush.fill_(1)
    torch.cuda.synchronize()
    rqa.rqa_workspace_status(buf.ws)

    events = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    shard.barrier(world)
    torch.cuda.synchronize()
    if rank == 0:
        sampler.start()
    launches0 = rqa.rqa_launch_count()
    for it in range(args.steps):
        step(events[it])
        flush.fill_(it & 1)                                            # L2 flush between timed iterations
    torch.cuda.synchronize()
    launches = rqa.rqa_launch_count() - launches0
    shard.barrier(world)
    clocks = sampler.stop() if rank == 0 else None

    t_sel = [e[0].elapsed_time(e[1]) for e in events]
    t_line = [e[1].elapsed_time(e[2]) for e in events]
    t_det = [e[2].elapsed_time(e[3]) for e in events]
    t_step = [e[0].elapsed_time(e[3]) for e in events]
    total_ms = sum(t_step)
    value, max_ms = shard.whole_job_throughput(units_per_step * args.steps, total_ms, world, dev)

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region)
    hs = torch.as_tensor(w.series).pin_memory()
    h_eps = torch.empty((w.batch, K), dtype=torch.float32).pin_memory()
    h_cnt = torch.empty((w.batch, K), dtype=torch.int64).pin_memory()
    h_rr = torch.empty((w.batch, K), dtype=torch.float64).pin_memory()
    h_det = torch.empty((w.batch, K), dtype=torch.float64).pin_memory()
    h_mean = torch.empty((w.batch,), dtype=torch.float64).pin_memory()
    h_hist = torch.empty((w.batch, K, n), dtype=torch.int64).pin_memory()
    sws = torch.empty(rqa.rqa_sweep_workspace_bytes(w.N, w.batch, w.m, w.tau, K), dtype=torch.uint8, device=dev)
    e2e_steps = max(1, min(args.steps, 5))
    rqa.rqa_sweep_host(hs, w.m, w.tau, w.norm, w.rr, 2, h_eps, h_cnt, h_rr, h_det, h_mean, h_hist, sws)
    shard.barrier(world)
    torch.cuda.synchronize()
    e2e_ms = 0.0
    for it in range(e2e_steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        rqa.rqa_sweep_host(hs, w.m, w.tau, w.norm, w.rr, 2, h_eps, h_cnt, h_rr, h_det, h_mean, h_hist, sws)
        b.record(stream)
        torch.cuda.synchronize()
        e2e_ms += a.elapsed_time(b)
        flush.fill_(it & 1)
    e2e_value, _ = shard.whole_job_throughput(units_per_step * e2e_steps, e2e_ms, world, dev)
    h2d = hs.numel() * 4
    d2h = h_eps.numel() * 4 + h_cnt.numel() * 8 + h_rr.numel() * 8 + h_det.numel() * 8 + h_mean.numel() * 8 + h_hist.numel() * 8

    if rank != 0:
        return 0

    peaks, peak_kind = measured_peaks()
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    peak_lane = SM_COUNT * LANES_PER_SM_CLK * sm_max_mhz * 1e6                      # lane-instr / s
    line_ms = statistics.mean(t_line)
    alg_line = w.batch * P * line_scan_lane_instr_per_cell(w.m, K)                   # per rqa_line_hist call
    achieved = alg_line / (line_ms * 1e-3)
    roofline = {"bound": "alu", "kernel": "rqa_line_hist (diagonal scan)", "achieved": achieved / 1e12, "peak": peak_lane / 1e12,
                "unit": "Tlane-instr/s", "frac": achieved / peak_lane,
                "traffic": (NCU_LINE_SCAN_DRAM_BYTES_PER_SERIES * w.batch) if (w.N == 100000 and K == 20) else None,
                "traffic_unit": "bytes per launch (ncu dram read+write, profiles/r1k_ncu_line_scan.md, x batch)",
                "peak_source": f"148 SM x 128 lanes/clk x {sm_max_mhz:.0f} MHz ({peak_kind} sm_max_mhz)",
                "algorithmic_lane_instr_per_cell": line_scan_lane_instr_per_cell(w.m, K),
                "avg_launch_ms": line_ms}

    cpu_baseline = None
    if not args.no_cpu_baseline:
        from oracle import rqa_oracle
        rqa_oracle.build()
        cores = rqa_oracle.max_threads()
        u, dt = oracle_sample_run(w.series[-1], w.m, w.tau, w.rr, w.norm, 2, args.cpu_sample, 0)
        cpu_baseline = {"value": u / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
                        "sample": f"first {args.cpu_sample} points of the last series of the workload, K={K}, whole path"}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": w.name, "series": [f"{l['signal']}@snr{l['snr']}" for l in w.labels], "N": w.N, "m": w.m,
                      "tau": w.tau, "K": K, "norm": "max", "l_min": 2, "batch": w.batch, "cells_per_series": P,
                      "l2": "flushed between timed iterations (256 MiB fill)", "parallelism": f"series-sharded x{world}"},
           "breakdown_ms": {"rqa_eps_for_rr": statistics.mean(t_sel), "rqa_line_hist": line_ms,
                            "rqa_det_avg": statistics.mean(t_det), "step_min": min(t_step), "step_median": statistics.median(t_step)},
           "roofline": roofline, "cpu_baseline": cpu_baseline,
           "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps},
           "gpu_launches": int(launches), "clocks": clocks}
    print(json.dumps(out), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--series", default="all", help="'all' or comma-separated indices into config4's five series")
    ap.add_argument("--N", type=int, default=100000, help="series length (the metric is quoted at the default 1e5)")
    ap.add_argument("--cpu-sample", type=int, default=12000, help="points of the cpu_baseline sample")
    ap.add_argument("--ref-sample", type=int, default=5000, help="points per step of the --impl reference arm")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
