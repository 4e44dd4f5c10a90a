#!/usr/bin/env python
"""bench.py — headline measurement of the averaged-RQA hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--mode series|split]

Metric (BASELINE.json): recurrence cells x thresholds per second at N = 1e5, K = 20 recurrence rates.
Workload at N=1 GPU: BASELINE.json configs[3] ("config4"): five series of N = 1e5 (logistic and Lorenz x at
SNR 1 and 0.1, white noise), m = 3, tau = 1, max norm, K = 20 log-spaced RRs 0.001..0.2, l_min = 2.
A step = one pass of the whole hot path (rqa_eps_for_rr -> rqa_line_hist -> rqa_det_avg; the embedding is a
strided view) over the batch of five series, 5 x 9.9995e10 = 5.0e11 cells x thresholds.

--gpus N > 1 without a torchrun environment: bench.py starts the N ranks itself (one process per GPU, NCCL over
127.0.0.1); under torchrun it is one of the ranks.  --mode series (default): every rank sweeps its own realisation of
the five series, no data-path collective (weak scaling).  --mode split: ONE batch of five series is split over the
ranks tile by tile (rqa_options.part_index/part_count), exact counters all-reduced by NCCL (strong scaling).

Prints ONE JSON line (rank 0).  See DESIGN.md "Roofline and measurement" for every field.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import socket
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

# ncu counters of every kernel of ONE step of this very workload (written by the command in profiles/step_counters.md:
# `ncu --metrics ... python bench.py --profile-step`).  Instruction counts are a property of the kernels and the
# seeded input, not of the run; the durations used below are measured live.
STEP_COUNTERS = ROOT / "profiles" / "step_counters.csv"
NCU_METRICS = ["gpu__time_duration.sum", "smsp__inst_executed.sum", "smsp__thread_inst_executed.sum",
               "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
               "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
               "dram__bytes_read.sum", "dram__bytes_write.sum"]


# algorithmic lane-instructions per cell of the line-scan kernel: distance 2m-1 = 5, plus one
# threshold test and one run update per threshold = 2K.
def line_scan_lane_instr_per_cell(m: int, K: int) -> int:
    return (2 * m - 1) + 2 * K


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        return json.loads(p.read_text()), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def read_step_counters(path: Path = STEP_COUNTERS):
    """-> {short kernel name: {"launches", "ms", "warp_instr", "thread_instr", "issue_active_pct", "lsu_pct", "alu_pct",
    "warps_active_pct", "dram_bytes"}} summed / time-weighted over the launches of one step, or None."""
    if not path.exists():
        return None
    rows = list(csv.reader(path.read_text().splitlines()))
    try:
        hi = next(i for i, r in enumerate(rows) if r and r[0] == "ID")
    except StopIteration:
        return None
    h = rows[hi]
    kn, mn, mu, mv = h.index("Kernel Name"), h.index("Metric Name"), h.index("Metric Unit"), h.index("Metric Value")
    per_launch = {}
    for r in rows[hi + 1:]:
        if len(r) <= mv:
            continue
        name = r[kn]
        if "at::" in name or "cub::" in name:                 # torch's own kernels (fills): not part of the step
            continue
        short = name.split("(")[0].replace("void ", "").replace("rqa::", "").replace("<unnamed>::", "").replace("unnamed>::", "").strip()
        v = float(r[mv].replace(",", ""))
        unit = r[mu]
        scale = {"ns": 1e-6, "us": 1e-3, "usecond": 1e-3, "msecond": 1.0, "ms": 1.0, "nsecond": 1e-6, "second": 1e3,
                 "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0}.get(unit, 1.0)
        per_launch.setdefault((r[0], short), {})[r[mn]] = v * scale
    out = {}
    for (_, short), m in per_launch.items():
        k = out.setdefault(short, {"launches": 0, "ms": 0.0, "warp_instr": 0.0, "thread_instr": 0.0, "dram_bytes": 0.0,
                                   "_issue": 0.0, "_lsu": 0.0, "_alu": 0.0, "_warps": 0.0})
        t = m.get("gpu__time_duration.sum", 0.0)
        k["launches"] += 1
        k["ms"] += t
        k["warp_instr"] += m.get("smsp__inst_executed.sum", 0.0)
        k["thread_instr"] += m.get("smsp__thread_inst_executed.sum", 0.0)
        k["dram_bytes"] += m.get("dram__bytes_read.sum", 0.0) + m.get("dram__bytes_write.sum", 0.0)
        k["_issue"] += t * m.get("smsp__issue_active.avg.pct_of_peak_sustained_active", 0.0)
        k["_lsu"] += t * m.get("sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", 0.0)
        k["_alu"] += t * m.get("sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", 0.0)
        k["_warps"] += t * m.get("sm__warps_active.avg.pct_of_peak_sustained_active", 0.0)
    for k in out.values():
        t = k["ms"] or 1.0
        k["issue_active_pct"] = k.pop("_issue") / t
        k["lsu_pct"] = k.pop("_lsu") / t
        k["alu_pct"] = k.pop("_alu") / t
        k["warps_active_pct"] = k.pop("_warps") / t
    return out


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
def host_info():
    model, ram = "unknown", None
    try:
        for line in Path("/proc/cpuinfo").read_text().splitlines():
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
        for line in Path("/proc/meminfo").read_text().splitlines():
            if line.startswith("MemTotal"):
                ram = round(int(line.split()[1]) / 1048576.0, 1)
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model, "ram_gb": ram}


def oracle_sample_run(series, m, tau, rr, norm, l_min, n_sample, threads):
    """The oracle as it stands on a bounded sample (the first n_sample points of one series)."""
    from oracle import rqa_oracle
    y = np.ascontiguousarray(series[:n_sample])
    t0 = time.perf_counter()
    rqa_oracle.sweep(y, m, tau, rr, norm, l_min, threads=threads)
    dt = time.perf_counter() - t0
    units = rqa_oracle.n_pairs(len(y), m, tau) * len(rr)
    return units, dt


def sample_text(n, K):
    return (f"bounded SAMPLE, not the full workload and not extrapolated: the first {n} points of the white-noise series "
            f"of config4 (N=1e5), K={K}, whole path (brute-force distances + std::sort + naive line scan + DET)")


def cpu_baseline_block(w, n_sample, single_sample):
    from oracle import rqa_oracle
    rqa_oracle.build()
    cores = rqa_oracle.max_threads()
    y = w.series[-1]
    u, dt = oracle_sample_run(y, w.m, w.tau, w.rr, w.norm, 2, n_sample, 0)
    out = {"value": u / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt, "sample": sample_text(n_sample, w.K),
           "host": host_info()}
    if single_sample > 0:
        u1, dt1 = oracle_sample_run(y, w.m, w.tau, w.rr, w.norm, 2, single_sample, 1)
        out["single_thread"] = {"value": u1 / dt1, "unit": UNIT, "cores": 1, "seconds": dt1, "sample": sample_text(single_sample, w.K)}
    return out


def run_reference(args):
    rank, world, _ = shard.env_rank_world()
    if rank != 0:
        return 0
    from oracle import rqa_oracle
    rqa_oracle.build()
    w = wl.config4(which=[4])
    cores = rqa_oracle.max_threads()
    n_sample = args.cpu_sample
    for _ in range(args.warmup):
        oracle_sample_run(w.series[0], w.m, w.tau, w.rr, w.norm, 2, min(n_sample, 2000), 0)
    total_units, total_t = 0, 0.0
    for _ in range(args.steps):
        u, dt = oracle_sample_run(w.series[0], w.m, w.tau, w.rr, w.norm, 2, n_sample, 0)
        total_units += u
        total_t += dt
    value = total_units / total_t
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": "config4_long_N100000 (bounded sample per step)", "N": n_sample, "m": w.m, "tau": w.tau, "K": w.K,
                      "norm": "max", "l_min": 2},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_text(n_sample, w.K),
                            "host": host_info()},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def time_call(fn, repeats=5, warm=2):
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(repeats):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return statistics.median(ts), min(ts)


def other_configs(rqa):
    """Whole path (rqa_eps_for_rr + rqa_line_hist + rqa_det_avg) per call on the other BASELINE.json configs and on the
    many-short-series regime of the paper's grid, device-resident inputs, CUDA events, median of 5."""
    import torch
    out = []
    cases = [wl.config1(), wl.config2(), wl.config3(0), wl.config3(1), wl.config5(),
             wl.paper_group("logistic", 1.0, 100, n_real=90), wl.paper_group("logistic", 1.0, 1000, n_real=90),
             wl.paper_group("lorenz", 1.0, 1000, n_real=10, K=99), wl.paper_group("logistic", 1.0, 10000, n_real=10, K=99)]
    for w in cases:
        s = torch.as_tensor(w.series).cuda()
        buf = rqa.SweepBuffers.allocate(s, w.m, w.tau, w.K)

        def call():
            rqa.rqa_eps_for_rr(buf.view, w.norm, w.rr, buf.eps, buf.count, buf.rr, buf.ws)
            rqa.rqa_line_hist(buf.view, w.norm, buf.eps, buf.hist, buf.ws)
            rqa.rqa_det_avg(buf.hist, 2, buf.det, buf.det_mean)
        n0 = rqa.rqa_launch_count()
        call()
        launches = rqa.rqa_launch_count() - n0
        med, mn = time_call(call)
        rqa.rqa_workspace_status(buf.ws)
        out.append({"workload": w.name, "batch": w.batch, "N": w.N, "m": w.m, "tau": w.tau, "K": w.K,
                    "norm": "max" if w.norm == 0 else "euclid", "ms_per_call": med, "ms_min": mn, "value": w.units / (med * 1e-3),
                    "unit": UNIT, "gpu_launches_per_call": int(launches)})
        del buf, s
        torch.cuda.empty_cache()
    # stream-level overlap for the grid (row f4): the nine groups of one series length, one stream vs four
    from paper_2208_09136_b200 import experiment
    for N in (100, 1000):
        groups = experiment.grid_groups(N)
        units = sum(w.units for w in groups)
        res = {}
        for ns in (1, 4):
            runner = experiment.GridRunner(groups, streams=ns)
            med, mn = time_call(runner.run)
            res[ns] = med
            del runner
            torch.cuda.empty_cache()
        out.append({"workload": f"paper_grid_9groups_x100_N{N}", "batch": 900, "N": N, "K": 99, "ms_per_call": res[4],
                    "ms_one_stream": res[1], "streams": 4, "value": units / (res[4] * 1e-3), "unit": UNIT,
                    "note": "nine groups (3 dynamics x 3 SNR levels) of 100 series each, every group its own call chain; host "
                            "enqueue time is inside the interval"})
    return out


def run_ours(args):
    import torch

    import paper_2208_09136_b200 as rqa
    from paper_2208_09136_b200 import binding as B, parts

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    rank, world, local = shard.env_rank_world()
    if args.same_gpu:                                               # functional test of the multi-rank path on a 1-GPU box
        local = 0
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    shard.init_process_group(args.backend)
    rqa.load_library()
    split = args.mode == "split" and world > 1

    which = None if args.series == "all" else [int(s) for s in args.series.split(",")]
    real = 0 if split else shard.realisations_for_rank(rank, world)[0]
    w = wl.config4(N=args.N, which=which, realisation=real)
    K, n, P = w.K, w.n_points, w.n_pairs
    units_per_step = w.units / world if split else w.units          # this rank's share; the job total is summed over ranks

    series = torch.as_tensor(w.series).to(dev)
    stream = torch.cuda.current_stream()
    ev_count = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev_scan = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    part = dict(part_index=rank, part_count=world, reduce=parts.dist_reduce("cuda")) if split else {}
    o_sel = B.make_options(kernel_events=ev_count, **part)
    knobs = {}
    if args.line_knobs:                                             # expert knobs of the diagonal scan (profiles/r2_scan_knobs.md)
        nb, ch, sg = (int(x) for x in args.line_knobs.split(","))
        knobs = dict(line_buffers=nb, line_chunk=ch, line_segment=sg)
    o_line = B.make_options(kernel_events=ev_scan, **knobs, **part)
    buf = rqa.SweepBuffers.allocate(series, w.m, w.tau, K, options=o_line if knobs else o_sel)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        rqa.rqa_eps_for_rr(buf.view, w.norm, w.rr, buf.eps, buf.count, buf.rr, buf.ws, options=o_sel)
        if ev:
            ev[1].record(stream)
        rqa.rqa_line_hist(buf.view, w.norm, buf.eps, buf.hist, buf.ws, options=o_line)
        if ev:
            ev[2].record(stream)
        rqa.rqa_det_avg(buf.hist, 2, buf.det, buf.det_mean)
        if ev:
            ev[3].record(stream)

    if args.profile_step:                                            # one bare step for ncu (profiles/step_counters.md)
        step()
        torch.cuda.synchronize()
        rqa.rqa_workspace_status(buf.ws)
        return 0

    for _ in range(args.warmup):
        step()
        flush.fill_(1)
    torch.cuda.synchronize()
    rqa.rqa_workspace_status(buf.ws)

    events = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    t_count_k, t_scan_k = [], []
    sampler = ClockSampler(local)
    shard.barrier(world)
    torch.cuda.synchronize()
    if rank == 0:
        sampler.start()
    launches0 = rqa.rqa_launch_count()
    for it in range(args.steps):
        step(events[it])
        flush.fill_(it & 1)                                            # L2 flush between timed iterations
        # the two kernel-event pairs are reused every step: read them before the next step records them again
        # (the wait falls between two steps, outside every timed interval)
        ev_scan[1].synchronize()
        t_count_k.append(ev_count[0].elapsed_time(ev_count[1]))
        t_scan_k.append(ev_scan[0].elapsed_time(ev_scan[1]))
    torch.cuda.synchronize()
    launches = rqa.rqa_launch_count() - launches0
    shard.barrier(world)
    clocks = sampler.stop() if rank == 0 else None

    t_sel = [e[0].elapsed_time(e[1]) for e in events]
    t_line = [e[1].elapsed_time(e[2]) for e in events]
    t_det = [e[2].elapsed_time(e[3]) for e in events]
    t_step = [e[0].elapsed_time(e[3]) for e in events]
    total_ms = sum(t_step)
    value, max_ms = shard.whole_job_throughput(units_per_step * args.steps, total_ms, world, dev if args.backend == "nccl" else "cpu")

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e and not split:
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
        e2e_value, _ = shard.whole_job_throughput(units_per_step * e2e_steps, e2e_ms, world, dev if args.backend == "nccl" else "cpu")
        h2d = hs.numel() * 4
        d2h = h_eps.numel() * 4 + h_cnt.numel() * 8 + h_rr.numel() * 8 + h_det.numel() * 8 + h_mean.numel() * 8 + h_hist.numel() * 8
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps, "api": "rqa_sweep_host (C ABI, pinned host buffers)"}
        del sws, h_hist

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (the diagonal scan) and of the step
    peaks, peak_kind = measured_peaks()
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    peak_lane = SM_COUNT * LANES_PER_SM_CLK * sm_max_mhz * 1e6                      # lane-instr / s
    step_ms = statistics.mean(t_step)
    scan_ms, count_ms = statistics.mean(t_scan_k), statistics.mean(t_count_k)
    warp_cells = w.batch * P / 32.0                                                  # per full pass over the triangle
    alg = w.batch * P * line_scan_lane_instr_per_cell(w.m, K)
    counters = read_step_counters() if (w.N == 100000 and w.batch == 5 and not split) else None
    kernels = []

    def kernel_entry(label, key, live_ms):
        e = {"name": label, "ms": live_ms, "share_of_step": live_ms / step_ms}
        c = counters.get(key) if counters else None
        if c:
            e.update({"warp_instr": c["warp_instr"], "warp_instr_per_warp_cell": c["warp_instr"] / warp_cells,
                      "active_lanes_per_instr": c["thread_instr"] / c["warp_instr"] if c["warp_instr"] else None,
                      "issue_frac": c["warp_instr"] * 32 / (live_ms * 1e-3) / peak_lane,
                      "lane_frac": c["thread_instr"] / (live_ms * 1e-3) / peak_lane,
                      "ncu": {"ms": c["ms"], "issue_active_pct": c["issue_active_pct"], "lsu_pipe_pct": c["lsu_pct"],
                              "alu_pipe_pct": c["alu_pct"], "warps_active_pct": c["warps_active_pct"],
                              "dram_bytes": c["dram_bytes"], "launches": c["launches"]}})
        return e
    scan_key = next((k for k in (counters or {}) if k.startswith("line_scan_kernel")), None)
    count_key = next((k for k in (counters or {}) if k.startswith("sel_count_kernel")), None)
    kernels.append(kernel_entry("line_scan_kernel (rqa_line_hist)", scan_key, scan_ms))
    kernels.append(kernel_entry("sel_count_kernel (rqa_eps_for_rr)", count_key, count_ms))
    kernels.append({"name": "all other kernels of the step", "ms": step_ms - scan_ms - count_ms,
                    "share_of_step": (step_ms - scan_ms - count_ms) / step_ms})
    alg_achieved = alg / (scan_ms * 1e-3)
    roofline = {"bound": "alu", "kernel": "line_scan_kernel (the diagonal scan of rqa_line_hist)", "unit": "Tlane-instr/s",
                "peak": peak_lane / 1e12, "peak_source": f"148 SM x 128 lanes/clk x {sm_max_mhz:.0f} MHz ({peak_kind} sm_max_mhz)",
                "avg_launch_ms": scan_ms,
                "algorithmic": {"lane_instr_per_cell": line_scan_lane_instr_per_cell(w.m, K), "achieved": alg_achieved / 1e12,
                                "frac": alg_achieved / peak_lane,
                                "note": "SURVEY 8d's K-linear formulation (2m-1+2K per cell) / live kernel time: a statement about the "
                                        "algorithm (the kernel does K-independent work per cell), not a hardware utilisation"},
                "kernels": kernels}
    if counters and scan_key:
        k0 = kernels[0]
        total_instr = sum(c["warp_instr"] for c in counters.values())
        roofline.update({"achieved": k0["issue_frac"] * peak_lane / 1e12, "frac": k0["issue_frac"],
                         "frac_kind": "hardware issue slots: warp-instructions the kernel executes on this workload (ncu "
                                      "smsp__inst_executed.sum, profiles/step_counters.csv) x 32 / live kernel time / peak",
                         "lane_frac": k0["lane_frac"],
                         "step_issue_frac": total_instr * 32 / (step_ms * 1e-3) / peak_lane,
                         "traffic": counters[scan_key]["dram_bytes"],
                         "traffic_unit": "bytes per launch: ncu dram__bytes_read.sum + dram__bytes_write.sum of this kernel at this "
                                         "batch (profiles/step_counters.csv)",
                         "counters_source": "profiles/step_counters.csv (regenerate: profiles/step_counters.md)"})
    else:
        roofline.update({"achieved": alg_achieved / 1e12, "frac": alg_achieved / peak_lane,
                         "frac_kind": "algorithmic only: no ncu counter file for this workload", "traffic": None})

    cpu_baseline = None if args.no_cpu_baseline else cpu_baseline_block(w, args.cpu_sample, args.cpu_single_sample)
    others = None if (args.no_others or world > 1) else other_configs(rqa)

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "strong" if split else "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": w.name, "series": [f"{l['signal']}@snr{l['snr']}" for l in w.labels], "N": w.N, "m": w.m,
                      "tau": w.tau, "K": K, "norm": "max", "l_min": 2, "batch": w.batch, "cells_per_series": P,
                      "l2": "flushed between timed iterations (256 MiB fill)",
                      "parallelism": (f"one batch split over {world} ranks by tiles, NCCL all-reduce of exact counters" if split
                                      else f"series-sharded x{world}, no data-path collective")},
           "breakdown_ms": {"rqa_eps_for_rr": statistics.mean(t_sel), "rqa_line_hist": statistics.mean(t_line),
                            "rqa_det_avg": statistics.mean(t_det), "step_min": min(t_step), "step_median": statistics.median(t_step)},
           "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e,
           "gpu_launches": int(launches), "clocks": clocks, "other_configs": others}
    if args.same_gpu:
        out["functional_test_only"] = "all ranks shared one GPU: not a measurement"
    print(json.dumps(out), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ launch
def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start one process per GPU (RANK/LOCAL_RANK/WORLD_SIZE, rendezvous on
    127.0.0.1), wait for all of them; rank 0 prints the JSON line."""
    port = free_port()
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(Path(__file__).resolve()), *sys.argv[1:]], env=env))
    rc = 0
    for p in procs:
        rc = rc or p.wait()
    return rc


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="series", choices=["series", "split"], help="multi-GPU: shard by series (weak) or split one batch (strong)")
    ap.add_argument("--series", default="all", help="'all' or comma-separated indices into config4's five series")
    ap.add_argument("--N", type=int, default=100000, help="series length (the metric is quoted at the default 1e5)")
    ap.add_argument("--cpu-sample", type=int, default=10000, help="points of the oracle's sample (cpu_baseline and --impl reference)")
    ap.add_argument("--cpu-single-sample", type=int, default=4000, help="points of the single-thread oracle sample (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the secondary timings of the other configs")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--profile-step", action="store_true", help="run ONE bare step and exit (for ncu; prints nothing)")
    ap.add_argument("--line-knobs", default="", help="'buffers,chunk,segment' for rqa_line_hist (rqa_options.line_buffers, "
                                                     "line_chunk, line_segment; 0 = automatic): the knob sweep of profiles/r2_scan_knobs.md")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="torch.distributed backend of the ranks")
    ap.add_argument("--same-gpu", action="store_true",
                    help="FUNCTIONAL TEST ONLY: all ranks share cuda:0 (use with --backend gloo; NCCL refuses one device "
                         "twice).  The ranks take turns on the device: the number printed is not a measurement.")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE')}", file=sys.stderr)
        return 2
    if args.warmup < 3 and not args.profile_step:
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
