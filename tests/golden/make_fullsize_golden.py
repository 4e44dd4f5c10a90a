#!/usr/bin/env python
"""Writes the stored expected values of the FULL-SIZE parity tests (tests/test_fullsize_gpu.py).

Calls ONLY the CPU oracle (oracle/rqa_oracle.py -> oracle/rqa_oracle.cpp) on the seeded inputs of
paper_2208_09136_b200/workloads.py (input generators only; no method arithmetic).  Nothing here touches the CUDA
path: no expected value comes from it.

    python tests/golden/make_fullsize_golden.py config4 <series 0..4> [--stage eps|hist|vhist|all] [--threads T]
    python tests/golden/make_fullsize_golden.py config5 <series 0..95> [--stage ...]

One text file per series, tests/golden/fullsize/<config>_s<index>.json:
  sha256      of the fp32 series bytes (the test checks it feeds the same input)
  rr          the K target recurrence rates as C99 hex floats (reading S5: both sides get the same doubles)
  eps_bits    uint32 bit patterns of eps_k = the ceil(rr_k*P)-th smallest distance: FULL enumeration + std::sort
              (oracle.eps_for_rr; 20 GB at N = 1e5), PAPER.md:78 with readings S4-S6
  count       C_k = #{d <= eps_k}
  hist        P_k(l) of all K thresholds (oracle.line_hist), sparse: per k a list of [l, count]
  vhist       vertical-line histogram (oracle.vert_hist, reading S19), sparse, same layout
Stages are separate because the sort is single-threaded (about 12 minutes per N = 1e5 series) and the histograms are
OpenMP loops over diagonals / columns; a stage adds its keys to the file the previous stage wrote.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from oracle import rqa_oracle as oracle          # noqa: E402
from paper_2208_09136_b200 import workloads as wl  # noqa: E402  (seeded input generators only)

OUT = Path(__file__).resolve().parent / "fullsize"

# config 5: the 12-series slice of the 96-series call that the test compares (4 per signal type: both ends of the
# SNR range, two realisations each).  Index = (signal*8 + snr_index)*4 + realisation.
CONFIG5_SLICE = [0, 1, 28, 31, 32, 34, 61, 63, 64, 67, 92, 95]


def workload(config: str):
    if config == "config4":
        return wl.config4()
    if config == "config5":
        return wl.config5()
    raise SystemExit(f"unknown config {config}")


def sparse(h: np.ndarray):
    out = []
    for k in range(h.shape[0]):
        nz = np.nonzero(h[k])[0]
        out.append([[int(l), int(h[k, l])] for l in nz])
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["config4", "config5"])
    ap.add_argument("series", type=int)
    ap.add_argument("--stage", default="all", choices=["eps", "hist", "vhist", "all"])
    ap.add_argument("--threads", type=int, default=0)
    a = ap.parse_args()
    w = workload(a.config)
    y = np.ascontiguousarray(w.series[a.series])
    path = OUT / f"{a.config}_s{a.series}.json"
    OUT.mkdir(exist_ok=True)
    rec = json.loads(path.read_text()) if path.exists() else {}
    sha = hashlib.sha256(y.tobytes()).hexdigest()
    if rec and rec["sha256"] != sha:
        raise SystemExit("input changed: delete the stale golden file first")
    rec.update({"workload": w.name, "series": a.series, "label": w.labels[a.series], "sha256": sha, "N": int(w.N),
                "m": int(w.m), "tau": int(w.tau), "norm": int(w.norm), "n_points": int(w.n_points),
                "rr": [float(r).hex() for r in w.rr]})
    rec.setdefault("seconds", {})
    if a.stage in ("eps", "all") and "eps_bits" not in rec:
        t = time.perf_counter()
        eps, cnt, _ = oracle.eps_for_rr(y, w.m, w.tau, w.rr, w.norm)
        rec["eps_bits"] = [int(b) for b in eps.view(np.uint32)]
        rec["count"] = [int(c) for c in cnt]
        rec["seconds"]["eps"] = time.perf_counter() - t
        path.write_text(json.dumps(rec) + "\n")
    if "eps_bits" not in rec:
        raise SystemExit("run --stage eps first")
    eps = np.array(rec["eps_bits"], dtype=np.uint32).view(np.float32)
    if a.stage in ("hist", "all") and "hist" not in rec:
        t = time.perf_counter()
        rec["hist"] = sparse(oracle.line_hist(y, w.m, w.tau, eps, w.norm, threads=a.threads))
        rec["seconds"]["hist"] = time.perf_counter() - t
        path.write_text(json.dumps(rec) + "\n")
    if a.stage in ("vhist", "all") and "vhist" not in rec:
        t = time.perf_counter()
        rec["vhist"] = sparse(oracle.vert_hist(y, w.m, w.tau, eps, w.norm, threads=a.threads))
        rec["seconds"]["vhist"] = time.perf_counter() - t
        path.write_text(json.dumps(rec) + "\n")
    print(path, {k: round(v, 1) for k, v in rec["seconds"].items()})


if __name__ == "__main__":
    main()
