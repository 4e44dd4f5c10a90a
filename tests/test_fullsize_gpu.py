"""Full-size parity (BASELINE.json north_star: "bit-exact eps_k / RR / P_k(l) against the oracle on all five configs"):
configs 4 and 5 at their stated sizes, in the launch configuration bench.py times, element by element against
expected values that the CPU oracle computed offline.

The expected values live in tests/golden/fullsize/*.json and were written by tests/golden/make_fullsize_golden.py,
which calls only oracle/ (full enumeration + std::sort for eps_k — 20 GB at N = 1e5 —, the naive per-diagonal run count
for all K histograms, the naive per-column run count for the vertical lines).  Nothing in them comes from the CUDA
path.  Each file carries the SHA-256 of the fp32 series it was computed from; the tests check that they feed the very
same input.  (Configs 1-3 are compared with the live oracle in test_parity_gpu.py.)
"""
import hashlib
import json
from pathlib import Path

import numpy as np
import pytest

from paper_2208_09136_b200 import workloads as wl

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

GOLDEN = Path(__file__).resolve().parent / "golden" / "fullsize"
CONFIG5_SLICE = [0, 1, 28, 31, 32, 34, 61, 63, 64, 67, 92, 95]      # as in make_fullsize_golden.py


def load_golden(config: str, series: int, y: np.ndarray, rr: np.ndarray):
    path = GOLDEN / f"{config}_s{series}.json"
    assert path.exists(), f"{path} missing: run tests/golden/make_fullsize_golden.py {config} {series}"
    rec = json.loads(path.read_text())
    assert rec["sha256"] == hashlib.sha256(np.ascontiguousarray(y).tobytes()).hexdigest(), "the golden file is for another input"
    assert [float.fromhex(h) for h in rec["rr"]] == [float(r) for r in rr], "the golden file is for another RR list"
    n, K = rec["n_points"], len(rec["rr"])

    def dense(sp):
        h = np.zeros((K, n), dtype=np.uint64)
        for k, rows in enumerate(sp):
            for l, c in rows:
                h[k, l] = c
        return h
    out = {"eps": np.array(rec["eps_bits"], dtype=np.uint32).view(np.float32), "count": np.array(rec["count"], dtype=np.uint64),
           "hist": dense(rec["hist"]) if "hist" in rec else None, "vhist": dense(rec["vhist"]) if "vhist" in rec else None}
    return out


def check_series(oracle, g, b, gold, n_pairs, l_mins, what):
    assert np.array_equal(g["eps"][b].view(np.uint32), gold["eps"].view(np.uint32)), f"{what}: eps"
    assert np.array_equal(g["count"][b], gold["count"]), f"{what}: count"
    assert np.array_equal(g["rr"][b], gold["count"].astype(np.float64) / float(n_pairs)), f"{what}: realised RR"
    assert gold["hist"] is not None, f"{what}: the golden file has no histograms"
    if not np.array_equal(g["hist"][b], gold["hist"]):
        bad = np.argwhere(g["hist"][b] != gold["hist"])
        k, l = bad[0]
        raise AssertionError(f"{what}: {len(bad)} histogram cells differ, first at k={k} l={l}: gpu {g['hist'][b][k, l]} "
                             f"oracle {gold['hist'][k, l]}")
    # the invariant that ties the two kernels together, on every row
    l = np.arange(gold["hist"].shape[1], dtype=np.uint64)
    assert np.array_equal((g["hist"][b] * l).sum(axis=1), gold["count"]), f"{what}: sum l*P(l) = C"
    for l_min, det, mean in l_mins:
        od, om = oracle.det_avg(gold["hist"], l_min)
        assert np.max(np.abs(det[b] - od)) <= 1e-12 and abs(mean[b] - om) <= 1e-12, f"{what}: DET at l_min={l_min}"


def test_config4_all_five_series_bench_call(rqa, oracle):
    """The headline workload exactly as bench.py runs it: ONE batched call over the five N = 1e5 series (logistic and
    Lorenz at SNR 1 and 0.1, white noise), K = 20.  Every series: eps_k, C_k, RR_k and all 20 histograms element by
    element (99 998 bins each) against the stored oracle results."""
    import torch
    w = wl.config4()
    s = torch.as_tensor(w.series).cuda()
    buf = rqa.averaged_rqa(s, w.m, w.tau, w.rr, w.norm, 2)
    torch.cuda.synchronize()
    g = {"eps": buf.eps.cpu().numpy(), "count": buf.count.cpu().numpy().view(np.uint64), "rr": buf.rr.cpu().numpy(),
         "hist": buf.hist.cpu().numpy().view(np.uint64)}
    det, mean = buf.det.cpu().numpy(), buf.det_mean.cpu().numpy()
    for b in range(w.batch):
        gold = load_golden("config4", b, w.series[b], w.rr)
        check_series(oracle, g, b, gold, w.n_pairs, [(2, det, mean)], f"config4 series {b} {w.labels[b]}")


def test_config5_one_call_of_96_series(rqa, oracle):
    """Config 5 as ONE call of 96 series of N = 2e4, K = 32 (m = 5, tau = 2): a 12-series slice (4 per signal type, both
    ends of the SNR range) element by element against the stored oracle results, DET at l_min = 2 and 3; the other 84
    series through the invariants that hold without an oracle."""
    import torch
    w = wl.config5()
    assert (w.batch, w.N, w.K) == (96, 20000, 32)
    s = torch.as_tensor(w.series).cuda()
    buf = rqa.averaged_rqa(s, w.m, w.tau, w.rr, w.norm, 2)
    det3 = torch.empty_like(buf.det)
    mean3 = torch.empty_like(buf.det_mean)
    rqa.rqa_det_avg(buf.hist, 3, det3, mean3)
    torch.cuda.synchronize()
    g = {"eps": buf.eps.cpu().numpy(), "count": buf.count.cpu().numpy().view(np.uint64), "rr": buf.rr.cpu().numpy()}
    det2, mean2, det3, mean3 = buf.det.cpu().numpy(), buf.det_mean.cpu().numpy(), det3.cpu().numpy(), mean3.cpu().numpy()
    l = torch.arange(w.n_points, device="cuda", dtype=torch.int64)
    sums = (buf.hist * l).sum(dim=2).cpu().numpy().view(np.uint64)
    assert np.array_equal(sums, g["count"]), "sum l*P(l) = C on all 96 x 32 rows"
    ranks = np.array([oracle.rank(r, w.n_pairs) for r in w.rr], dtype=np.uint64)
    assert np.all(g["count"] >= ranks[None, :]) and np.all(np.diff(g["eps"], axis=1) >= 0)
    g["hist"] = {}
    for b in CONFIG5_SLICE:
        g["hist"][b] = buf.hist[b].cpu().numpy().view(np.uint64)
        gold = load_golden("config5", b, w.series[b], w.rr)
        check_series(oracle, g, b, gold, w.n_pairs, [(2, det2, mean2), (3, det3, mean3)], f"config5 series {b} {w.labels[b]}")


def vert_call(rqa, s, w, eps):
    import torch
    from paper_2208_09136_b200 import binding as B
    view = B.rqa_embed(s, w.m, w.tau)
    vh = torch.empty((s.shape[0], w.K, w.n_points), dtype=torch.int64, device="cuda")
    ws = torch.empty(B.rqa_workspace_bytes(view, w.K), dtype=torch.uint8, device="cuda")
    B.rqa_vert_hist(view, w.norm, eps, vh, ws)
    B.rqa_workspace_status(ws)
    return vh


def test_config5_vertical_lines_one_call_of_96_series(rqa, oracle):
    """rqa_vert_hist on config 5 as ONE call of 96 series (N = 2e4, K = 32) at the stored oracle thresholds: the
    12-series slice element by element against the stored oracle vertical-line histograms, LAM / TT against the oracle's
    reduction of them; all 96 x 32 rows through sum_v v*P(v) = 2*C."""
    import torch
    w = wl.config5()
    s = torch.as_tensor(w.series).cuda()
    buf = rqa.averaged_rqa(s, w.m, w.tau, w.rr, w.norm, 2)
    vh = vert_call(rqa, s, w, buf.eps)
    lam = torch.empty_like(buf.det)
    tt = torch.empty_like(buf.det)
    rqa.rqa_lam_tt(vh, 2, lam, tt)
    v = torch.arange(w.n_points, device="cuda", dtype=torch.int64)
    sums = (vh * v).sum(dim=2).cpu().numpy().view(np.uint64)
    assert np.array_equal(sums, 2 * buf.count.cpu().numpy().view(np.uint64)), "sum v*P(v) = 2C on all 96 x 32 rows"
    lam, tt = lam.cpu().numpy(), tt.cpu().numpy()
    for b in CONFIG5_SLICE:
        gold = load_golden("config5", b, w.series[b], w.rr)
        assert gold["vhist"] is not None
        assert np.array_equal(buf.eps[b].cpu().numpy().view(np.uint32), gold["eps"].view(np.uint32))
        got = vh[b].cpu().numpy().view(np.uint64)
        if not np.array_equal(got, gold["vhist"]):
            bad = np.argwhere(got != gold["vhist"])
            raise AssertionError(f"config5 series {b}: {len(bad)} vertical-histogram cells differ, first at {bad[0]}")
        ol, ot = oracle.lam_tt(gold["vhist"], 2)
        assert np.max(np.abs(lam[b] - ol)) <= 1e-12 and np.max(np.abs(tt[b] - ot)) <= 1e-9 * max(1.0, float(np.max(ot)))


def test_config4_vertical_lines_full_size(rqa, oracle):
    """rqa_vert_hist at N = 1e5 (1e10 cells per series and threshold set): the series that have a stored oracle
    vertical-line histogram element by element; all five through sum_v v*P(v) = 2*C."""
    import torch
    w = wl.config4()
    s = torch.as_tensor(w.series).cuda()
    buf = rqa.averaged_rqa(s, w.m, w.tau, w.rr, w.norm, 2)
    vh = vert_call(rqa, s, w, buf.eps)
    v = torch.arange(w.n_points, device="cuda", dtype=torch.int64)
    sums = (vh * v).sum(dim=2).cpu().numpy().view(np.uint64)
    assert np.array_equal(sums, 2 * buf.count.cpu().numpy().view(np.uint64))
    checked = 0
    for b in range(w.batch):
        gold = load_golden("config4", b, w.series[b], w.rr)
        if gold["vhist"] is None:
            continue
        assert np.array_equal(vh[b].cpu().numpy().view(np.uint64), gold["vhist"]), f"config4 series {b}"
        checked += 1
    assert checked == w.batch, "a stored vertical-line histogram is missing: run make_fullsize_golden.py config4 <s> --stage vhist"
