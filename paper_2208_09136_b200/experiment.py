"""The paper's experiment on one group of its grid: ten series of ascending SNR x R realisations, the
K = 99 integer-percent recurrence rates, DET_RR (Eq. 4) and the averaged DET_{RR*} (Eq. 5) for every RR*, and the sorting
rate S (Eq. 6) of both measures at every RR*.  Call chain only (rqa_eps_for_rr -> rqa_line_hist -> rqa_det_avg ->
rqa_det_prefix_avg -> rqa_sorting_rate_host, one batched call each); no arithmetic of the method lives here.
Reproducing the paper's Tables 1-2 is out of scope (they need the authors' seeds and RobPer's generator): the series
come from workloads.paper_group."""
from __future__ import annotations

import numpy as np

from . import binding as B
from .api import averaged_rqa


def sorting_experiment(workload, l_min: int = 2, buffers=None):
    """workload: workloads.paper_group(...) — rows ordered realisation*10 + snr_index, ascending SNR.
    -> {"det": [R*10][K] DET_RR, "det_avg": [R*10][K] averaged DET_{RR*}, "S_det": [K], "S_avg": [K] sorting rates in
    [0, 1] (1 = sorted by SNR in every realisation), "buffers": the SweepBuffers (device results)}."""
    import torch
    w = workload
    assert w.batch % 10 == 0, "a group holds ten SNRs per realisation"
    series = torch.as_tensor(w.series).cuda()
    buf = averaged_rqa(series, w.m, w.tau, w.rr, w.norm, l_min, buffers=buffers)
    prefix = torch.empty_like(buf.det)
    B.rqa_det_prefix_avg(buf.det, prefix)
    torch.cuda.synchronize()
    det, avg = buf.det.cpu().numpy(), prefix.cpu().numpy()
    R = w.batch // 10
    s_det = np.array([B.rqa_sorting_rate_host(det[:, k].reshape(R, 10)) for k in range(w.K)])
    s_avg = np.array([B.rqa_sorting_rate_host(avg[:, k].reshape(R, 10)) for k in range(w.K)])
    return {"det": det, "det_avg": avg, "S_det": s_det, "S_avg": s_avg, "buffers": buf}
