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


def grid_groups(N: int, n_real: int = 10, K: int = 99):
    """The nine groups of the paper's grid at one series length: 3 dynamics x 3 SNR levels, each 10 SNRs x
    n_real realisations."""
    from . import workloads as wl
    return [wl.paper_group(sig, level, N, n_real=n_real, K=K) for sig in ("sine", "logistic", "lorenz") for level in (0.1, 1.0, 10.0)]


class GridRunner:
    """Stream-level overlap for the grid: every library call is asynchronous on the caller's stream and
    the library keeps no global state, so independent groups run on separate CUDA streams with their own buffers.  A group
    of 100 short series fills only part of the GPU (one block per series on the short-series path); several groups in
    flight fill the rest.  `run()` enqueues every group's call chain round robin over `streams` streams and synchronises
    once at the end; results are the same device buffers a sequential run fills."""

    def __init__(self, groups, streams: int = 4, l_min: int = 2):
        import torch
        from .api import SweepBuffers
        self.groups, self.l_min = groups, l_min
        self.streams = [torch.cuda.Stream() for _ in range(max(1, streams))]
        self.series = [torch.as_tensor(w.series).cuda() for w in groups]
        self.buffers = [SweepBuffers.allocate(s, w.m, w.tau, w.K) for s, w in zip(self.series, groups)]
        self.prefix = [torch.empty_like(b.det) for b in self.buffers]
        torch.cuda.synchronize()

    def run(self):
        import torch
        for g, (w, s, buf, pre) in enumerate(zip(self.groups, self.series, self.buffers, self.prefix)):
            with torch.cuda.stream(self.streams[g % len(self.streams)]):
                averaged_rqa(s, w.m, w.tau, w.rr, w.norm, self.l_min, buffers=buf, check=False)
                B.rqa_det_prefix_avg(buf.det, pre)
        for st in self.streams:
            st.synchronize()
        return self.buffers, self.prefix
