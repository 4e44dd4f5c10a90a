"""Convenience layer: allocate the output tensors and call the four C-ABI entry points in order.
No arithmetic of the method lives here."""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import binding as B


@dataclass
class SweepBuffers:
    """Device buffers for one shape (batch, N, m, tau, K); reusable across calls."""
    view: object
    eps: object
    count: object
    rr: object
    hist: object
    det: object
    det_mean: object
    ws: object

    @staticmethod
    def allocate(series, m: int, tau: int, K: int, theiler: int = 0, options=None):
        import torch
        if series.dim() == 1:
            series = series.unsqueeze(0)
        batch, N = series.shape
        view = B.rqa_embed(series, m, tau, theiler=theiler)
        n = int(view.n_points)
        dev = series.device
        return SweepBuffers(
            view=view,
            eps=torch.empty((batch, K), dtype=torch.float32, device=dev),
            count=torch.empty((batch, K), dtype=torch.int64, device=dev),
            rr=torch.empty((batch, K), dtype=torch.float64, device=dev),
            hist=torch.empty((batch, K, n), dtype=torch.int64, device=dev),
            det=torch.empty((batch, K), dtype=torch.float64, device=dev),
            det_mean=torch.empty((batch,), dtype=torch.float64, device=dev),
            ws=torch.empty(B.rqa_workspace_bytes(view, K, options), dtype=torch.uint8, device=dev),
        )


def averaged_rqa(series, m: int, tau: int, rr, norm: int = B.RQA_NORM_MAX, l_min: int = 2, buffers: SweepBuffers = None,
                 check: bool = True, theiler: int = 0, options=None):
    """series: float32 CUDA tensor [batch][N] or [N].  Runs rqa_embed (view) -> rqa_eps_for_rr -> rqa_line_hist ->
    rqa_det_avg on the current stream and returns the SweepBuffers holding the results (device tensors).
    With check=True the stream is synchronised and device-side errors (non-finite input) are raised.
    theiler = w > 1: only pairs with j - i >= w (rqa_points.theiler); buffers must have been allocated for the same w
    and the same `options` (rqa_options: expert knobs, or the share of a call split over several GPUs)."""
    rr = np.ascontiguousarray(rr, dtype=np.float64)
    if series.dim() == 1:
        series = series.unsqueeze(0)
    buf = buffers if buffers is not None else SweepBuffers.allocate(series, m, tau, len(rr), theiler, options)
    if buffers is not None:
        buf.view = B.rqa_embed(series, m, tau, theiler=theiler)
    B.rqa_eps_for_rr(buf.view, norm, rr, buf.eps, buf.count, buf.rr, buf.ws, options=options)
    B.rqa_line_hist(buf.view, norm, buf.eps, buf.hist, buf.ws, options=options)
    B.rqa_det_avg(buf.hist, l_min, buf.det, buf.det_mean)
    if check:
        B.rqa_workspace_status(buf.ws)
    return buf
