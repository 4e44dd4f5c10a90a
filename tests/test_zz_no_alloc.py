"""rqa_line_hist_static — rqa_line_hist for callers that cannot allocate device memory (include/rqa.h): the scratch is a
static device array of RQA_STATIC_SCRATCH_BYTES inside librqa.so, the caller passes only inputs and outputs.

The entry point runs the kernels of rqa_line_hist, so its histograms must equal the existing path's bit for bit (the bar
of tests/test_parity_gpu.py for integer outputs), on calls made back to back on the shared scratch.  This file is named
to be collected LAST (`pytest --collect-only`): the suite runs with `pytest -x`, and a failure here must not hide
another test.  It passes alone in a fresh process and after the other tests (nothing here depends on earlier state:
the first call of a process does the per-device set-up itself).
"""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

from paper_2208_09136_b200 import workloads as wl


def _existing_path(rqa, w):
    """thresholds and histograms of a workload from the existing calls (caller workspace)"""
    import torch
    s = torch.as_tensor(np.ascontiguousarray(np.atleast_2d(w.series), dtype=np.float32)).cuda()
    buf = rqa.averaged_rqa(s, w.m, w.tau, w.rr, w.norm)
    torch.cuda.synchronize()
    return s, buf


def _cases():
    # config 3: six series of 10^4 points, K = 20 — the tiled scan with stitched segments, 113 of the 128 MiB of scratch;
    # config 2: five series of 10^3 points — the scan at a few tiles; config 1: the one-block short-series kernel
    return [wl.config3(0), wl.config2(), wl.config3(1), wl.config1()]


@pytest.mark.gpu
def test_static_scratch_matches_existing_path_on_calls_in_a_row(rqa):
    import torch
    prepared = []
    for w in _cases():
        s, buf = _existing_path(rqa, w)
        out = torch.empty_like(buf.hist)
        prepared.append((w, s, buf, out))
    # three rounds over all cases, back to back on one stream, no synchronisation in between: every call starts on the
    # scratch as the previous (different) call left it, and on an output buffer full of garbage.  Round 0 is also the
    # set-up: cudaGetSymbolAddress, and the driver's lazy loading of every kernel the cases use (which takes device
    # memory the first time a kernel is launched in a process, whoever launches it); from then on the free device memory
    # must not move.
    free = []
    for rnd in range(3):
        for w, s, buf, out in prepared:
            out.fill_(-0x0123456789ABCDF)
            rqa.rqa_line_hist_static(buf.view, w.norm, buf.eps, out)
        torch.cuda.synchronize()
        for w, s, buf, out in prepared:
            got, want = out.cpu().numpy().view(np.uint64), buf.hist.cpu().numpy().view(np.uint64)
            if not np.array_equal(got, want):
                bad = np.argwhere(got != want)
                raise AssertionError(f"{w.name}, round {rnd}: {len(bad)} of {got.size} histogram cells differ from "
                                     f"rqa_line_hist, first at {tuple(bad[0])}: {got[tuple(bad[0])]} vs {want[tuple(bad[0])]}")
            # the invariant tying the histogram to the thresholds' counts: sum_l l*P_k(l) = C_k
            l = np.arange(got.shape[-1], dtype=np.uint64)
            assert np.array_equal((got * l).sum(axis=-1), buf.count.cpu().numpy().view(np.uint64))
        free.append(torch.cuda.mem_get_info()[0])
    assert free[2] == free[1], f"calls after the set-up round changed the free device memory: {free}"


@pytest.mark.gpu
def test_static_scratch_twice_on_the_same_input(rqa):
    """the plainest reading of 'two calls in a row': same input, same output buffer, results equal both times"""
    import torch
    w = wl.config3(0)
    s, buf = _existing_path(rqa, w)
    want = buf.hist.cpu().numpy()
    out = torch.zeros_like(buf.hist)
    for call in range(2):
        rqa.rqa_line_hist_static(buf.view, w.norm, buf.eps, out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), want), f"call {call}"


@pytest.mark.gpu
def test_static_scratch_takes_a_large_batch_of_moderate_series(rqa):
    """A batch that runs as one block per series needs no scratch beyond the status block, whatever its size: a group
    of the paper's grid (900 series of 10^3 points, K = 99) goes through the static entry point, twice in a row."""
    import torch
    w = wl.paper_group("logistic", 1.0, 1000, n_real=90)
    s, buf = _existing_path(rqa, w)
    out = torch.empty_like(buf.hist)
    for call in range(2):
        out.fill_(-1)
        rqa.rqa_line_hist_static(buf.view, w.norm, buf.eps, out)
        torch.cuda.synchronize()
        assert torch.equal(out, buf.hist), f"call {call}"


@pytest.mark.gpu
def test_static_scratch_rejects_a_shape_beyond_the_maximum_on_the_gpu(rqa):
    import torch
    N = 100_000                                                 # config 4's length: 207 MiB of scratch for one series
    s = torch.zeros((1, N), dtype=torch.float32, device="cuda")
    view = rqa.rqa_embed(s, 3, 1)
    eps = torch.full((1, 20), 0.5, dtype=torch.float32, device="cuda")
    hist = torch.full((1, 20, int(view.n_points)), 7, dtype=torch.int64, device="cuda")
    launches = rqa.rqa_launch_count()
    with pytest.raises(rqa.RqaError) as e:
        rqa.rqa_line_hist_static(view, 0, eps, hist)
    assert e.value.status == rqa.RQA_ERR_UNSUPPORTED and "RQA_STATIC_SCRATCH_BYTES" in str(e.value)
    assert rqa.rqa_launch_count() == launches, "nothing may be launched for a rejected shape"
    torch.cuda.synchronize()
    assert bool((hist == 7).all()), "the output of a rejected call is untouched"


def test_static_scratch_size_check_needs_no_device():
    """CPU: the size check precedes every CUDA call, so it can be exercised without a GPU (dummy non-NULL pointers)."""
    from paper_2208_09136_b200 import binding as B
    lib = B.load_library()
    p = B.RqaPoints()
    p.data, p.n_points, p.m, p.batch = 256, 99998, 3, 5
    p.point_stride, p.coord_stride, p.batch_stride, p.theiler = 1, 1, 100000, 0
    st = lib.rqa_line_hist_static(ctypes.byref(p), 0, 256, 20, 256, None)
    msg = lib.rqa_last_error().decode()
    assert st == B.RQA_ERR_UNSUPPORTED, msg
    assert str(B.RQA_STATIC_SCRATCH_BYTES) in msg and "rqa_line_hist with a caller workspace" in msg
    # the binding's constant is the header's
    header = (Path(__file__).resolve().parent.parent / "include" / "rqa.h").read_text()
    mib = re.search(r"#define RQA_STATIC_SCRATCH_BYTES \((\d+)u << 20\)", header)
    assert mib and int(mib.group(1)) << 20 == B.RQA_STATIC_SCRATCH_BYTES
    # argument errors as rqa_line_hist
    assert lib.rqa_line_hist_static(None, 0, 256, 20, 256, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist_static(ctypes.byref(p), 0, None, 20, 256, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist_static(ctypes.byref(p), 0, 256, 20, None, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist_static(ctypes.byref(p), 0, 256, 0, 256, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist_static(ctypes.byref(p), 7, 256, 20, 256, None) == B.RQA_ERR_INVALID_ARG
