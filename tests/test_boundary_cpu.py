"""CPU-side checks of the boundary: librqa.so loads, exports every symbol include/rqa.h declares, and rejects bad
arguments before launching anything.  No compute calls (no GPU needed)."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

import paper_2208_09136_b200 as pkg
from paper_2208_09136_b200 import binding as B

ROOT = Path(__file__).resolve().parent.parent
FAKE = 0x10000   # a non-NULL, 256-byte aligned "device pointer" that validation never dereferences


@pytest.fixture(scope="module")
def lib():
    from paper_2208_09136_b200 import build
    build.build()
    return pkg.load_library()


def _declared_functions():
    text = (ROOT / "include" / "rqa.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rqa_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_functions()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), f"librqa.so does not export {n}"
    assert sorted(B.EXPORTS) == names
    assert lib.rqa_version().decode().endswith("sm_100a")


def test_status_strings(lib):
    assert lib.rqa_status_string(0) == b"RQA_OK"
    assert lib.rqa_status_string(2) == b"RQA_ERR_NONFINITE_INPUT"
    assert lib.rqa_status_string(5) == b"RQA_ERR_CUDA"


def _pts(n=100, m=3, batch=1, ps=1, cs=1, bs=100, data=FAKE):
    return B.RqaPoints(data, n, m, batch, ps, cs, bs)


def test_workspace_bytes_and_validation(lib):
    sz = ctypes.c_size_t(0)
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts()), 20, ctypes.byref(sz)) == B.RQA_OK and sz.value >= 256
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(data=None)), 20, ctypes.byref(sz)) == B.RQA_OK
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(n=1)), 20, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(m=0)), 20, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(m=17)), 20, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts()), 0, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts()), 129, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(n=(1 << 24) + 1)), 4, ctypes.byref(sz)) == B.RQA_ERR_UNSUPPORTED
    assert b"n_points" in lib.rqa_last_error()
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(batch=65536)), 4, ctypes.byref(sz)) == B.RQA_ERR_UNSUPPORTED
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(batch=65535)), 4, ctypes.byref(sz)) == B.RQA_OK
    # materialised points: wide points still get a (larger) workspace; sizes grow with the batch
    a, b2 = ctypes.c_size_t(0), ctypes.c_size_t(0)
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(n=5000, m=16, ps=16, cs=1, bs=80000)), 20, ctypes.byref(a)) == B.RQA_OK
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts(n=5000, m=16, ps=16, cs=1, bs=80000, batch=3)), 20, ctypes.byref(b2)) == B.RQA_OK
    assert b2.value > a.value > 256
    sw = ctypes.c_size_t(0)
    assert lib.rqa_sweep_workspace_bytes(1000, 5, 4, 6, 10, ctypes.byref(sw)) == B.RQA_OK
    assert sw.value > 5 * 10 * 982 * 8
    assert lib.rqa_sweep_workspace_bytes(10, 1, 4, 6, 10, ctypes.byref(sw)) == B.RQA_ERR_INVALID_ARG


def test_eps_for_rr_rejects_bad_arguments(lib):
    rr = np.array([0.1, 0.2], dtype=np.float64)

    def call(pts=None, norm=0, rrv=rr, K=2, eps=FAKE, cnt=FAKE, rrr=FAKE, ws=FAKE, wsb=1 << 30):
        return lib.rqa_eps_for_rr(ctypes.byref(pts or _pts()), norm, rrv.ctypes.data if rrv is not None else None, K,
                                  eps, cnt, rrr, ws, wsb, None)

    assert call(K=0) == B.RQA_ERR_INVALID_ARG
    assert call(K=129) == B.RQA_ERR_INVALID_ARG
    assert call(norm=7) == B.RQA_ERR_INVALID_ARG
    assert call(eps=None) == B.RQA_ERR_INVALID_ARG
    assert call(rrv=None) == B.RQA_ERR_INVALID_ARG
    assert call(ws=FAKE + 8) == B.RQA_ERR_INVALID_ARG           # misaligned workspace
    assert call(rrv=np.array([0.1, 0.0])) == B.RQA_ERR_INVALID_ARG
    assert call(rrv=np.array([0.1, 1.5])) == B.RQA_ERR_INVALID_ARG
    assert call(rrv=np.array([0.1, np.nan])) == B.RQA_ERR_INVALID_ARG
    assert call(pts=_pts(ps=0)) == B.RQA_ERR_INVALID_ARG
    assert call(wsb=16) == B.RQA_ERR_WORKSPACE_TOO_SMALL
    assert b"workspace" in lib.rqa_last_error()


def test_line_hist_det_embed_reject_bad_arguments(lib):
    assert lib.rqa_line_hist(ctypes.byref(_pts()), 0, None, 2, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist(ctypes.byref(_pts()), 0, FAKE, 0, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist(ctypes.byref(_pts()), 0, FAKE, 2, FAKE, FAKE, 8, None) == B.RQA_ERR_WORKSPACE_TOO_SMALL
    # the vertical-line calls validate the same way (reading S19)
    assert lib.rqa_vert_hist(ctypes.byref(_pts()), 0, None, 2, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_vert_hist(ctypes.byref(_pts()), 2, FAKE, 2, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG     # unknown norm
    assert lib.rqa_vert_hist(ctypes.byref(_pts()), 0, FAKE, 129, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_vert_hist(ctypes.byref(_pts()), 0, FAKE, 2, FAKE, FAKE, 8, None) == B.RQA_ERR_WORKSPACE_TOO_SMALL
    assert lib.rqa_vert_hist(None, 0, FAKE, 2, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_lam_tt(None, 1, 2, 100, 2, FAKE, FAKE, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_lam_tt(FAKE, 1, 2, 100, 0, FAKE, FAKE, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_det_avg(None, 1, 2, 100, 2, FAKE, FAKE, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_det_avg(FAKE, 1, 2, 100, 0, FAKE, FAKE, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_det_avg(FAKE, 0, 2, 100, 2, FAKE, FAKE, None) == B.RQA_ERR_INVALID_ARG
    view = B.RqaPoints()
    assert lib.rqa_embed(FAKE, 10, 1, 10, 4, 6, None, ctypes.byref(view), None) == B.RQA_ERR_INVALID_ARG   # N' < 2
    assert lib.rqa_embed(FAKE, 100, 1, 100, 0, 1, None, ctypes.byref(view), None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_embed(FAKE, 100, 2, 50, 3, 1, None, ctypes.byref(view), None) == B.RQA_ERR_INVALID_ARG   # stride < N
    # the view form needs no launch, so it works without a GPU
    assert lib.rqa_embed(FAKE, 1000, 5, 1000, 4, 6, None, ctypes.byref(view), None) == B.RQA_OK
    assert (view.n_points, view.m, view.batch, view.point_stride, view.coord_stride, view.batch_stride) == \
        (982, 4, 5, 1, 6, 1000)


def test_options_are_per_call_and_validated(lib):
    """struct rqa_options travels with the call (the library has no global state): bad fields are rejected before any
    launch, and workspace sizes follow the options passed to rqa_workspace_bytes_opt."""
    assert not hasattr(lib, "rqa_set_option_does_not_exist")
    with pytest.raises(AttributeError):
        lib.rqa_set_option                                   # the process-wide knobs of round 1 are gone
    sz = ctypes.c_size_t(0)
    pts = _pts(n=5000, bs=5002)

    def size(**kw):
        o = B.make_options(**kw)
        st = lib.rqa_workspace_bytes_opt(ctypes.byref(pts), 20, ctypes.byref(o), ctypes.byref(sz))
        return st, sz.value
    assert size(select_path=5)[0] == B.RQA_ERR_INVALID_ARG
    assert size(select_path=-1)[0] == B.RQA_ERR_INVALID_ARG
    assert size(line_chunk=1024)[0] == B.RQA_ERR_INVALID_ARG
    assert size(line_buffers=3)[0] == B.RQA_ERR_INVALID_ARG
    assert size(line_path=3)[0] == B.RQA_ERR_INVALID_ARG
    assert size(group_size=33)[0] == B.RQA_ERR_INVALID_ARG
    assert size(line_segment=-1)[0] == B.RQA_ERR_INVALID_ARG
    assert size(sample_size=-1)[0] == B.RQA_ERR_INVALID_ARG
    assert size(part_index=2, part_count=2)[0] == B.RQA_ERR_INVALID_ARG
    assert size(part_index=1, part_count=0)[0] == B.RQA_ERR_INVALID_ARG
    assert size(part_index=0, part_count=2)[0] == B.RQA_ERR_INVALID_ARG      # a split call needs a reduce callback
    assert size(part_index=1, part_count=2, reduce=lambda p, n, s: None)[0] == B.RQA_OK
    # the bracket path needs the sample and candidate buffers, the radix path does not
    st0, sz0 = size(select_path=3)
    st2, sz2 = size(select_path=2, sample_size=50_000_000)
    assert st0 == st2 == B.RQA_OK and sz2 >= 4 * 50_000_000 > sz0
    # NULL options = automatic = the plain call
    assert lib.rqa_workspace_bytes_opt(ctypes.byref(pts), 20, None, ctypes.byref(sz)) == B.RQA_OK
    auto = sz.value
    assert lib.rqa_workspace_bytes(ctypes.byref(pts), 20, ctypes.byref(sz)) == B.RQA_OK and sz.value == auto
    # the same call from two threads with different options: no interference (there is nothing to interfere with)
    import threading
    out = {}

    def worker(name, **kw):
        out[name] = [size_local(**kw) for _ in range(50)]

    def size_local(**kw):
        o, z = B.make_options(**kw), ctypes.c_size_t(0)
        assert lib.rqa_workspace_bytes_opt(ctypes.byref(pts), 20, ctypes.byref(o), ctypes.byref(z)) == B.RQA_OK
        return z.value
    ts = [threading.Thread(target=worker, args=("a",), kwargs={"select_path": 3}),
          threading.Thread(target=worker, args=("b",), kwargs={"select_path": 2, "sample_size": 50_000_000})]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert set(out["a"]) == {sz0} and set(out["b"]) == {sz2}


def test_null_arguments_never_crash(lib):
    """Every entry point returns a status for NULL pointers (round-1 finding: rqa_workspace_bytes(NULL, ...) crashed)."""
    sz = ctypes.c_size_t(0)
    assert lib.rqa_workspace_bytes(None, 20, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes(ctypes.byref(_pts()), 20, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_bytes_opt(None, 20, None, ctypes.byref(sz)) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_eps_for_rr(None, 0, FAKE, 2, FAKE, FAKE, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_line_hist(None, 0, FAKE, 2, FAKE, FAKE, 1 << 30, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_workspace_status(None, None) == B.RQA_ERR_INVALID_ARG
    assert lib.rqa_embed(None, 100, 1, 100, 3, 1, None, None, None) == B.RQA_ERR_INVALID_ARG
    assert b"NULL" in lib.rqa_last_error()


def test_no_cpu_fallback_without_gpu(lib):
    """Without a CUDA device a compute call must fail loudly with RQA_ERR_CUDA, never silently succeed."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    st = lib.rqa_det_avg(FAKE, 1, 2, 100, 2, FAKE, FAKE, None)
    assert st == B.RQA_ERR_CUDA
    assert lib.rqa_launch_count() >= 1


def test_product_path_does_not_import_the_oracle():
    pat = re.compile(r"import\s+oracle|from\s+oracle|rqa_oracle|#include.*oracle")
    for f in list((ROOT / "paper_2208_09136_b200").rglob("*")) + list((ROOT / "include").rglob("*")):
        if f.suffix in {".py", ".cu", ".cuh", ".h", ".cpp"}:
            assert not pat.search(f.read_text()), f
