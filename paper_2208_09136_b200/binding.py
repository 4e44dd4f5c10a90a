"""Thin ctypes binding over librqa.so (include/rqa.h).  Same names as the C ABI; argument marshalling only —
every step of the path runs in the library's CUDA kernels.  PyTorch supplies device memory and streams.

There is no fallback: if librqa.so is missing or cannot be loaded, load_library() raises.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

PKG = Path(__file__).resolve().parent
LIB_PATH = PKG / "librqa.so"

RQA_OK = 0
RQA_ERR_INVALID_ARG = 1
RQA_ERR_NONFINITE_INPUT = 2
RQA_ERR_WORKSPACE_TOO_SMALL = 3
RQA_ERR_UNSUPPORTED = 4
RQA_ERR_CUDA = 5
RQA_NORM_MAX = 0
RQA_NORM_EUCLID = 1
RQA_MAX_K = 128
RQA_MAX_M = 16
RQA_STATIC_SCRATCH_BYTES = 128 << 20

# every symbol include/rqa.h declares (tests check that the library exports them all)
EXPORTS = ["rqa_status_string", "rqa_last_error", "rqa_version", "rqa_workspace_bytes", "rqa_workspace_status",
           "rqa_embed", "rqa_eps_for_rr", "rqa_line_hist", "rqa_det_avg", "rqa_sweep_workspace_bytes",
           "rqa_sweep_host", "rqa_launch_count", "rqa_workspace_bytes_opt", "rqa_eps_for_rr_opt", "rqa_line_hist_opt",
           "rqa_det_prefix_avg", "rqa_line_measures", "rqa_sorting_rate_host", "rqa_vert_hist", "rqa_vert_hist_opt",
           "rqa_lam_tt", "rqa_line_hist_static"]


class RqaPoints(ctypes.Structure):
    """struct rqa_points"""
    _fields_ = [("data", ctypes.c_void_p), ("n_points", ctypes.c_int64), ("m", ctypes.c_int32),
                ("batch", ctypes.c_int32), ("point_stride", ctypes.c_int64), ("coord_stride", ctypes.c_int64),
                ("batch_stride", ctypes.c_int64), ("theiler", ctypes.c_int64)]


REDUCE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)


class RqaOptions(ctypes.Structure):
    """struct rqa_options (per call; every field 0 = automatic)"""
    _fields_ = [("select_path", ctypes.c_int32), ("line_chunk", ctypes.c_int32), ("line_segment", ctypes.c_int32),
                ("part_index", ctypes.c_int32), ("part_count", ctypes.c_int32), ("line_buffers", ctypes.c_int32),
                ("sample_size", ctypes.c_int64), ("cand_cap", ctypes.c_int64), ("reduce", REDUCE_FN),
                ("reduce_ctx", ctypes.c_void_p), ("ev_kernel_begin", ctypes.c_void_p), ("ev_kernel_end", ctypes.c_void_p),
                ("line_path", ctypes.c_int32), ("group_size", ctypes.c_int32)]


def make_options(select_path=0, line_chunk=0, line_segment=0, line_buffers=0, sample_size=0, cand_cap=0, part_index=0,
                 part_count=0, reduce=None, kernel_events=None, line_path=0, group_size=0) -> RqaOptions:
    """reduce: a Python callable (d_ptr: int, n: int, stream: int) -> None that sums n uint64 device counters over the
    parts of a split call (see parts.py); kept alive by the returned struct.
    kernel_events: a pair of torch.cuda.Event(enable_timing=True) that the call records just before / after its dominant
    kernel (rqa_options.ev_kernel_begin / ev_kernel_end)."""
    o = RqaOptions()
    o.select_path, o.line_chunk, o.line_segment, o.line_buffers = select_path, line_chunk, line_segment, line_buffers
    o.sample_size, o.cand_cap, o.part_index, o.part_count = sample_size, cand_cap, part_index, part_count
    o.line_path, o.group_size = line_path, group_size
    if reduce is not None:
        def _cb(ctx, ptr, n, stream):
            try:
                reduce(int(ptr or 0), int(n), int(stream or 0))
                return 0
            except Exception:                                # never let an exception cross the C ABI
                import traceback
                traceback.print_exc()
                return 1
        o._cb = REDUCE_FN(_cb)
        o.reduce = o._cb
    if kernel_events is not None:
        a, b = kernel_events
        a.record(); b.record()                               # torch creates the cudaEvent_t lazily, on the first record
        o._events = (a, b)
        o.ev_kernel_begin, o.ev_kernel_end = a.cuda_event, b.cuda_event
    return o


def _opt(options):
    return None if options is None else ctypes.byref(options)


class RqaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{msg} (status {status})")
        self.status = status


_lib = None


def load_library() -> ctypes.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2208_09136_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(str(LIB_PATH))
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    pts = ctypes.POINTER(RqaPoints)
    lib.rqa_status_string.restype = ctypes.c_char_p
    lib.rqa_status_string.argtypes = [ctypes.c_int]
    lib.rqa_last_error.restype = ctypes.c_char_p
    lib.rqa_version.restype = ctypes.c_char_p
    lib.rqa_launch_count.restype = ctypes.c_uint64
    lib.rqa_workspace_bytes.argtypes = [pts, i32, ctypes.POINTER(sz)]
    lib.rqa_workspace_status.argtypes = [vp, vp]
    lib.rqa_embed.argtypes = [vp, i64, i32, i64, i32, i64, vp, pts, vp]
    lib.rqa_eps_for_rr.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp, vp, vp, sz, vp]
    lib.rqa_line_hist.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp, sz, vp]
    lib.rqa_det_avg.argtypes = [vp, i32, i32, i64, i64, vp, vp, vp]
    lib.rqa_sweep_workspace_bytes.argtypes = [i64, i32, i32, i64, i32, ctypes.POINTER(sz)]
    lib.rqa_sweep_host.argtypes = [vp, i64, i32, i32, i64, ctypes.c_int, vp, i32, i64, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    opt = ctypes.POINTER(RqaOptions)
    lib.rqa_workspace_bytes_opt.argtypes = [pts, i32, opt, ctypes.POINTER(sz)]
    lib.rqa_eps_for_rr_opt.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp, vp, vp, sz, vp, opt]
    lib.rqa_line_hist_opt.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp, sz, vp, opt]
    lib.rqa_det_prefix_avg.argtypes = [vp, i32, i32, vp, vp]
    lib.rqa_line_measures.argtypes = [vp, i32, i32, i64, i64, i64, vp, vp, vp, vp, vp]
    lib.rqa_sorting_rate_host.argtypes = [vp, i32, i32, ctypes.POINTER(ctypes.c_double)]
    lib.rqa_vert_hist.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp, sz, vp]
    lib.rqa_vert_hist_opt.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp, sz, vp, opt]
    lib.rqa_lam_tt.argtypes = [vp, i32, i32, i64, i64, vp, vp, vp]
    lib.rqa_line_hist_static.argtypes = [pts, ctypes.c_int, vp, i32, vp, vp]
    _lib = lib
    return lib


def _check(st: int):
    if st != RQA_OK:
        lib = load_library()
        raise RqaError(st, f"{lib.rqa_status_string(st).decode()}: {lib.rqa_last_error().decode()}")


def _stream(stream=None) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _dev(t, dtype, what: str, numel: int = None) -> int:
    """Device pointer of a contiguous CUDA tensor of the given dtype on the current device (and, when `numel` is given,
    of exactly that many elements: a wrong shape would otherwise be a silent out-of-bounds device write)."""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{what} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{what} must be a contiguous {dtype} tensor")
    if t.device.index != torch.cuda.current_device():
        raise ValueError(f"{what} lives on {t.device}, the current device is cuda:{torch.cuda.current_device()}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{what} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def rqa_version() -> str:
    return load_library().rqa_version().decode()


def rqa_launch_count() -> int:
    return int(load_library().rqa_launch_count())


def rqa_workspace_bytes(pts: RqaPoints, K: int, options: RqaOptions = None) -> int:
    n = ctypes.c_size_t(0)
    _check(load_library().rqa_workspace_bytes_opt(ctypes.byref(pts), K, _opt(options), ctypes.byref(n)))
    return int(n.value)


def rqa_workspace_status(ws, stream=None) -> None:
    """Synchronises the stream; raises RqaError (e.g. RQA_ERR_NONFINITE_INPUT) if the last call recorded one."""
    import torch
    _check(load_library().rqa_workspace_status(_dev(ws, torch.uint8, "ws"), _stream(stream)))


def rqa_embed(series, m: int, tau: int, X=None, stream=None, theiler: int = 0) -> RqaPoints:
    """series: float32 CUDA tensor [batch][N] (or [N]).  Returns the rqa_points view (of `series` itself when
    X is None, else of the materialised X[batch][N'][m] the call writes).  The returned view holds a reference to
    the tensor it points into."""
    import torch
    if series.dim() == 1:
        series = series.unsqueeze(0)
    p = _dev(series, torch.float32, "series")
    batch, N = series.shape
    view = RqaPoints()
    xp = None if X is None else _dev(X, torch.float32, "X", batch * (N - (m - 1) * tau) * m)
    _check(load_library().rqa_embed(p, N, batch, N, m, tau, xp, ctypes.byref(view), _stream(stream)))
    view._owner = series if X is None else X                 # the view points into this tensor: keep it alive
    view.theiler = theiler                                   # a field of the view, not an argument of rqa_embed
    return view


def rqa_eps_for_rr(pts: RqaPoints, norm: int, rr, eps, count, rr_realised, ws, stream=None,
                   options: RqaOptions = None) -> None:
    """rr: host float64 array [K]; eps float32 / count int64(uint64 bits) / rr_realised float64 CUDA tensors
    [batch][K]; ws: uint8 CUDA workspace."""
    import torch
    rr = np.ascontiguousarray(rr, dtype=np.float64)
    K = len(rr)
    bk = int(pts.batch) * K
    _check(load_library().rqa_eps_for_rr_opt(ctypes.byref(pts), norm, rr.ctypes.data, K,
                                             _dev(eps, torch.float32, "eps", bk), _dev(count, torch.int64, "count", bk),
                                             _dev(rr_realised, torch.float64, "rr_realised", bk),
                                             _dev(ws, torch.uint8, "ws"), ws.numel(), _stream(stream), _opt(options)))


def rqa_line_hist(pts: RqaPoints, norm: int, eps, hist, ws, stream=None, options: RqaOptions = None) -> None:
    """eps float32 CUDA [batch][K]; hist int64 (uint64 bits) CUDA [batch][K][n_points]."""
    import torch
    K = eps.shape[-1]
    bk = int(pts.batch) * K
    _check(load_library().rqa_line_hist_opt(ctypes.byref(pts), norm, _dev(eps, torch.float32, "eps", bk), K,
                                            _dev(hist, torch.int64, "hist", bk * int(pts.n_points)),
                                            _dev(ws, torch.uint8, "ws"), ws.numel(), _stream(stream), _opt(options)))


def rqa_line_hist_static(pts: RqaPoints, norm: int, eps, hist, stream=None) -> None:
    """rqa_line_hist without a workspace argument: the scratch is a static device array inside the library
    (RQA_STATIC_SCRATCH_BYTES; larger shapes raise RQA_ERR_UNSUPPORTED).  No device allocation is made by the call."""
    import torch
    K = eps.shape[-1]
    bk = int(pts.batch) * K
    _check(load_library().rqa_line_hist_static(ctypes.byref(pts), norm, _dev(eps, torch.float32, "eps", bk), K,
                                               _dev(hist, torch.int64, "hist", bk * int(pts.n_points)),
                                               _stream(stream)))


def rqa_vert_hist(pts: RqaPoints, norm: int, eps, vhist, ws, stream=None, options: RqaOptions = None) -> None:
    """eps float32 CUDA [batch][K]; vhist int64 (uint64 bits) CUDA [batch][K][n_points]: vertical-line histograms."""
    import torch
    K = eps.shape[-1]
    bk = int(pts.batch) * K
    _check(load_library().rqa_vert_hist_opt(ctypes.byref(pts), norm, _dev(eps, torch.float32, "eps", bk), K,
                                            _dev(vhist, torch.int64, "vhist", bk * int(pts.n_points)),
                                            _dev(ws, torch.uint8, "ws"), ws.numel(), _stream(stream), _opt(options)))


def rqa_lam_tt(vhist, v_min: int, lam=None, tt=None, stream=None) -> None:
    """vhist int64 CUDA [batch][K][n_points]; lam, tt float64 [batch][K] (either may be None)."""
    import torch
    batch, K, n = vhist.shape
    _check(load_library().rqa_lam_tt(_dev(vhist, torch.int64, "vhist"), batch, K, n, v_min,
                                     None if lam is None else _dev(lam, torch.float64, "lam", batch * K),
                                     None if tt is None else _dev(tt, torch.float64, "tt", batch * K), _stream(stream)))


def rqa_det_avg(hist, l_min: int, det, det_mean, stream=None) -> None:
    """hist int64 CUDA [batch][K][n_points]; det float64 [batch][K]; det_mean float64 [batch]."""
    import torch
    batch, K, n = hist.shape
    _check(load_library().rqa_det_avg(_dev(hist, torch.int64, "hist"), batch, K, n, l_min,
                                      _dev(det, torch.float64, "det", batch * K),
                                      _dev(det_mean, torch.float64, "det_mean", batch), _stream(stream)))


def rqa_det_prefix_avg(det, prefix, stream=None) -> None:
    """det, prefix float64 CUDA [batch][K]: Eq. 5 for every cut-off."""
    import torch
    batch, K = det.shape
    _check(load_library().rqa_det_prefix_avg(_dev(det, torch.float64, "det"), batch, K,
                                             _dev(prefix, torch.float64, "prefix"), _stream(stream)))


def rqa_line_measures(hist, l_min: int, L=None, Lmax=None, rr_hist=None, entr=None, stream=None, theiler: int = 0) -> None:
    """hist int64 CUDA [batch][K][n_points]; L, rr_hist, entr float64 [batch][K]; Lmax int64 [batch][K]; each may be
    None."""
    import torch
    batch, K, n = hist.shape
    _check(load_library().rqa_line_measures(_dev(hist, torch.int64, "hist"), batch, K, n, l_min, theiler,
                                            None if L is None else _dev(L, torch.float64, "L"),
                                            None if Lmax is None else _dev(Lmax, torch.int64, "Lmax"),
                                            None if rr_hist is None else _dev(rr_hist, torch.float64, "rr_hist"),
                                            None if entr is None else _dev(entr, torch.float64, "entr"),
                                            _stream(stream)))


def rqa_sorting_rate_host(measure) -> float:
    """measure: host array [R][n] of float64 (n series in their natural order, R realisations) -> S of Eq. 6."""
    import numpy as np
    a = np.ascontiguousarray(measure, dtype=np.float64)
    if a.ndim != 2:
        raise ValueError("measure must be [R][n]")
    out = ctypes.c_double(0.0)
    _check(load_library().rqa_sorting_rate_host(a.ctypes.data, a.shape[0], a.shape[1], ctypes.byref(out)))
    return float(out.value)


def rqa_sweep_workspace_bytes(N: int, batch: int, m: int, tau: int, K: int) -> int:
    n = ctypes.c_size_t(0)
    _check(load_library().rqa_sweep_workspace_bytes(N, batch, m, tau, K, ctypes.byref(n)))
    return int(n.value)


def rqa_sweep_host(series, m: int, tau: int, norm: int, rr, l_min: int, eps, count, rr_realised, det, det_mean, hist,
                   ws, stream=None) -> None:
    """Host buffers in, host buffers out (CPU torch tensors, pinned for asynchronous copies); `ws` is a CUDA
    uint8 workspace of rqa_sweep_workspace_bytes(...).  hist may be None."""
    import torch
    rr = np.ascontiguousarray(rr, dtype=np.float64)

    def host(t, dtype, what):
        if t.is_cuda or t.dtype != dtype or not t.is_contiguous():
            raise TypeError(f"{what} must be a contiguous CPU {dtype} tensor")
        return t.data_ptr()

    batch, N = series.shape
    _check(load_library().rqa_sweep_host(
        host(series, torch.float32, "series"), N, batch, m, tau, norm, rr.ctypes.data, len(rr), l_min,
        host(eps, torch.float32, "eps"), host(count, torch.int64, "count"),
        host(rr_realised, torch.float64, "rr_realised"), host(det, torch.float64, "det"),
        host(det_mean, torch.float64, "det_mean"), None if hist is None else host(hist, torch.int64, "hist"),
        _dev(ws, torch.uint8, "ws"), ws.numel(), _stream(stream)))
