"""ctypes loader for the CPU oracle (oracle/rqa_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  Nothing under paper_2208_09136_b200/ imports this module, and this module imports
nothing from the package: the oracle and the CUDA path share no code.

All arithmetic lives in rqa_oracle.cpp; this file only builds it (g++ -O2 -ffp-contract=off -fopenmp) and
marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rqa_oracle.cpp"
_LIB = _HERE / "librqa_oracle.so"

NORM_MAX = 0
NORM_EUCLID = 1

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle into oracle/librqa_oracle.so (building the checker is not using it)."""
    if not force and _LIB.exists() and _LIB.stat().st_mtime >= _SRC.stat().st_mtime:
        return _LIB
    tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c++17",
           "-o", str(tmp), str(_SRC)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(str(_LIB))
    f32p = ctypes.POINTER(ctypes.c_float)
    f64p = ctypes.POINTER(ctypes.c_double)
    u64p = ctypes.POINTER(ctypes.c_uint64)
    i64, i32 = ctypes.c_int64, ctypes.c_int
    lib.rqa_oracle_max_threads.restype = i32
    lib.rqa_oracle_embed.argtypes = [f32p, i64, i32, i64, f32p]
    lib.rqa_oracle_distances.argtypes = [f32p, i64, i32, i64, i32, f32p]
    lib.rqa_oracle_rank.argtypes = [ctypes.c_double, ctypes.c_uint64]
    lib.rqa_oracle_rank.restype = ctypes.c_uint64
    lib.rqa_oracle_eps_for_rr.argtypes = [f32p, i64, i32, i64, i32, f64p, i32, f32p, u64p, f64p, i64]
    lib.rqa_oracle_count_lt_le.argtypes = [f32p, i64, i32, i64, i32, f32p, i32, u64p, u64p, i32, i64]
    lib.rqa_oracle_line_hist.argtypes = [f32p, i64, i32, i64, i32, f32p, i32, u64p, i32, i32, i64]
    lib.rqa_oracle_vert_hist.argtypes = [f32p, i64, i32, i64, i32, f32p, i32, u64p, i32, i64]
    lib.rqa_oracle_lam_tt.argtypes = [u64p, i32, i64, i64, f64p, f64p]
    lib.rqa_oracle_det_avg.argtypes = [u64p, i32, i64, i64, f64p, f64p]
    lib.rqa_oracle_det_prefix_avg.argtypes = [f64p, i32, f64p]
    lib.rqa_oracle_line_measures.argtypes = [u64p, i32, i64, i64, f64p, u64p, f64p, f64p, i64]
    lib.rqa_oracle_sorting_rate.argtypes = [f64p, i32, i32, f64p]
    _lib = lib
    return lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def _series(y) -> np.ndarray:
    y = np.ascontiguousarray(y, dtype=np.float32)
    if y.ndim != 1:
        raise ValueError("series must be 1-D")
    return y


def _check(st: int, what: str):
    if st != 0:
        raise RuntimeError(f"oracle {what} failed with status {st}")


def max_threads() -> int:
    return int(_load().rqa_oracle_max_threads())


def n_embedded(N: int, m: int, tau: int) -> int:
    return N - (m - 1) * tau


def n_pairs(N: int, m: int, tau: int) -> int:
    n = n_embedded(N, m, tau)
    return n * (n - 1) // 2


def embed(y, m: int, tau: int) -> np.ndarray:
    y = _series(y)
    n = n_embedded(len(y), m, tau)
    X = np.empty((n, m), dtype=np.float32)
    _check(_load().rqa_oracle_embed(_p(y, ctypes.c_float), len(y), m, tau, _p(X, ctypes.c_float)), "embed")
    return X


def distances(y, m: int, tau: int, norm: int = NORM_MAX) -> np.ndarray:
    y = _series(y)
    out = np.empty(n_pairs(len(y), m, tau), dtype=np.float32)
    _check(_load().rqa_oracle_distances(_p(y, ctypes.c_float), len(y), m, tau, norm, _p(out, ctypes.c_float)),
           "distances")
    return out


def rank(rr: float, P: int) -> int:
    return int(_load().rqa_oracle_rank(float(rr), int(P)))


def eps_for_rr(y, m: int, tau: int, rr, norm: int = NORM_MAX, theiler: int = 1):
    """-> (eps[K] float32, count[K] uint64, rr_realised[K] float64); theiler = w > 1: pairs with j - i >= w only"""
    y = _series(y)
    rr = np.ascontiguousarray(rr, dtype=np.float64)
    K = len(rr)
    eps = np.empty(K, dtype=np.float32)
    cnt = np.empty(K, dtype=np.uint64)
    rrr = np.empty(K, dtype=np.float64)
    _check(_load().rqa_oracle_eps_for_rr(_p(y, ctypes.c_float), len(y), m, tau, norm, _p(rr, ctypes.c_double), K,
                                         _p(eps, ctypes.c_float), _p(cnt, ctypes.c_uint64),
                                         _p(rrr, ctypes.c_double), max(1, theiler)), "eps_for_rr")
    return eps, cnt, rrr


def count_lt_le(y, m: int, tau: int, eps, norm: int = NORM_MAX, threads: int = 0, theiler: int = 1):
    """-> (#{d < eps_k}, #{d <= eps_k}) as uint64[K] over the pairs with j - i >= theiler — the counting certificate."""
    y = _series(y)
    eps = np.ascontiguousarray(eps, dtype=np.float32)
    K = len(eps)
    lt = np.empty(K, dtype=np.uint64)
    le = np.empty(K, dtype=np.uint64)
    _check(_load().rqa_oracle_count_lt_le(_p(y, ctypes.c_float), len(y), m, tau, norm, _p(eps, ctypes.c_float), K,
                                          _p(lt, ctypes.c_uint64), _p(le, ctypes.c_uint64), threads, max(1, theiler)),
           "count_lt_le")
    return lt, le


def line_hist(y, m: int, tau: int, eps, norm: int = NORM_MAX, lower: bool = False, threads: int = 1,
              theiler: int = 1) -> np.ndarray:
    """-> hist[K][N'] uint64 (theiler = w > 1: only the diagonals j - i >= w)"""
    y = _series(y)
    eps = np.ascontiguousarray(eps, dtype=np.float32)
    K = len(eps)
    n = n_embedded(len(y), m, tau)
    hist = np.empty((K, n), dtype=np.uint64)
    _check(_load().rqa_oracle_line_hist(_p(y, ctypes.c_float), len(y), m, tau, norm, _p(eps, ctypes.c_float), K,
                                        _p(hist, ctypes.c_uint64), 1 if lower else 0, threads, max(1, theiler)),
           "line_hist")
    return hist


def vert_hist(y, m: int, tau: int, eps, norm: int = NORM_MAX, threads: int = 1, theiler: int = 1) -> np.ndarray:
    """-> vhist[K][N'] uint64: vertical-line lengths over the columns of the full symmetric matrix (reading S19)"""
    y = _series(y)
    eps = np.ascontiguousarray(eps, dtype=np.float32)
    K = len(eps)
    n = n_embedded(len(y), m, tau)
    vhist = np.empty((K, n), dtype=np.uint64)
    _check(_load().rqa_oracle_vert_hist(_p(y, ctypes.c_float), len(y), m, tau, norm, _p(eps, ctypes.c_float), K,
                                        _p(vhist, ctypes.c_uint64), threads, max(1, theiler)), "vert_hist")
    return vhist


def lam_tt(vhist, v_min: int = 2):
    """-> (LAM[K], TT[K]) float64 from the vertical-line histogram"""
    vhist = np.ascontiguousarray(vhist, dtype=np.uint64)
    K, n = vhist.shape
    lam = np.empty(K, dtype=np.float64)
    tt = np.empty(K, dtype=np.float64)
    _check(_load().rqa_oracle_lam_tt(_p(vhist, ctypes.c_uint64), K, n, v_min, _p(lam, ctypes.c_double),
                                     _p(tt, ctypes.c_double)), "lam_tt")
    return lam, tt


def det_avg(hist, l_min: int = 2):
    """-> (det[K] float64, det_mean float)"""
    hist = np.ascontiguousarray(hist, dtype=np.uint64)
    K, n = hist.shape
    det = np.empty(K, dtype=np.float64)
    mean = ctypes.c_double(0.0)
    _check(_load().rqa_oracle_det_avg(_p(hist, ctypes.c_uint64), K, n, l_min, _p(det, ctypes.c_double),
                                      ctypes.byref(mean)), "det_avg")
    return det, float(mean.value)


def det_prefix_avg(det) -> np.ndarray:
    """Eq. 5 for every cut-off: prefix[k] = mean(det[0..k])."""
    det = np.ascontiguousarray(det, dtype=np.float64)
    out = np.empty_like(det)
    _check(_load().rqa_oracle_det_prefix_avg(_p(det, ctypes.c_double), det.shape[0], _p(out, ctypes.c_double)),
           "det_prefix_avg")
    return out


def line_measures(hist, l_min: int = 2, theiler: int = 1):
    """-> (L[K] float64, Lmax[K] uint64, rr_hist[K] float64, entr[K] float64)"""
    hist = np.ascontiguousarray(hist, dtype=np.uint64)
    K, n = hist.shape
    L = np.empty(K, dtype=np.float64)
    Lmax = np.empty(K, dtype=np.uint64)
    rr = np.empty(K, dtype=np.float64)
    entr = np.empty(K, dtype=np.float64)
    _check(_load().rqa_oracle_line_measures(_p(hist, ctypes.c_uint64), K, n, l_min, _p(L, ctypes.c_double),
                                            _p(Lmax, ctypes.c_uint64), _p(rr, ctypes.c_double),
                                            _p(entr, ctypes.c_double), max(1, theiler)), "line_measures")
    return L, Lmax, rr, entr


def sorting_rate(measure) -> float:
    """Eq. 6: measure [R][n] (n series in natural order, R realisations) -> S in [.., 1]."""
    a = np.ascontiguousarray(measure, dtype=np.float64)
    S = np.zeros(1, dtype=np.float64)
    _check(_load().rqa_oracle_sorting_rate(_p(a, ctypes.c_double), a.shape[0], a.shape[1], _p(S, ctypes.c_double)),
           "sorting_rate")
    return float(S[0])


def sweep(y, m: int, tau: int, rr, norm: int = NORM_MAX, l_min: int = 2, threads: int = 1, theiler: int = 1):
    """The whole hot path on one series: eps -> hist -> DET.  Returns a dict."""
    eps, cnt, rrr = eps_for_rr(y, m, tau, rr, norm, theiler)
    hist = line_hist(y, m, tau, eps, norm, threads=threads, theiler=theiler)
    det, mean = det_avg(hist, l_min)
    return {"eps": eps, "count": cnt, "rr": rrr, "hist": hist, "det": det, "det_mean": mean}
