"""Build librqa.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2208_09136_b200.build [--force]

-fmad=false: no implicit FMA contraction anywhere (BASELINE.json north_star; the Euclidean distance is
additionally written with __fsub_rn/__fmul_rn/__fadd_rn so it is flag-independent).  No -use_fast_math,
no -ftz=true: denormals are kept (reading S14).
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "librqa.so"

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
    "-Xcompiler", "-fPIC",
    "-I", str(ROOT / "include"), "-I", str(CSRC),
]


def sources():
    return sorted(CSRC.glob("*.cu"))


def _stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + [ROOT / "include" / "rqa.h", Path(__file__)]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = PKG / "build"
    objdir.mkdir(exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    # one nvcc per translation unit, side by side (the two big ones take about a minute each), then link
    jobs = []
    for src in sources():
        obj = objdir / f"{src.stem}.{os.getpid()}.o"
        jobs.append((obj, subprocess.Popen([nvcc, *NVCC_FLAGS, *extra, "-c", "-o", str(obj), str(src)])))
    failed = [str(obj) for obj, proc in jobs if proc.wait() != 0]
    if failed:
        raise RuntimeError(f"nvcc failed for {failed}")
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", str(tmp), *[str(obj) for obj, _ in jobs]],
                   check=True)
    os.replace(tmp, LIB)
    for obj, _ in jobs:
        obj.unlink(missing_ok=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
