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


def _objects():
    objdir = PKG / "build"
    return [(src, objdir / f"{src.stem}.o") for src in sources()]


def _newest_header() -> float:
    headers = list(CSRC.glob("*.cuh")) + [ROOT / "include" / "rqa.h", Path(__file__)]
    return max(h.stat().st_mtime for h in headers)


def _src_mtime(src: Path) -> float:
    """mtime of a translation unit = its own and that of any .cu file it includes (rqa_fused_scan.cu includes rqa_line.cu)."""
    import re
    t = src.stat().st_mtime
    for inc in re.findall(r'#include\s+"([^"]+\.cu)"', src.read_text()):
        if (CSRC / inc).exists():
            t = max(t, (CSRC / inc).stat().st_mtime)
    return t


def _obj_stale(src: Path, obj: Path, newest_header: float) -> bool:
    return not obj.exists() or obj.stat().st_mtime <= max(_src_mtime(src), newest_header)


def _stale() -> bool:
    """The library is stale if it is missing, if an object is older than its source or any header, or if it is older than
    an object (an object rebuilt after the last link)."""
    if not LIB.exists():
        return True
    nh = _newest_header()
    t = LIB.stat().st_mtime
    return any(_obj_stale(src, obj, nh) or obj.stat().st_mtime > t for src, obj in _objects())


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = PKG / "build"
    objdir.mkdir(exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    # one nvcc per translation unit, side by side (the big ones take minutes each), then link.  Objects are kept and
    # reused while they are newer than their source, every header and this file (force=True rebuilds all of them).
    newest_header = _newest_header()
    jobs, objs = [], []
    for src, obj in _objects():
        objs.append(obj)
        if not force and not _obj_stale(src, obj, newest_header):
            continue
        tmp = objdir / f"{src.stem}.{os.getpid()}.tmp.o"
        jobs.append((obj, tmp, subprocess.Popen([nvcc, *NVCC_FLAGS, *extra, "-c", "-o", str(tmp), str(src)])))
    failed = []
    for obj, tmp, proc in jobs:
        if proc.wait() != 0:
            failed.append(str(obj))
            tmp.unlink(missing_ok=True)
        else:
            os.replace(tmp, obj)
    if failed:
        raise RuntimeError(f"nvcc failed for {failed}")
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", str(tmp), *[str(o) for o in objs]],
                   check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
