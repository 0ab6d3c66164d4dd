"""Build ``librt_b200.so`` in-tree with nvcc for sm_100a (``python -m paper_2508_15967_b200.build [--force]``)."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

_HERE = Path(__file__).resolve().parent
CSRC = _HERE / "csrc"
LIB = _HERE / "librt_b200.so"
SOURCES = ("rt_api.cu", "spline_fit.cpp")
HEADERS = ("rt_math.cuh", "rt_kernels.cuh", "rt_params.h", "spline_fit.h", "../../include/rt.h", "../../include/rt_bench.h")
NVCC_FLAGS = ("-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "-shared", "-Xptxas", "-v")


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found (set NVCC=/path/to/nvcc)")


def stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any((CSRC / f).stat().st_mtime > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> Path:
    """Compile the CUDA extension if it is missing or older than its sources.  Returns the library path; the ptxas
    resource report (registers, spills) is written beside it as ``librt_b200.ptxas.txt``."""
    if not force and not stale():
        return LIB
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc_path(), *NVCC_FLAGS, *[str(CSRC / s) for s in SOURCES], "-o", str(tmp)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    (_HERE / "librt_b200.ptxas.txt").write_text("$ " + " ".join(cmd) + "\n" + r.stderr)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed")
    os.replace(tmp, LIB)
    if verbose:
        print(r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
