"""Small helpers for the tests (no method arithmetic): golden-file parsing and error norms (reading A15)."""
from pathlib import Path

import numpy as np

GOLDEN = Path(__file__).resolve().parent / "golden"


def paper_facts() -> dict:
    out = {}
    for line in (GOLDEN / "paper_facts.txt").read_text().splitlines():
        line = line.split("#", 1)[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


def rel_err_xk(a: np.ndarray, b: np.ndarray):
    """Per-ray ||dx||_2/||x||_2 and ||dk||_2/||k||_2 (reading A15), maxima over rays.  a, b: [6, n]."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    ex = np.linalg.norm(a[:3] - b[:3], axis=0) / np.linalg.norm(b[:3], axis=0)
    ek = np.linalg.norm(a[3:] - b[3:], axis=0) / np.linalg.norm(b[3:], axis=0)
    return float(ex.max()), float(ek.max())


def build_host_shim(tmp_dir):
    """Compile tests/host_shim.cpp (the library's HOST-side logic behind C entry points: spline fit, constant folding, the
    range of the ion terms' series) with g++ and load it; no GPU involved."""
    import ctypes
    import subprocess
    here = Path(__file__).resolve().parent
    csrc = here.parent / "paper_2508_15967_b200" / "csrc"
    so = Path(tmp_dir) / "libspline_shim.so"
    subprocess.run(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", str(here / "host_shim.cpp"),
                    str(csrc / "spline_fit.cpp"), "-o", str(so)], check=True)
    lib = ctypes.CDLL(str(so))
    P = ctypes.c_void_p
    lib.shim_fit_cubic.argtypes = [P, P, ctypes.c_long, ctypes.c_int, P]
    lib.shim_fit_bicubic.argtypes = [P, P, P, ctypes.c_int, ctypes.c_int, P]
    lib.shim_fold_params.argtypes = [P, ctypes.c_double, ctypes.c_double, ctypes.c_int, P]
    lib.shim_series_cap.argtypes = [ctypes.c_double, ctypes.c_double]
    lib.shim_series_cap.restype = ctypes.c_double
    return lib
