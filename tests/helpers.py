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
