"""CPU oracle for batched RF ray tracing -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_2508_15967_b200`` (the CUDA path) and never
imports it.  The arithmetic lives in ``rt_oracle.cpp`` (plain C++17, fp64, dual-number differentiation of
the literal dispersion function, classical RK4); this file only builds it with g++, marshals numpy arrays
through ctypes, and -- for the grid equilibrium -- fits the not-a-knot cubic splines with
``scipy.interpolate.CubicSpline`` (a library primitive used as a step; reading A10).

Citations: /root/reference/PAPER.md Eq. 2-3 (L139-145) ray equations, L147 RK4 kernel inputs/outputs,
Eq. 5-10 (L165-189) cold-plasma dispersion, L60 spline equilibria, L159 launch conditions.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rt_oracle.cpp"
_LIB = _HERE / "librt_oracle.so"

EQ_SLAB_PARABOLIC, EQ_SLAB_LINEAR_BR, EQ_TOKAMAK_CIRCULAR, EQ_GRID_RZ = 0, 1, 2, 3
DISP_OMODE, DISP_XMODE, DISP_COLD_FULL = 0, 1, 2
EQ_KINDS = {"slab_parabolic": 0, "slab_linear_br": 1, "tokamak_circular": 2, "grid_rz": 3}
DISP_KINDS = {"omode": 0, "xmode": 1, "cold_full": 2}


def build(force: bool = False) -> Path:
    """Compile rt_oracle.cpp into librt_oracle.so (g++ -O2 -fopenmp, no FMA contraction)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wno-misleading-indentation", str(_SRC), "-o", str(tmp)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _CEq(ctypes.Structure):
    _fields_ = [
        ("kind", ctypes.c_int32), ("nR", ctypes.c_int32), ("nZ", ctypes.c_int32), ("nPsi", ctypes.c_int32),
        ("n_ref", ctypes.c_double), ("L", ctypes.c_double),
        ("x_foot", ctypes.c_double), ("L_ramp", ctypes.c_double), ("B0", ctypes.c_double), ("R0", ctypes.c_double),
        ("a", ctypes.c_double), ("q0", ctypes.c_double), ("q1", ctypes.c_double), ("p_exp", ctypes.c_double),
        ("rho_max", ctypes.c_double),
        ("Rmin", ctypes.c_double), ("Rmax", ctypes.c_double), ("Zmin", ctypes.c_double), ("Zmax", ctypes.c_double),
        ("psi_min", ctypes.c_double), ("psi_max", ctypes.c_double),
        ("psi_pp", ctypes.c_void_p), ("F_pp", ctypes.c_void_p), ("ne_pp", ctypes.c_void_p),
        ("ion_mass", ctypes.c_double), ("ion_charge", ctypes.c_double),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        # RT_ORACLE_LIB: load an alternative build of rt_oracle.cpp (tests/test_sanitizers.py: the ASan / UBSan build)
        lib = ctypes.CDLL(os.environ.get("RT_ORACLE_LIB") or str(build()))
        P, D, I64, I32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int64, ctypes.c_int
        lib.oracle_trace.argtypes = [ctypes.POINTER(_CEq), I32, P, P, D, I64, I64, D, I64, P, P, P, P, I32]
        lib.oracle_trace_w.argtypes = [ctypes.POINTER(_CEq), I32, P, P, P, I64, I64, D, I64, P, P, P, P, I32]
        lib.oracle_trace_until.argtypes = [ctypes.POINTER(_CEq), I32, P, P, D, I64, I64, I64, D, D, P, P, P, P, P, I32]
        lib.oracle_launch_w.argtypes = [ctypes.POINTER(_CEq), I32, I32, P, P, P, I64, P, P]
        lib.oracle_diagnostics.argtypes = [ctypes.POINTER(_CEq), P, P, P, I64, P]
        lib.oracle_orbit.argtypes = [ctypes.POINTER(_CEq), P, P, D, I64, I64, D, I64, P, P, P, P, I32]
        lib.oracle_dispersion.argtypes = [ctypes.POINTER(_CEq), I32, P, P, D, I64, P, P, P]
        lib.oracle_dispersion_value.argtypes = [ctypes.POINTER(_CEq), I32, P, P, P, I64, P]
        lib.oracle_plasma.argtypes = [ctypes.POINTER(_CEq), P, D, I64, P, P, P, P]
        lib.oracle_launch.argtypes = [ctypes.POINTER(_CEq), I32, I32, P, P, D, I64, P, P]
        lib.oracle_launch_kx.argtypes = [ctypes.POINTER(_CEq), I32, P, P, D, P, I64, I32, D, P, P, P]
        lib.oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def fit_bicubic_pp(psi: np.ndarray, R: np.ndarray, Z: np.ndarray) -> np.ndarray:
    """Tensor-product not-a-knot cubic spline of nodal psi[iR, iZ] as pieces pp[iR, iZ, p, q] multiplying
    (R-R_i)^p (Z-Z_j)^q.  The 1-D not-a-knot interpolation operator is linear, so the tensor-product
    spline is the R-spline of the Z-spline's coefficients (reading A10)."""
    from scipy.interpolate import CubicSpline
    cz = CubicSpline(Z, psi, axis=1).c                       # (4, nZ-1, nR): power 3-k of (Z-Z_j), per R node
    cr = CubicSpline(R, np.moveaxis(cz, 2, 0), axis=0).c     # (4, nR-1, 4, nZ-1)
    pp = np.transpose(cr[::-1, :, ::-1, :], (1, 3, 0, 2))    # (nR-1, nZ-1, p, q), ascending powers
    return np.ascontiguousarray(pp, dtype=np.float64)


def fit_cubic_pp(y: np.ndarray, x: np.ndarray) -> np.ndarray:
    """Not-a-knot cubic spline of nodal y[i] as pieces pp[i, m] multiplying (x-x_i)^m."""
    from scipy.interpolate import CubicSpline
    c = CubicSpline(x, y).c                                  # (4, n-1), power 3-k
    return np.ascontiguousarray(c[::-1, :].T, dtype=np.float64)


class Equilibrium:
    """Holds the C descriptor (and the spline pieces it points to) for the oracle.

    ``desc`` is the plain dict produced by ``paper_2508_15967_b200.inputs`` (numbers and nodal arrays only)."""

    def __init__(self, desc: dict):
        d = dict(desc)
        kind = d["kind"]
        self.kind = EQ_KINDS[kind] if isinstance(kind, str) else int(kind)
        c = _CEq()
        c.kind = self.kind
        for name in ("n_ref", "L", "x_foot", "L_ramp", "B0", "R0", "a", "q0", "q1", "p_exp",
                     "Rmin", "Rmax", "Zmin", "Zmax", "psi_min", "psi_max", "ion_mass", "ion_charge"):
            setattr(c, name, float(d.get(name, 0.0)))
        c.rho_max = float(d.get("rho_max", 0.98))
        self._keep = []
        if self.kind == EQ_GRID_RZ:
            psi = np.asarray(d["psi_RZ"], dtype=np.float64)
            F = np.asarray(d["F_psi"], dtype=np.float64)
            ne = np.asarray(d["ne_psi"], dtype=np.float64)
            c.nR, c.nZ, c.nPsi = psi.shape[0], psi.shape[1], F.shape[0]
            # node coordinates exactly as rt_oracle.cpp computes them (Rmin + i*h), so offsets agree
            Rg = c.Rmin + np.arange(c.nR) * ((c.Rmax - c.Rmin) / (c.nR - 1))
            Zg = c.Zmin + np.arange(c.nZ) * ((c.Zmax - c.Zmin) / (c.nZ - 1))
            Pg = c.psi_min + np.arange(c.nPsi) * ((c.psi_max - c.psi_min) / (c.nPsi - 1))
            self.psi_pp = fit_bicubic_pp(psi, Rg, Zg)
            self.F_pp = fit_cubic_pp(F, Pg)
            self.ne_pp = fit_cubic_pp(ne, Pg)
            self._keep = [self.psi_pp, self.F_pp, self.ne_pp]
            c.psi_pp = self.psi_pp.ctypes.data
            c.F_pp = self.F_pp.ctypes.data
            c.ne_pp = self.ne_pp.ctypes.data
        self.c = c


def _eq(eq) -> Equilibrium:
    return eq if isinstance(eq, Equilibrium) else Equilibrium(eq)


def _disp(disp) -> int:
    return DISP_KINDS[disp] if isinstance(disp, str) else int(disp)


def _soa(a, n=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.ndim == 2 and a.shape[0] == 3, a.shape
    return a


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def trace(eq, disp, x0, k0, omega, n_steps, dt, save_stride=1, *, traj=False, final=True, residual=True,
          status=True, n_threads=0) -> dict:
    """Integrate the ray equations; returns a dict with 'traj' [n_saved,6,n], 'final' [6,n],
    'residual' ([n_saved,n] with traj else [n]) and 'status' [n] for the outputs requested.
    ``omega`` is one frequency for all rays or an array [n] with one frequency per ray (L147)."""
    lib, e = _load(), _eq(eq)
    x0, k0 = _soa(x0), _soa(k0)
    n = x0.shape[1]
    per_ray = np.ndim(omega) > 0
    if per_ray:
        omega = np.ascontiguousarray(omega, dtype=np.float64)
        assert omega.shape == (n,), omega.shape
    n_saved = n_steps // save_stride + 1
    out = {}
    if traj:
        out["traj"] = np.empty((n_saved, 6, n))
    if final:
        out["final"] = np.empty((6, n))
    if residual:
        out["residual"] = np.empty((n_saved, n) if traj else (n,))
    if status:
        out["status"] = np.empty((n,), dtype=np.int32)
    ptr = lambda key: out[key].ctypes.data if key in out else None
    fn, w = (lib.oracle_trace_w, omega.ctypes.data) if per_ray else (lib.oracle_trace, float(omega))
    rc = fn(ctypes.byref(e.c), _disp(disp), x0.ctypes.data, k0.ctypes.data, w, n,
            int(n_steps), float(dt), int(save_stride), ptr("traj"), ptr("final"), ptr("residual"),
            ptr("status"), int(n_threads))
    if rc != 0:
        raise ValueError(f"oracle_trace rejected its arguments (rc={rc})")
    return out


def trace_until(eq, disp, x0, k0, omega, chunk_steps, max_chunks, dt, tol=np.inf, n_threads=0) -> dict:
    """The convergence workflow (L80): advance the ensemble in chunks of ``chunk_steps`` steps until every
    ray is frozen, max |D| exceeds ``tol``, or ``max_chunks`` chunks have run.  Returns 'final' [6,n], 'residual' [n],
    'status' [n], 'chunks', 'n_active', 'reason' (0 max_chunks, 1 all frozen, 2 tolerance exceeded) and 'max_D'."""
    lib, e = _load(), _eq(eq)
    x0, k0 = _soa(x0), _soa(k0)
    n = x0.shape[1]
    fin, res, st = np.empty((6, n)), np.empty(n), np.empty(n, dtype=np.int32)
    info, mx = np.zeros(4, dtype=np.int64), np.zeros(1)
    rc = lib.oracle_trace_until(ctypes.byref(e.c), _disp(disp), x0.ctypes.data, k0.ctypes.data, float(omega), n,
                                int(chunk_steps), int(max_chunks), float(dt), float(tol), fin.ctypes.data, res.ctypes.data,
                                st.ctypes.data, info.ctypes.data, mx.ctypes.data, int(n_threads))
    if rc != 0:
        raise ValueError(f"oracle_trace_until rejected its arguments (rc={rc})")
    return dict(final=fin, residual=res, status=st, chunks=int(info[0]), n_active=int(info[1]), reason=int(info[2]),
                max_D=float(mx[0]))


def dispersion(eq, disp, x, k, omega):
    """D, its 7 partials (x,y,z,kx,ky,kz,w) and the inside-domain flag at points x,k [3,n]."""
    lib, e = _load(), _eq(eq)
    x, k = _soa(x), _soa(k)
    n = x.shape[1]
    D, g, ins = np.empty(n), np.empty((7, n)), np.empty(n, dtype=np.int32)
    rc = lib.oracle_dispersion(ctypes.byref(e.c), _disp(disp), x.ctypes.data, k.ctypes.data, float(omega), n,
                               D.ctypes.data, g.ctypes.data, ins.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_dispersion rejected its arguments")
    return D, g, ins


def dispersion_value(eq, disp, x, k, omega):
    """D alone in plain double arithmetic; omega may be a scalar or an [n] array."""
    lib, e = _load(), _eq(eq)
    x, k = _soa(x), _soa(k)
    n = x.shape[1]
    w = np.ascontiguousarray(np.broadcast_to(np.asarray(omega, dtype=np.float64), (n,)))
    D = np.empty(n)
    rc = lib.oracle_dispersion_value(ctypes.byref(e.c), _disp(disp), x.ctypes.data, k.ctypes.data, w.ctypes.data,
                                     n, D.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_dispersion_value rejected its arguments")
    return D


def plasma(eq, x, omega):
    """n_e [n], B [3,n], (S, Dx, P) [3,n] and the inside flag [n] at points x [3,n]."""
    lib, e = _load(), _eq(eq)
    x = _soa(x)
    n = x.shape[1]
    ne, B, sdp, ins = np.empty(n), np.empty((3, n)), np.empty((3, n)), np.empty(n, dtype=np.int32)
    rc = lib.oracle_plasma(ctypes.byref(e.c), x.ctypes.data, float(omega), n, ne.ctypes.data, B.ctypes.data,
                           sdp.ctypes.data, ins.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_plasma rejected its arguments")
    return ne, B, sdp, ins


def launch(eq, disp, x0, dirs, omega, branch=0):
    """On-shell launch wave vectors k0 [3,n] along unit directions dirs [3,n] (L159); also returns D there.
    ``omega``: a scalar or one frequency per ray [n]."""
    lib, e = _load(), _eq(eq)
    x0, dirs = _soa(x0), _soa(dirs)
    n = x0.shape[1]
    k0, D = np.empty((3, n)), np.empty(n)
    if np.ndim(omega) > 0:
        w = np.ascontiguousarray(omega, dtype=np.float64)
        assert w.shape == (n,), w.shape
        rc = lib.oracle_launch_w(ctypes.byref(e.c), _disp(disp), int(branch), x0.ctypes.data, dirs.ctypes.data,
                                 w.ctypes.data, n, k0.ctypes.data, D.ctypes.data)
    else:
        rc = lib.oracle_launch(ctypes.byref(e.c), _disp(disp), int(branch), x0.ctypes.data, dirs.ctypes.data,
                               float(omega), n, k0.ctypes.data, D.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_launch rejected its arguments")
    return k0, D


def launch_kx(eq, disp, x0, k_guess, omega, max_iter=50, tol=1e-15):
    """The paper's own launch iteration (L159): w, x, k_y, k_z fixed (rows 1, 2 of ``k_guess`` [3,n]); k_x found by
    Newton's method from the initial guess in row 0, which selects the root, until |D| < tol.  Returns (k0 [3,n], D [n],
    iters [n]: Newton updates used, -1 = not converged / outside the domain).  ``omega``: scalar or per ray [n]."""
    lib, e = _load(), _eq(eq)
    x0, kg = _soa(x0), _soa(k_guess)
    n = x0.shape[1]
    k0, D, it = np.empty((3, n)), np.empty(n), np.empty(n, dtype=np.int32)
    w = None
    if np.ndim(omega) > 0:
        w = np.ascontiguousarray(omega, dtype=np.float64)
        assert w.shape == (n,), w.shape
    rc = lib.oracle_launch_kx(ctypes.byref(e.c), _disp(disp), x0.ctypes.data, kg.ctypes.data,
                              0.0 if w is not None else float(omega), w.ctypes.data if w is not None else None, n,
                              int(max_iter), float(tol), k0.ctypes.data, D.ctypes.data, it.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_launch_kx rejected its arguments")
    return k0, D, it


DIAG_ROWS = ("n_e", "B", "X", "Y", "S", "D", "P", "R", "L", "n_par2")


def diagnostics(eq, x, k, omega):
    """Critical-surface diagnostics (L149, Fig. 3-4) at points x, k [3,n]: array [10,n] with rows ``DIAG_ROWS``;
    ``omega`` a scalar or one frequency per point [n]."""
    lib, e = _load(), _eq(eq)
    x, k = _soa(x), _soa(k)
    n = x.shape[1]
    w = np.ascontiguousarray(np.broadcast_to(np.asarray(omega, dtype=np.float64), (n,)))
    out = np.empty((10, n))
    rc = lib.oracle_diagnostics(ctypes.byref(e.c), x.ctypes.data, k.ctypes.data, w.ctypes.data, n, out.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_diagnostics rejected its arguments")
    return out


def orbit(eq, x0, v0, charge_over_mass, n_steps, dt, save_stride=1, *, traj=False, final=True, drift=True, status=True,
          n_threads=0) -> dict:
    """Full-orbit particles (L121, L213): dx/dt = v, dv/dt = (q/m) v x B(x), classical RK4 with step dt [s].
    x0, v0 [3,n]; returns 'traj' [n_saved,6,n], 'final' [6,n], 'drift' (|v|^2/|v0|^2 - 1; [n_saved,n] with traj else [n])
    and 'status' [n] for the outputs requested."""
    lib, e = _load(), _eq(eq)
    x0, v0 = _soa(x0), _soa(v0)
    n = x0.shape[1]
    n_saved = n_steps // save_stride + 1
    out = {}
    if traj:
        out["traj"] = np.empty((n_saved, 6, n))
    if final:
        out["final"] = np.empty((6, n))
    if drift:
        out["drift"] = np.empty((n_saved, n) if traj else (n,))
    if status:
        out["status"] = np.empty((n,), dtype=np.int32)
    ptr = lambda key: out[key].ctypes.data if key in out else None
    rc = lib.oracle_orbit(ctypes.byref(e.c), x0.ctypes.data, v0.ctypes.data, float(charge_over_mass), n, int(n_steps),
                          float(dt), int(save_stride), ptr("traj"), ptr("final"), ptr("drift"), ptr("status"), int(n_threads))
    if rc != 0:
        raise ValueError(f"oracle_orbit rejected its arguments (rc={rc})")
    return out
