"""Thin ctypes binding of the C-ABI library declared in ``include/rt.h`` -- argument marshalling only.

Every step of the hot path (RK4 on the ray equations Eq. 2-3; Eq. 5-10 dispersion; L60 spline
equilibria; L159 launch conditions) runs inside ``librt_b200.so``'s sm_100a kernels.  This module turns torch tensors
into raw device pointers + the current CUDA stream, turns an equilibrium dict into ``rt_equilibrium_desc``, and raises
``RtError`` on a non-zero return.  There is no CPU fallback: if the library is missing, ``load()`` raises.

Function names mirror the C ABI: ``create_equilibrium / destroy / trace / trace_host / launch / rhs / reduce /
fma_peak / launch_count``.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "librt_b200.so"

RT_OK, RT_ERR_INVALID, RT_ERR_UNSUPPORTED, RT_ERR_CUDA, RT_ERR_NOMEM = 0, -1, -2, -3, -4
EQ_KINDS = {"slab_parabolic": 0, "slab_linear_br": 1, "tokamak_circular": 2, "grid_rz": 3}
DISP_KINDS = {"omode": 0, "xmode": 1, "cold_full": 2}
PRECISIONS = {"f64": 0, "f32": 1}

# every symbol include/rt.h declares (tests check the library exports each of them)
SYMBOLS = ("rt_create_equilibrium", "rt_destroy", "rt_trace", "rt_trace_w", "rt_trace_host", "rt_trace_host_noalloc", "rt_trace_until", "rt_launch", "rt_launch_w",
           "rt_launch_kx", "rt_diagnostics", "rt_orbit", "rt_rhs", "rt_reduce", "rt_fma_peak", "rt_fma_peak_shape", "rt_math_probe", "rt_launch_count", "rt_last_error", "rt_version")
NDIAG = 10
DIAG_ROWS = ("n_e", "B", "X", "Y", "S", "D", "P", "R", "L", "n_par2")


class RtError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"rt error {code}: {msg}")
        self.code = code


class EquilibriumDesc(ctypes.Structure):
    """Mirror of ``rt_equilibrium_desc`` (include/rt.h)."""
    _fields_ = [
        ("kind", ctypes.c_int32), ("nR", ctypes.c_int32), ("nZ", ctypes.c_int32), ("nPsi", ctypes.c_int32),
        ("n_ref", ctypes.c_double), ("L", ctypes.c_double),
        ("x_foot", ctypes.c_double), ("L_ramp", ctypes.c_double), ("B0", ctypes.c_double), ("R0", ctypes.c_double),
        ("a", ctypes.c_double), ("q0", ctypes.c_double), ("q1", ctypes.c_double), ("p_exp", ctypes.c_double),
        ("rho_max", ctypes.c_double),
        ("Rmin", ctypes.c_double), ("Rmax", ctypes.c_double), ("Zmin", ctypes.c_double), ("Zmax", ctypes.c_double),
        ("psi_min", ctypes.c_double), ("psi_max", ctypes.c_double),
        ("psi_RZ", ctypes.c_void_p), ("F_psi", ctypes.c_void_p), ("ne_psi", ctypes.c_void_p),
        ("ion_mass", ctypes.c_double), ("ion_charge", ctypes.c_double),
    ]


_SCALARS = ("n_ref", "L", "x_foot", "L_ramp", "B0", "R0", "a", "q0", "q1", "p_exp", "rho_max", "Rmin", "Rmax", "Zmin",
            "Zmax", "psi_min", "psi_max", "ion_mass", "ion_charge")


def make_desc(eq: dict):
    """Equilibrium dict (``inputs.py``) -> (EquilibriumDesc, keep-alive list of the nodal numpy arrays)."""
    d = EquilibriumDesc()
    kind = eq["kind"]
    d.kind = EQ_KINDS[kind] if isinstance(kind, str) else int(kind)
    for name in _SCALARS:
        setattr(d, name, float(eq.get(name, 0.0)))
    keep = []
    if d.kind == EQ_KINDS["grid_rz"]:
        psi = np.ascontiguousarray(eq["psi_RZ"], dtype=np.float64)
        F = np.ascontiguousarray(eq["F_psi"], dtype=np.float64)
        ne = np.ascontiguousarray(eq["ne_psi"], dtype=np.float64)
        if psi.ndim != 2 or F.ndim != 1 or ne.shape != F.shape:
            raise ValueError("grid_rz: psi_RZ must be [nR, nZ]; F_psi and ne_psi must be [nPsi]")
        d.nR, d.nZ, d.nPsi = psi.shape[0], psi.shape[1], F.shape[0]
        d.psi_RZ, d.F_psi, d.ne_psi = psi.ctypes.data, F.ctypes.data, ne.ctypes.data
        keep = [psi, F, ne]
    return d, keep


_lib = None


def load() -> ctypes.CDLL:
    """Load librt_b200.so (built in-tree by ``paper_2508_15967_b200.build``).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RtError(RT_ERR_CUDA, f"{LIB_PATH} is missing: build it with `python -m paper_2508_15967_b200.build` "
                                       "(there is no CPU fallback)")
        lib = ctypes.CDLL(str(LIB_PATH))
        P, D, I64, I32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int64, ctypes.c_int
        lib.rt_create_equilibrium.argtypes = [ctypes.POINTER(EquilibriumDesc), ctypes.POINTER(P)]
        lib.rt_destroy.argtypes = [P]
        lib.rt_trace.argtypes = [P, I32, I32, P, P, D, I64, I64, D, I64, P, P, P, P, P]
        lib.rt_trace_w.argtypes = [P, I32, I32, P, P, P, I64, I64, D, I64, P, P, P, P, P]
        lib.rt_trace_until.argtypes = [P, I32, I32, P, P, D, I64, I64, I64, D, D, P, P, P, P, P]
        lib.rt_launch_w.argtypes = [P, I32, I32, P, P, P, I64, P, P, P]
        lib.rt_diagnostics.argtypes = [P, P, P, D, P, I64, P, P]
        lib.rt_launch_kx.argtypes = [P, I32, P, P, D, P, I64, I32, D, P, P, P, P]
        lib.rt_orbit.argtypes = [P, I32, P, P, D, I64, I64, D, I64, P, P, P, P, P]
        lib.rt_trace_host.argtypes = [P, I32, I32, P, P, D, I64, I64, D, I64, P, P, P, P]
        lib.rt_trace_host_noalloc.argtypes = [P, I32, I32, P, P, D, I64, I64, D, I64, P, P, P, P, P]
        lib.rt_launch.argtypes = [P, I32, I32, P, P, D, I64, P, P, P]
        lib.rt_rhs.argtypes = [P, I32, I32, P, P, D, I64, P, P, P, P]
        lib.rt_reduce.argtypes = [I32, P, P, I64, P, P]
        lib.rt_fma_peak.argtypes = [I32, D, ctypes.POINTER(D), ctypes.POINTER(D)]
        lib.rt_fma_peak_shape.argtypes = [I32, I32, I32, D, ctypes.POINTER(D), ctypes.POINTER(D)]
        lib.rt_math_probe.argtypes = [I32, I32, P, I64, P, P]
        lib.rt_launch_count.restype = I64
        lib.rt_last_error.restype = ctypes.c_char_p
        lib.rt_version.restype = ctypes.c_char_p
        for name in SYMBOLS:
            fn = getattr(lib, name)
            if name not in ("rt_launch_count", "rt_last_error", "rt_version"):
                fn.restype = I32
        _lib = lib
    return _lib


def _check(rc: int):
    if rc != 0:
        raise RtError(rc, load().rt_last_error().decode())


def version() -> str:
    return load().rt_version().decode()


def launch_count() -> int:
    return int(load().rt_launch_count())


class Equilibrium:
    """Owns an ``rt_equilibrium*``."""

    def __init__(self, eq: dict):
        lib = load()
        desc, keep = make_desc(eq)
        h = ctypes.c_void_p()
        _check(lib.rt_create_equilibrium(ctypes.byref(desc), ctypes.byref(h)))
        self.handle = h
        self.kind = desc.kind

    def close(self):
        if getattr(self, "handle", None):
            load().rt_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def create_equilibrium(eq: dict) -> Equilibrium:
    return Equilibrium(eq)


def destroy(eq: Equilibrium):
    eq.close()


def _disp(disp) -> int:
    return DISP_KINDS[disp] if isinstance(disp, str) else int(disp)


def _prec_of(t) -> int:
    import torch
    if t.dtype == torch.float64:
        return 0
    if t.dtype == torch.float32:
        return 1
    raise TypeError(f"ray buffers must be float64 or float32, got {t.dtype}")


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _dev_soa(t, rows, n=None):
    if not t.is_cuda or not t.is_contiguous() or t.dim() != 2 or t.shape[0] != rows or (n is not None and t.shape[1] != n):
        raise ValueError(f"expected a contiguous CUDA tensor of shape [{rows}, {n if n is not None else 'n'}], got "
                         f"{tuple(t.shape)} on {t.device}")
    return t


def _omega_rays(omega, n):
    """None for a scalar frequency, else the validated per-ray tensor (float64 CUDA [n])."""
    import torch
    if not torch.is_tensor(omega):
        return None
    if not omega.is_cuda or omega.dtype != torch.float64 or not omega.is_contiguous() or tuple(omega.shape) != (n,):
        raise ValueError(f"per-ray omega must be a contiguous float64 CUDA tensor of shape [{n}]")
    return omega


def trace(eq: Equilibrium, disp, x0, k0, omega, n_steps: int, dt: float, save_stride: int = 1, *, traj=False,
          final=True, residual=True, status=True, out: dict | None = None) -> dict:
    """``rt_trace`` (``rt_trace_w`` when ``omega`` is a float64 CUDA tensor [n_rays]) on the current CUDA stream.
    x0, k0: CUDA tensors [3, n_rays] (float64 or float32).  Returns a dict
    of freshly allocated (or, via ``out``, caller-provided) device tensors: 'traj' [n_saved, 6, n], 'final' [6, n],
    'residual' ([n_saved, n] with traj else [n]), 'status' [n] int32.  Does not synchronise."""
    import torch
    lib = load()
    x0 = _dev_soa(x0, 3)
    n = x0.shape[1]
    k0 = _dev_soa(k0, 3, n)
    if k0.dtype != x0.dtype:
        raise TypeError("x0 and k0 must have the same dtype")
    prec = _prec_of(x0)
    n_saved = n_steps // save_stride + 1 if traj else 0
    o = {} if out is None else out
    kw = dict(dtype=x0.dtype, device=x0.device)
    if traj and "traj" not in o:
        o["traj"] = torch.empty((n_saved, 6, n), **kw)
    if final and "final" not in o:
        o["final"] = torch.empty((6, n), **kw)
    if residual and "residual" not in o:
        o["residual"] = torch.empty((n_saved, n) if traj else (n,), **kw)
    if status and "status" not in o:
        o["status"] = torch.empty((n,), dtype=torch.int32, device=x0.device)
    outs = (_ptr(o.get("traj") if traj else None), _ptr(o.get("final") if final else None),
            _ptr(o.get("residual") if residual else None), _ptr(o.get("status") if status else None))
    w = _omega_rays(omega, n)
    if w is None:
        _check(lib.rt_trace(eq.handle, _disp(disp), prec, _ptr(x0), _ptr(k0), float(omega), n, int(n_steps), float(dt),
                            int(save_stride), *outs, _stream()))
    else:
        _check(lib.rt_trace_w(eq.handle, _disp(disp), prec, _ptr(x0), _ptr(k0), _ptr(w), n, int(n_steps), float(dt),
                              int(save_stride), *outs, _stream()))
    return o


UNTIL_INFO_WORDS = 16
UNTIL_REASONS = ("max_chunks", "all_frozen", "tolerance")


def trace_until(eq: Equilibrium, disp, x0, k0, omega: float, chunk_steps: int, max_chunks: int, dt: float,
                tol: float = float("inf"), out: dict | None = None) -> dict:
    """``rt_trace_until`` on the current CUDA stream: advance the ensemble in chunks of ``chunk_steps`` steps until every
    ray is frozen, max |D| > ``tol`` or ``max_chunks`` chunks have run; the loop runs on the device (CUDA-graph WHILE node)
    and the call does not synchronise.  Returns device tensors 'final' [6, n], 'residual' [n], 'status' [n] int32 and
    'info' int64 [16] (see ``until_info``)."""
    import torch
    lib = load()
    x0 = _dev_soa(x0, 3)
    n = x0.shape[1]
    k0 = _dev_soa(k0, 3, n)
    if k0.dtype != x0.dtype:
        raise TypeError("x0 and k0 must have the same dtype")
    o = {} if out is None else out
    o.setdefault("final", torch.empty((6, n), dtype=x0.dtype, device=x0.device))
    o.setdefault("residual", torch.empty((n,), dtype=x0.dtype, device=x0.device))
    o.setdefault("status", torch.empty((n,), dtype=torch.int32, device=x0.device))
    o.setdefault("info", torch.empty((UNTIL_INFO_WORDS,), dtype=torch.int64, device=x0.device))
    _check(lib.rt_trace_until(eq.handle, _disp(disp), _prec_of(x0), _ptr(x0), _ptr(k0), float(omega), n, int(chunk_steps),
                              int(max_chunks), float(dt), float(tol), _ptr(o["final"]), _ptr(o["residual"]),
                              _ptr(o["status"]), _ptr(o["info"]), _stream()))
    return o


def until_info(info) -> dict:
    """Decode ``rt_trace_until``'s out_info (synchronises: it copies the 16 words to the host)."""
    import torch
    h = info.cpu()
    return dict(chunks=int(h[0]), n_active=int(h[1]), max_D=float(h[2:3].view(torch.float64)[0]), reason=int(h[3]))


def trace_host(eq: Equilibrium, disp, x0, k0, omega: float, n_steps: int, dt: float, save_stride: int = 1, *,
               traj=False, final=True, residual=True, status=True, out: dict | None = None) -> dict:
    """``rt_trace_host``: x0, k0 and all outputs are HOST arrays (numpy, or CPU torch tensors -- pinned memory makes
    the copies asynchronous).  Returns when the results are in host memory."""
    lib = load()
    is_torch = not isinstance(x0, np.ndarray)

    def hp(a):
        if a is None:
            return None
        return ctypes.c_void_p(a.data_ptr() if is_torch else a.ctypes.data)

    n = x0.shape[1]
    if is_torch:
        import torch
        if x0.is_cuda or k0.is_cuda or not x0.is_contiguous() or not k0.is_contiguous():
            raise ValueError("trace_host wants contiguous CPU tensors")
        prec = _prec_of(x0)
        empty = lambda shape, dtype=x0.dtype: torch.empty(shape, dtype=dtype)
        i32 = torch.int32
    else:
        x0 = np.ascontiguousarray(x0)
        k0 = np.ascontiguousarray(k0)
        prec = {np.dtype(np.float64): 0, np.dtype(np.float32): 1}[x0.dtype]
        empty = lambda shape, dtype=x0.dtype: np.empty(shape, dtype=dtype)
        i32 = np.int32
    if tuple(x0.shape) != (3, n) or tuple(k0.shape) != (3, n) or k0.dtype != x0.dtype:
        raise ValueError("x0, k0 must both be [3, n] of the same dtype")
    n_saved = n_steps // save_stride + 1 if traj else 0
    o = {} if out is None else out
    if traj and "traj" not in o:
        o["traj"] = empty((n_saved, 6, n))
    if final and "final" not in o:
        o["final"] = empty((6, n))
    if residual and "residual" not in o:
        o["residual"] = empty((n_saved, n) if traj else (n,))
    if status and "status" not in o:
        o["status"] = empty((n,), i32)
    _check(lib.rt_trace_host(eq.handle, _disp(disp), prec, hp(x0), hp(k0), float(omega), n, int(n_steps), float(dt),
                             int(save_stride), hp(o.get("traj") if traj else None), hp(o.get("final") if final else None),
                             hp(o.get("residual") if residual else None), hp(o.get("status") if status else None)))
    return o


NOALLOC_SCRATCH_BYTES = 64 << 20          # RT_NOALLOC_SCRATCH_BYTES (include/rt.h)


def trace_host_noalloc(eq: Equilibrium, disp, x0, k0, omega: float, n_steps: int, dt: float, save_stride: int = 1, *,
                       traj=False, final=True, residual=True, status=True, out: dict | None = None) -> dict:
    """``rt_trace_host_noalloc``: ``trace_host`` for a program that must not allocate device memory when it calls the
    library -- one that keeps the whole GPU in its own memory pool, one that cannot stand the device-wide stall of a
    cudaMalloc / cudaFree in the middle of its run, or one whose device memory is fixed before it starts.  The rays and
    their results are staged in a 64 MiB array built into the library (``NOALLOC_SCRATCH_BYTES``) instead of in buffers
    from cudaMalloc, so the whole call has to fit in it at once: a larger one raises ``RtError`` (``RT_ERR_INVALID``).
    x0, k0 and the outputs are HOST arrays (numpy, or CPU torch tensors) as for ``trace_host``, and the results are the
    same bits.  The work is enqueued on torch's current stream (numpy arrays: on the default stream) and the call returns
    when the results are in host memory.  Make the first call on each device outside any stream capture;
    never run two calls at the same time on one device -- they share the array (include/rt.h has the details).
    Only the C call is allocation-free: host output arrays that are not passed in through ``out`` are created here."""
    lib = load()
    is_torch = not isinstance(x0, np.ndarray)
    if is_torch:
        import torch
        if x0.is_cuda or k0.is_cuda or not x0.is_contiguous() or not k0.is_contiguous():
            raise ValueError("trace_host_noalloc wants contiguous CPU tensors")
        prec = _prec_of(x0)
        empty = lambda shape, dtype=x0.dtype: torch.empty(shape, dtype=dtype)
        i32 = torch.int32
        hp = lambda a: None if a is None else ctypes.c_void_p(a.data_ptr())
    else:
        x0, k0 = np.ascontiguousarray(x0), np.ascontiguousarray(k0)
        prec = {np.dtype(np.float64): 0, np.dtype(np.float32): 1}[x0.dtype]
        empty = lambda shape, dtype=x0.dtype: np.empty(shape, dtype=dtype)
        i32 = np.int32
        hp = lambda a: None if a is None else ctypes.c_void_p(a.ctypes.data)
    n = x0.shape[1]
    if tuple(x0.shape) != (3, n) or tuple(k0.shape) != (3, n) or k0.dtype != x0.dtype:
        raise ValueError("x0, k0 must both be [3, n] of the same dtype")
    n_saved = n_steps // save_stride + 1 if traj else 0
    o = {} if out is None else out
    shapes = {"traj": (n_saved, 6, n), "final": (6, n), "residual": (n_saved, n) if traj else (n,), "status": (n,)}
    wanted = {"traj": traj, "final": final, "residual": residual, "status": status}
    for key, want in wanted.items():
        if want and key not in o:
            o[key] = empty(shapes[key], i32) if key == "status" else empty(shapes[key])
    arg = lambda key: hp(o[key]) if wanted[key] else None
    _check(lib.rt_trace_host_noalloc(eq.handle, _disp(disp), prec, hp(x0), hp(k0), float(omega), n, int(n_steps), float(dt),
                                     int(save_stride), arg("traj"), arg("final"), arg("residual"), arg("status"),
                                     _stream() if is_torch else None))
    return o


def launch(eq: Equilibrium, disp, x0, dirs, omega, branch: int = 0):
    """``rt_launch`` (``rt_launch_w`` when ``omega`` is a float64 CUDA tensor [n]): on-shell k0 [3, n] along unit
    directions dirs [3, n] from positions x0 (float64 CUDA tensors); also returns D at the launch state."""
    import torch
    lib = load()
    x0 = _dev_soa(x0, 3)
    n = x0.shape[1]
    dirs = _dev_soa(dirs, 3, n)
    if x0.dtype != torch.float64 or dirs.dtype != torch.float64:
        raise TypeError("rt_launch is fp64 only")
    k0 = torch.empty((3, n), dtype=torch.float64, device=x0.device)
    D = torch.empty((n,), dtype=torch.float64, device=x0.device)
    w = _omega_rays(omega, n)
    if w is None:
        _check(lib.rt_launch(eq.handle, _disp(disp), int(branch), _ptr(x0), _ptr(dirs), float(omega), n, _ptr(k0), _ptr(D),
                             _stream()))
    else:
        _check(lib.rt_launch_w(eq.handle, _disp(disp), int(branch), _ptr(x0), _ptr(dirs), _ptr(w), n, _ptr(k0), _ptr(D),
                               _stream()))
    return k0, D


def launch_kx(eq: Equilibrium, disp, x0, k_guess, omega, max_iter: int = 50, tol: float = 1e-15):
    """``rt_launch_kx``: the paper's own launch iteration.  ``k_guess`` [3, n] float64 CUDA tensor: rows 1, 2
    the fixed k_y, k_z, row 0 the initial guess for k_x; ``omega`` a float or a float64 CUDA tensor [n].  Returns
    (k0 [3, n], D [n], iters int32 [n]: Newton updates used, -1 = tolerance not reached)."""
    import torch
    lib = load()
    x0 = _dev_soa(x0, 3)
    n = x0.shape[1]
    kg = _dev_soa(k_guess, 3, n)
    if x0.dtype != torch.float64 or kg.dtype != torch.float64:
        raise TypeError("rt_launch_kx is fp64 only")
    k0 = torch.empty((3, n), dtype=torch.float64, device=x0.device)
    D = torch.empty((n,), dtype=torch.float64, device=x0.device)
    it = torch.empty((n,), dtype=torch.int32, device=x0.device)
    w = _omega_rays(omega, n)
    _check(lib.rt_launch_kx(eq.handle, _disp(disp), _ptr(x0), _ptr(kg), 0.0 if w is not None else float(omega), _ptr(w), n,
                            int(max_iter), float(tol), _ptr(k0), _ptr(D), _ptr(it), _stream()))
    return k0, D, it


def diagnostics(eq: Equilibrium, x, k, omega):
    """``rt_diagnostics``: [NDIAG, n] float64 device tensor, rows ``DIAG_ROWS`` (n_e, |B|, X, Y, S, D, P, R, L, n_par^2)
    at points x, k [3, n] (float64 CUDA tensors); ``omega`` a float or a float64 CUDA tensor [n]."""
    import torch
    lib = load()
    x = _dev_soa(x, 3)
    n = x.shape[1]
    k = _dev_soa(k, 3, n)
    if x.dtype != torch.float64 or k.dtype != torch.float64:
        raise TypeError("rt_diagnostics is fp64 only")
    out = torch.empty((NDIAG, n), dtype=torch.float64, device=x.device)
    w = _omega_rays(omega, n)
    _check(lib.rt_diagnostics(eq.handle, _ptr(x), _ptr(k), 0.0 if w is not None else float(omega), _ptr(w), n, _ptr(out),
                              _stream()))
    return out


def orbit(eq: Equilibrium, x0, v0, charge_over_mass: float, n_steps: int, dt: float, save_stride: int = 1, *, traj=False,
          final=True, drift=True, status=True, out: dict | None = None) -> dict:
    """``rt_orbit`` on the current CUDA stream: full-orbit particles, x0, v0 CUDA tensors [3, n] (float64 or float32).
    Returns device tensors 'traj' [n_saved, 6, n], 'final' [6, n], 'drift' ([n_saved, n] with traj else [n]) and
    'status' [n] int32 for the outputs requested.  Does not synchronise."""
    import torch
    lib = load()
    x0 = _dev_soa(x0, 3)
    n = x0.shape[1]
    v0 = _dev_soa(v0, 3, n)
    if v0.dtype != x0.dtype:
        raise TypeError("x0 and v0 must have the same dtype")
    prec = _prec_of(x0)
    n_saved = n_steps // save_stride + 1 if traj else 0
    o = {} if out is None else out
    kw = dict(dtype=x0.dtype, device=x0.device)
    if traj and "traj" not in o:
        o["traj"] = torch.empty((n_saved, 6, n), **kw)
    if final and "final" not in o:
        o["final"] = torch.empty((6, n), **kw)
    if drift and "drift" not in o:
        o["drift"] = torch.empty((n_saved, n) if traj else (n,), **kw)
    if status and "status" not in o:
        o["status"] = torch.empty((n,), dtype=torch.int32, device=x0.device)
    _check(lib.rt_orbit(eq.handle, prec, _ptr(x0), _ptr(v0), float(charge_over_mass), n, int(n_steps), float(dt),
                        int(save_stride), _ptr(o.get("traj") if traj else None), _ptr(o.get("final") if final else None),
                        _ptr(o.get("drift") if drift else None), _ptr(o.get("status") if status else None), _stream()))
    return o


def rhs(eq: Equilibrium, disp, x, k, omega: float):
    """``rt_rhs``: D [n], (dx/dtau, dn/dtau) [6, n] and the inside flag [n] at points x, k [3, n] (CUDA tensors)."""
    import torch
    lib = load()
    x = _dev_soa(x, 3)
    n = x.shape[1]
    k = _dev_soa(k, 3, n)
    prec = _prec_of(x)
    D = torch.empty((n,), dtype=x.dtype, device=x.device)
    f = torch.empty((6, n), dtype=x.dtype, device=x.device)
    ins = torch.empty((n,), dtype=torch.int32, device=x.device)
    _check(lib.rt_rhs(eq.handle, _disp(disp), prec, _ptr(x), _ptr(k), float(omega), n, _ptr(D), _ptr(f), _ptr(ins), _stream()))
    return D, f, ins


def reduce(residual, status=None):
    """``rt_reduce``: device tensor [6] = (max|D|, sum|D|, #finite, #status0, #status1, #status2)."""
    import torch
    lib = load()
    ref = residual if residual is not None else status
    out = torch.empty((6,), dtype=torch.float64, device=ref.device)
    prec = _prec_of(residual) if residual is not None else 0
    n = ref.numel()
    if residual is not None and not residual.is_contiguous():
        raise ValueError("residual must be contiguous")
    if status is not None and (status.numel() != n or status.dtype != torch.int32 or not status.is_contiguous()):
        raise ValueError("status must be a contiguous int32 tensor with as many entries as residual")
    _check(lib.rt_reduce(prec, _ptr(residual), _ptr(status), n, _ptr(out), _stream()))
    return out


def fma_peak(precision="f64", min_ms: float = 100.0):
    """``rt_fma_peak``: (fused multiply-adds per second, observed SM clock in MHz)."""
    lib = load()
    rate, mhz = ctypes.c_double(), ctypes.c_double()
    p = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
    _check(lib.rt_fma_peak(p, float(min_ms), ctypes.byref(rate), ctypes.byref(mhz)))
    return rate.value, mhz.value


def fma_peak_shape(precision="f64", shape: int = 0, blocks_per_sm: int = 4, min_ms: float = 100.0):
    """``rt_fma_peak_shape``: the same microbenchmark with its instruction shape (0: acc*a+acc, 1: acc*a+b) and
    occupancy (256-thread blocks per SM) exposed (shape 2: acc_j*a_j+b_j, three register-file reads per instruction).  Returns (fused multiply-adds per second, SM clock in MHz)."""
    lib = load()
    rate, mhz = ctypes.c_double(), ctypes.c_double()
    p = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
    _check(lib.rt_fma_peak_shape(p, int(shape), int(blocks_per_sm), float(min_ms), ctypes.byref(rate), ctypes.byref(mhz)))
    return rate.value, mhz.value


MATH_FNS = {"rcp": 0, "rsqrt": 1, "sqrt": 2}


def math_probe(fn, x):
    """``rt_math_probe``: the hot loop's own 1/x, 1/sqrt(x) or sqrt(x) (``fn`` = "rcp" / "rsqrt" / "sqrt") applied to the
    CUDA tensor ``x`` (float64 or float32, 1-D contiguous); returns a tensor like ``x``.  A unit-test hook."""
    import torch
    lib = load()
    if not (x.is_cuda and x.is_contiguous() and x.dim() == 1):
        raise ValueError("math_probe wants a contiguous 1-D CUDA tensor")
    out = torch.empty_like(x)
    _check(lib.rt_math_probe(_prec_of(x), MATH_FNS[fn] if isinstance(fn, str) else int(fn), _ptr(x), x.numel(), _ptr(out),
                             _stream()))
    return out
