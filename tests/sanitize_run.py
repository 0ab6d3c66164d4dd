"""Workload of tests/test_sanitizers.py, run in a subprocess with the ASan / UBSan builds preloaded (not a test itself).

    RT_ORACLE_LIB=<sanitized librt_oracle.so> python tests/sanitize_run.py <sanitized libspline_shim.so>

Drives every entry point of the oracle (each equilibrium: 64 rays x 50 steps, launch, dispersion, diagnostics, the
convergence workflow, orbits) and the library's host-side spline fit (33 x 29 nodes) + constant folding through the shim."""
import ctypes
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

import oracle  # noqa: E402
from paper_2508_15967_b200 import binding, inputs  # noqa: E402  (binding: the descriptor struct only, no library load)


def main(shim_path: str) -> int:
    small_grid = inputs.synth_grid(seed=5, eps=1e-3, nR=33, nZ=29, nPsi=31)
    for cfg in (1, 3, 4, 5):
        w = inputs.config(cfg if cfg != 5 else 4, n_rays=64, n_steps=50)
        eq = oracle.Equilibrium(small_grid if cfg == 5 else w.eq)
        k0, D0 = oracle.launch(eq, w.disp, w.x0, w.dirs, w.omega, w.branch)
        out = oracle.trace(eq, w.disp, w.x0, k0, w.omega, 50, w.dt, 10, traj=True, n_threads=2)
        assert np.isfinite(out["final"]).all() and (out["status"] == 0).all()
        oracle.trace(eq, w.disp, w.x0, k0, np.full(64, w.omega), 20, w.dt)
        oracle.dispersion(eq, w.disp, w.x0, k0, w.omega)
        oracle.diagnostics(eq, w.x0, k0, w.omega)
        oracle.launch_kx(eq, w.disp, w.x0, k0, w.omega, max_iter=5)
        u = oracle.trace_until(eq, w.disp, w.x0, k0, w.omega, 10, 3, w.dt, n_threads=2)
        assert u["chunks"] == 3
        if cfg != 1:
            ow = inputs.orbit_config(4 if cfg == 5 else cfg, n=64, n_steps=50)
            oracle.orbit(small_grid if cfg == 5 else ow.eq, ow.x0, ow.v0, ow.charge_over_mass, 50, ow.dt, 10, traj=True)
        # rays that leave the domain and a NaN ray: the freeze paths
        x_bad = w.x0.copy()
        x_bad[0, 0] = np.nan
        oracle.trace(eq, w.disp, x_bad, k0, w.omega, 5, w.dt)
    shim = ctypes.CDLL(shim_path)
    P = ctypes.c_void_p
    shim.shim_fit_cubic.argtypes = [P, P, ctypes.c_long, ctypes.c_int, P]
    shim.shim_fit_bicubic.argtypes = [P, P, P, ctypes.c_int, ctypes.c_int, P]
    shim.shim_fold_params.argtypes = [P, ctypes.c_double, ctypes.c_double, ctypes.c_int, P]
    R, Z = np.linspace(0.95, 2.45, 33), np.linspace(-0.75, 0.75, 29)
    f = np.ascontiguousarray(np.cos(R)[:, None] * np.sin(2 * Z)[None, :])
    pp = np.empty((32, 28, 4, 4))
    assert shim.shim_fit_bicubic(R.ctypes.data, Z.ctypes.data, f.ctypes.data, 33, 29, pp.ctypes.data) == pp.size
    for n in (4, 5, 33):
        x = np.linspace(0.0, 1.0, n)
        y = np.ascontiguousarray(np.exp(x))
        p1 = np.empty((n - 1, 4))
        assert shim.shim_fit_cubic(x.ctypes.data, y.ctypes.data, 1, n, p1.ctypes.data) == 0
    out16 = np.empty(16)
    for cfg in (1, 3, 4):
        desc, keep = binding.make_desc(inputs.config(cfg, n_rays=1).eq)
        for fp32 in (0, 1):
            shim.shim_fold_params(ctypes.byref(desc), 0.98, 6.9e11, fp32, out16.ctypes.data)
    print("sanitize_run ok")
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1]))
