"""GPU parity tests (-m gpu) for SURVEY 8(f)-3 and the output staging: per-ray wave frequency (rt_trace_w, rt_launch_w;
PAPER.md L147), critical-surface diagnostics (rt_diagnostics; L149, Fig. 3-4) and the 128-bit store path at ragged
sizes -- all through the C ABI, against the CPU oracle on the same seeded inputs.  Tolerances as in test_gpu_parity.py.
"""
import numpy as np
import pytest

from paper_2508_15967_b200 import inputs
from helpers import rel_err_xk
from test_gpu_parity import RES_ATOL, TOL, _dev, _host, rt  # noqa: F401  (rt is the module-scoped fixture)

pytestmark = pytest.mark.gpu
C = inputs.C_LIGHT


def _scan_workload(oracle, cfg, n_rays, n_steps, disp=None, spread=0.08):
    w = inputs.config(cfg, n_rays=n_rays, n_steps=n_steps)
    if disp is not None:
        w.disp = disp
    om = inputs.frequency_scan(n_rays, w.omega, seed=1000 + cfg, spread=spread)
    oeq = oracle.Equilibrium(w.eq)
    k0, D0 = oracle.launch(oeq, w.disp, w.x0, w.dirs, om, w.branch)
    assert np.isfinite(k0).all() and np.abs(D0).max() < 2e-15
    return w, om, oeq, k0


@pytest.mark.parametrize("cfg,n_steps,stride,precs", [(1, 600, 100, ("f64", "f32")), (3, 1200, 400, ("f64",)),
                                                      (4, 500, 50, ("f64", "f32")), (5, 300, 100, ("f64", "f32"))])
def test_per_ray_frequency_trace_parity(rt, oracle, cfg, n_steps, stride, precs):
    """rt_trace_w against the oracle's per-ray-frequency integration: trajectory samples, final state, |D|, status."""
    n_rays = 64 * 5 + 37
    w, om, oeq, k0 = _scan_workload(oracle, cfg, n_rays, n_steps)
    ref = oracle.trace(oeq, w.disp, w.x0, k0, om, n_steps, w.dt, stride, traj=True)
    assert (ref["status"] == 0).all()
    eq = rt.create_equilibrium(w.eq)
    for prec in precs:
        out = rt.trace(eq, w.disp, _dev(w.x0, prec), _dev(k0, prec), _dev(om), n_steps, w.dt, stride, traj=True)
        tr = _host(out["traj"])
        assert tr.shape == ref["traj"].shape
        for m in range(tr.shape[0]):
            ex, ek = rel_err_xk(tr[m], ref["traj"][m])
            assert ex < TOL[prec] and ek < TOL[prec], (cfg, prec, m, ex, ek)
        np.testing.assert_array_equal(_host(out["final"]), tr[-1])
        assert np.array_equal(_host(out["status"]), ref["status"])
        # |D| compared at one and the same state (reading A18): the oracle's D at the states the kernel wrote
        st = np.moveaxis(tr, -2, 0).reshape(6, -1)
        D_at = np.abs(oracle.dispersion_value(oeq, w.disp, st[:3], st[3:], np.tile(om, tr.shape[0]))).reshape(tr.shape[0], -1)
        assert np.abs(_host(out["residual"]) - D_at).max() <= RES_ATOL[prec]
    # the scan is not a no-op: tracing every ray at the central frequency gives different rays
    same = rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), w.omega, n_steps, w.dt)
    assert np.abs(_host(same["final"])[:3] - ref["final"][:3]).max() > 1e-5
    eq.close()


def test_per_ray_frequency_equals_scalar_call_at_equal_frequencies(rt, oracle):
    """With all w_i equal, rt_trace_w follows the same rays as rt_trace (the constants are folded at another reference
    frequency and rescaled per thread, so equality is to rounding, not bit for bit)."""
    w = inputs.config(4, n_rays=300, n_steps=400)
    oeq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    eq = rt.create_equilibrium(w.eq)
    a = _host(rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), w.omega, 400, w.dt)["final"])
    b = _host(rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), _dev(np.full(300, w.omega)), 400, w.dt)["final"])
    ex, ek = rel_err_xk(b, a)
    assert ex < 1e-12 and ek < 1e-12, (ex, ek)
    eq.close()


@pytest.mark.parametrize("cfg,disp,branch", [(1, "omode", 0), (3, "xmode", 0), (4, "cold_full", 0), (5, "cold_full", 1)])
def test_per_ray_frequency_launch_parity(rt, oracle, cfg, disp, branch):
    w = inputs.config(cfg, n_rays=777)
    om = inputs.frequency_scan(777, w.omega, seed=2000 + cfg)
    oeq = oracle.Equilibrium(w.eq)
    k_ref, _ = oracle.launch(oeq, disp, w.x0, w.dirs, om, branch)
    eq = rt.create_equilibrium(w.eq)
    k, D = rt.launch(eq, disp, _dev(w.x0), _dev(w.dirs), _dev(om), branch)
    k, D = _host(k), _host(D)
    assert np.array_equal(np.isnan(k), np.isnan(k_ref))
    ok = np.isfinite(k_ref).all(axis=0)
    assert ok.sum() > 700
    err = np.linalg.norm(k[:, ok] - k_ref[:, ok], axis=0) / np.linalg.norm(k_ref[:, ok], axis=0)
    assert err.max() < 1e-12 and np.abs(D[ok]).max() < 2e-15, (err.max(), np.abs(D[ok]).max())
    assert np.abs(oracle.dispersion_value(oeq, disp, w.x0[:, ok], k[:, ok], om[ok])).max() < 4e-15
    eq.close()


def test_per_ray_frequency_argument_errors(rt, oracle):
    import torch
    w = inputs.config(1, n_rays=16)
    eq = rt.create_equilibrium(w.eq)
    k0, _ = oracle.launch(w.eq, w.disp, w.x0, w.dirs, w.omega)
    with pytest.raises(ValueError):
        rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), _dev(np.full(15, w.omega)), 5, w.dt)          # wrong length
    with pytest.raises(ValueError):
        rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), torch.full((16,), w.omega), 5, w.dt)           # host tensor
    eq.close()


@pytest.mark.parametrize("cfg,prec", [(1, "f64"), (4, "f64"), (5, "f32")])
def test_a_ray_with_a_bad_frequency_is_never_advanced(rt, oracle, cfg, prec):
    """Reading A20 / include/rt.h (rt_trace_w): w_i that is not positive and finite (0, negative, inf, NaN) gives status 2,
    the launch state back bit for bit at every sample and |D| = NaN -- for that ray only; as in the oracle."""
    n = 70
    w = inputs.config(cfg, n_rays=n, n_steps=20)
    oeq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    om = np.full(n, w.omega)
    bad = [3, 31, 32, 69]
    om[bad] = [0.0, -w.omega, np.inf, np.nan]
    ref = oracle.trace(oeq, w.disp, w.x0, k0, om, 20, w.dt, 10, traj=True)
    assert (ref["status"][bad] == 2).all() and ref["status"].sum() == 8
    eq = rt.create_equilibrium(w.eq)
    x0d, k0d = _dev(w.x0, prec), _dev(k0, prec)
    out = rt.trace(eq, w.disp, x0d, k0d, _dev(om), 20, w.dt, 10, traj=True)
    assert np.array_equal(_host(out["status"]), ref["status"])
    launch_state = np.concatenate([_host(x0d), _host(k0d)])
    tr, res = _host(out["traj"]), _host(out["residual"])
    for m in range(3):
        assert np.array_equal(tr[m][:, bad], launch_state[:, bad])
    assert np.array_equal(_host(out["final"])[:, bad], launch_state[:, bad])
    assert np.isnan(res[:, bad]).all() and np.array_equal(np.isnan(res), np.isnan(ref["residual"]))
    good = np.setdiff1d(np.arange(n), bad)
    ex, ek = rel_err_xk(_host(out["final"])[:, good], ref["final"][:, good])
    tol = 1e-10 if prec == "f64" else 1e-4
    assert ex < tol and ek < tol, (ex, ek)
    eq.close()


# --------------------------------------------------------------------------------- diagnostics
@pytest.mark.parametrize("cfg", [1, 3, 4, 5])
@pytest.mark.parametrize("per_ray", [False, True])
def test_diagnostics_parity_along_trajectories(rt, oracle, cfg, per_ray):
    """rt_diagnostics at the samples of a traced trajectory against oracle.diagnostics: n_e, |B|, X, Y, S, D, P, R, L,
    n_par^2.  Relative 1e-12 on each row's scale (the kernel folds constants and, on the grid, fits its own splines)."""
    n_rays, n_steps, stride = 200, 300, 100
    w = inputs.config(cfg, n_rays=n_rays, n_steps=n_steps)
    om = inputs.frequency_scan(n_rays, w.omega, seed=3000 + cfg) if per_ray else np.full(n_rays, w.omega)
    oeq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, om, w.branch)
    eq = rt.create_equilibrium(w.eq)
    omd = _dev(om) if per_ray else w.omega
    tr = rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), omd, n_steps, w.dt, stride, traj=True)["traj"]
    for m in range(tr.shape[0]):
        got = _host(rt.diagnostics(eq, tr[m, :3].contiguous(), tr[m, 3:].contiguous(), omd))
        s = _host(tr[m])
        ref = oracle.diagnostics(oeq, s[:3], s[3:], om)
        assert got.shape == ref.shape == (10, n_rays) and np.isfinite(ref).all()
        for r, name in enumerate(oracle.DIAG_ROWS):
            scale = max(np.abs(ref[r]).max(), 1.0 if name not in ("n_e",) else 1e19)
            tol = 1e-12 if cfg != 5 else 1e-10      # grid: two independent spline fits agree to ~1e-11 in psi's derivatives
            assert np.abs(got[r] - ref[r]).max() <= tol * scale, (cfg, m, name, np.abs(got[r] - ref[r]).max())
    eq.close()


def test_diagnostics_outside_domain_and_errors(rt, oracle):
    w = inputs.config(4, n_rays=8)
    w.x0[:, 0] = [inputs.TOKAMAK["R0"] + 0.99 * inputs.TOKAMAK["a"], 0.0, 0.0]       # outside rho_max
    k = np.ones((3, 8))
    eq = rt.create_equilibrium(w.eq)
    got = _host(rt.diagnostics(eq, _dev(w.x0), _dev(k), w.omega))
    ref = oracle.diagnostics(w.eq, w.x0, k, w.omega)
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.isnan(got[:, 0]).all() and np.isfinite(got[:, 1:]).all()
    with pytest.raises(rt.RtError):
        rt.diagnostics(eq, _dev(w.x0), _dev(k), -1.0)
    eq.close()


def test_cutoff_layer_is_where_the_xmode_ray_turns(rt, oracle):
    """"the wave is reflected at a cut-off".  Config 3's normal-incidence X-mode ray turns where R = 0
    (pin P6): along the kernel's trajectory min R is reached at the turning point and is ~0, S stays > 0 (the upper-hybrid
    layer is never reached)."""
    w = inputs.config(3, n_rays=1, n_steps=3000)
    w.x0[1] = 0.0
    w.dirs[:] = np.array([[-1.0], [0.0], [0.0]])
    k0, _ = oracle.launch(w.eq, w.disp, w.x0, w.dirs, w.omega)
    eq = rt.create_equilibrium(w.eq)
    tr = rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), w.omega, 3000, w.dt, 10, traj=True)["traj"]
    xs, ks = tr[:, :3, 0].T.contiguous(), tr[:, 3:, 0].T.contiguous()
    d = dict(zip(rt.DIAG_ROWS, _host(rt.diagnostics(eq, xs, ks, w.omega))))
    x = _host(xs)[0]
    i_turn = int(np.argmin(x))
    assert 0 < i_turn < len(x) - 1 and abs(int(np.argmin(d["R"])) - i_turn) <= 1
    assert 0 <= d["R"][i_turn] < 2e-3 and d["S"].min() > 0.05 and (d["L"] >= d["R"]).all()
    eq.close()


# --------------------------------------------------------------------------------- 128-bit store path at ragged sizes
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n_rays", [1, 2, 3, 4, 31, 32, 33, 62, 63, 64, 65, 66, 68, 127, 130, 1001, 1002, 1004])
def test_store_paths_at_ragged_sizes(rt, oracle, n_rays, prec):
    """The vectorised store path needs the row pitch to be a multiple of 2 (fp64) / 4 (fp32) elements and falls back to
    scalar stores otherwise; the last warp / block is partial.  Every output array must be written exactly: compare all
    of traj / final / residual / status with the oracle and check that nothing outside them is touched."""
    import torch
    w = inputs.config(4, n_rays=n_rays, n_steps=40)
    oeq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    ref = oracle.trace(oeq, w.disp, w.x0, k0, w.omega, 40, w.dt, 20, traj=True)
    eq = rt.create_equilibrium(w.eq)
    dt = torch.float64 if prec == "f64" else torch.float32
    # outputs carved out of one guarded allocation: [guard | traj | guard | final | guard | residual | guard]
    G = 64
    sizes = [3 * 6 * n_rays, 6 * n_rays, 3 * n_rays]
    sizes = [(s + 3) // 4 * 4 for s in sizes]                       # keep every sub-buffer 16-byte aligned
    buf = torch.full((G * 4 + sum(sizes),), -777.0, dtype=dt, device="cuda")
    o0 = G
    o1 = o0 + sizes[0] + G
    o2 = o1 + sizes[1] + G
    out = {"traj": buf[o0:o0 + 18 * n_rays].view(3, 6, n_rays), "final": buf[o1:o1 + 6 * n_rays].view(6, n_rays),
           "residual": buf[o2:o2 + 3 * n_rays].view(3, n_rays)}
    rt.trace(eq, w.disp, _dev(w.x0, prec), _dev(k0, prec), w.omega, 40, w.dt, 20, traj=True, out=out)
    torch.cuda.synchronize()
    tr = _host(out["traj"])
    for m in range(3):
        ex, ek = rel_err_xk(tr[m], ref["traj"][m])
        assert ex < TOL[prec] and ek < TOL[prec], (m, ex, ek)
    np.testing.assert_array_equal(_host(out["final"]), tr[-1])
    assert np.abs(_host(out["residual"]) - ref["residual"]).max() < (1e-11 if prec == "f64" else 1e-3)
    assert np.array_equal(_host(out["status"]), ref["status"])
    mask = torch.ones_like(buf, dtype=torch.bool)
    mask[o0:o0 + 18 * n_rays] = False
    mask[o1:o1 + 6 * n_rays] = False
    mask[o2:o2 + 3 * n_rays] = False
    assert bool((buf[mask] == -777.0).all()), "a store went outside its output array"
    # final-only mode (no trajectory): residual is [n_rays]
    out2 = rt.trace(eq, w.disp, _dev(w.x0, prec), _dev(k0, prec), w.omega, 40, w.dt)
    np.testing.assert_array_equal(_host(out2["final"]), tr[-1])
    np.testing.assert_array_equal(_host(out2["residual"]), _host(out["residual"])[-1])
    eq.close()


@pytest.mark.parametrize("cfg", [4, 5])
def test_low_frequency_scan_straddles_the_ion_series_range(rt, oracle, cfg):
    """Deuterium plasma of configs 4 / 5 at 20-28 GHz, one frequency per ray, second root of the biquadratic: Y2 = (W_ce / w)^2
    at launch runs from 2.3 to 4.7, on both sides of the 3.35 below which the fp64 kernels take the ion terms of the Stix elements
    from their series (rt_params.h: series_cap).  Inside one warp some rays stay in the fast step loop, some
    are in the exact one from the first step and some change over on the way in -- all must follow the oracle."""
    n_rays, n_steps, stride = 64 * 5 + 37, 400, 100
    w = inputs.config(cfg, n_rays=n_rays, n_steps=n_steps)
    om = 2 * np.pi * np.random.default_rng(4242).uniform(20e9, 28e9, n_rays)
    oeq = oracle.Equilibrium(w.eq)
    k0, D0 = oracle.launch(oeq, w.disp, w.x0, w.dirs, om, 1)
    assert np.isfinite(k0).all() and np.abs(D0).max() < 2e-15
    ref = oracle.trace(oeq, w.disp, w.x0, k0, om, n_steps, w.dt, stride, traj=True)
    assert (ref["status"] == 0).all()
    Y2 = np.stack([oracle.diagnostics(oeq, ref["traj"][m, :3], ref["traj"][m, 3:], om)[3] ** 2 for m in range(ref["traj"].shape[0])])
    assert (Y2.max(axis=0) < 3.3).mean() > 0.2 and (Y2[0] > 3.4).mean() > 0.2 and ((Y2[0] < 3.3) & (Y2.max(axis=0) > 3.4)).mean() > 0.1
    eq = rt.create_equilibrium(w.eq)
    out = rt.trace(eq, w.disp, _dev(w.x0), _dev(k0), _dev(om), n_steps, w.dt, stride, traj=True)
    tr = _host(out["traj"])
    for m in range(tr.shape[0]):
        ex, ek = rel_err_xk(tr[m], ref["traj"][m])
        assert ex < 1e-10 and ek < 1e-10, (cfg, m, ex, ek)
    assert np.array_equal(_host(out["status"]), ref["status"])
    # the scalar-frequency kernel on the rays of one frequency bin, wholly beyond the range (every step in the exact loop)
    sel = np.argsort(om)[:64]
    k0s, _ = oracle.launch(oeq, w.disp, w.x0[:, sel], w.dirs[:, sel], om[sel[0]], 1)
    refs = oracle.trace(oeq, w.disp, w.x0[:, sel], k0s, om[sel[0]], n_steps, w.dt)
    outs = rt.trace(eq, w.disp, _dev(w.x0[:, sel]), _dev(k0s), float(om[sel[0]]), n_steps, w.dt)
    ex, ek = rel_err_xk(_host(outs["final"]), refs["final"])
    assert ex < 1e-10 and ek < 1e-10 and np.array_equal(_host(outs["status"]), refs["status"]), (ex, ek)
    eq.close()
