"""Pins for the oracle's per-ray-frequency tracing and critical-surface diagnostics (CPU only).

P13  per-ray w on the parabolic slab: each ray is a harmonic oscillator with its own W_i = sqrt(X0_i)/L (closed form)
P14  a per-ray-w run is, ray by ray, bit-identical to single-frequency runs at that ray's w (indexing)
P15  diagnostics against textbook plasma formulas that are NOT the sums of PAPER.md Eq. 8-10:
     f_ce = 27.99 GHz/T, f_pe = 8.98 sqrt(n_e) Hz, Stix's R, L = 1 - sum_s wps^2/(w (w +- eps_s W_s)), the cut-off
     frequencies w_R, w_L, w_pe and the upper-hybrid resonance w_uh (Fig. 3: w_r, w_l, w_pe, w_h)
"""
import numpy as np
import scipy.constants as sc

from paper_2508_15967_b200 import inputs

C = inputs.C_LIGHT
GHZ = 2 * np.pi * 1e9


def test_p13_per_ray_frequency_harmonic_oscillators(oracle):
    """Config 1's equilibrium at frequencies w_i = w0 (1 +- 10 %): X0_i = 0.5 (w0/w_i)^2 and, on D = 0,
    x'' = -grad X / 2 = -X0_i x / L^2, so x = x0 cos(W tau) + (n0/W) sin(W tau), W_i = sqrt(X0_i)/L."""
    w = inputs.config(1, n_rays=96, n_steps=600)
    om = inputs.frequency_scan(w.n_rays, w.omega, seed=1001)
    assert om.min() < 0.95 * w.omega and om.max() > 1.05 * w.omega
    eq = oracle.Equilibrium(w.eq)
    k0, D0 = oracle.launch(eq, w.disp, w.x0, w.dirs, om)
    assert np.abs(D0).max() < 1e-15
    out = oracle.trace(eq, w.disp, w.x0, k0, om, w.n_steps, w.dt, 50, traj=True)
    X0 = w.eq["n_ref"] * sc.e**2 / (sc.epsilon_0 * sc.m_e * om**2)
    np.testing.assert_allclose(X0, 0.5 * (w.omega / om) ** 2, rtol=1e-9)      # CODATA revisions differ at 1e-10
    X0 = 0.5 * (w.omega / om) ** 2
    n0 = k0 * C / om
    np.testing.assert_allclose(np.sum(n0**2, axis=0), 1 - X0 * (1 + w.x0[0] ** 2 + w.x0[1] ** 2), rtol=1e-13)
    W = np.sqrt(X0)                                                         # L = 1 m
    for m in range(out["traj"].shape[0]):
        tau = m * 50 * w.dt
        x_exact = w.x0 * np.cos(W * tau) + n0 / W * np.sin(W * tau)
        n_exact = n0 * np.cos(W * tau) - W * w.x0 * np.sin(W * tau)
        assert np.abs(out["traj"][m, :3] - x_exact).max() < 1e-12
        assert np.abs(out["traj"][m, 3:] * C / om - n_exact).max() < 1e-12
    assert np.nanmax(out["residual"]) < 1e-13 and (out["status"] == 0).all()
    # the frequencies really differ ray to ray: the fastest and slowest oscillators end far apart
    assert np.ptp(W) > 0.1


def test_a_ray_with_a_bad_frequency_is_never_advanced(oracle):
    """Reading A20: w_i that is not positive and finite (0, negative, inf, NaN) defines no ray: status 2, every sample is
    the launch state bit for bit, |D| is NaN; the rays beside it are the same as in a call without it."""
    w = inputs.config(4, n_rays=6, n_steps=40)
    eq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(eq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    om = np.full(6, w.omega)
    om[[1, 2, 3, 4]] = [0.0, -w.omega, np.inf, np.nan]
    out = oracle.trace(eq, w.disp, w.x0, k0, om, 40, w.dt, 20, traj=True)
    assert list(out["status"]) == [0, 2, 2, 2, 2, 0]
    launch_state = np.concatenate([w.x0, k0])
    for m in range(3):
        np.testing.assert_array_equal(out["traj"][m][:, 1:5], launch_state[:, 1:5])
    np.testing.assert_array_equal(out["final"][:, 1:5], launch_state[:, 1:5])
    assert np.isnan(out["residual"][:, 1:5]).all()
    ref = oracle.trace(eq, w.disp, w.x0, k0, w.omega, 40, w.dt, 20, traj=True)
    np.testing.assert_array_equal(out["traj"][:, :, [0, 5]], ref["traj"][:, :, [0, 5]])
    assert (oracle.trace(eq, w.disp, w.x0, k0, -w.omega, 5, w.dt)["status"] == 2).all()


def test_p14_per_ray_run_equals_single_frequency_runs(oracle):
    w = inputs.config(4, n_rays=12, n_steps=150)
    om = inputs.frequency_scan(w.n_rays, w.omega, seed=1004, spread=0.05)
    eq = oracle.Equilibrium(w.eq)
    k0, D0 = oracle.launch(eq, w.disp, w.x0, w.dirs, om, w.branch)
    out = oracle.trace(eq, w.disp, w.x0, k0, om, w.n_steps, w.dt, 50, traj=True)
    for i in (0, 5, 11):
        sl = slice(i, i + 1)
        k1, D1 = oracle.launch(eq, w.disp, w.x0[:, sl], w.dirs[:, sl], float(om[i]), w.branch)
        np.testing.assert_array_equal(k1, k0[:, sl])
        one = oracle.trace(eq, w.disp, w.x0[:, sl], k1, float(om[i]), w.n_steps, w.dt, 50, traj=True)
        np.testing.assert_array_equal(one["traj"], out["traj"][:, :, sl])
        np.testing.assert_array_equal(one["residual"], out["residual"][:, sl])
    # and a different frequency gives a different ray
    other = oracle.trace(eq, w.disp, w.x0[:, :1], k0[:, :1], float(om[0]) * 1.01, w.n_steps, w.dt)
    assert np.abs(other["final"] - out["traj"][-1, :, :1]).max() > 1e-6


def _slab(n_e, ion=True):
    """Linear slab whose density at x = 1 is n_e and whose field there is 2 T."""
    return dict(kind="slab_linear_br", n_ref=n_e, x_foot=2.0, L_ramp=1.0, B0=2.0, R0=1.0,
                ion_mass=inputs.M_D if ion else 0.0, ion_charge=1.0 if ion else 0.0)


def test_p15_diagnostics_match_textbook_frequencies(oracle):
    n_e, B = 3.0e19, 2.0
    x = np.array([[1.0], [0.3], [-0.2]])
    k = np.array([[100.0], [0.0], [50.0]])
    f = 60e9
    d = oracle.diagnostics(_slab(n_e, ion=False), x, k, 2 * np.pi * f)[:, 0]
    row = dict(zip(oracle.DIAG_ROWS, d))
    assert row["n_e"] == n_e and abs(row["B"] - B) < 1e-15
    # NRL formulary: f_ce = 2.80e6 B[G] Hz = 27.99 GHz/T ; f_pe = 8.98e3 sqrt(n_e[cm^-3]) Hz = 8.98 sqrt(n_e[m^-3]) Hz
    assert abs(row["Y"] * f / B - 27.99e9) < 0.01e9
    assert abs(np.sqrt(row["X"]) * f / np.sqrt(n_e) - 8.98) < 0.005
    # n_par^2 = (n.b)^2 with b = z^: n_z = c k_z / w
    np.testing.assert_allclose(row["n_par2"], (C * 50.0 / (2 * np.pi * f)) ** 2, rtol=1e-14)
    wpe = np.sqrt(n_e * sc.e**2 / (sc.epsilon_0 * sc.m_e))
    wce = sc.e * B / sc.m_e
    # electrons only: cut-offs and the upper-hybrid resonance (Fig. 3: w_r, w_l, w_pe, w_h)
    w_R = 0.5 * (wce + np.sqrt(wce**2 + 4 * wpe**2))
    w_L = 0.5 * (-wce + np.sqrt(wce**2 + 4 * wpe**2))
    w_uh = np.sqrt(wpe**2 + wce**2)
    for w_crit, name in ((w_R, "R"), (w_L, "L"), (w_uh, "S"), (wpe, "P")):
        at = dict(zip(oracle.DIAG_ROWS, oracle.diagnostics(_slab(n_e, ion=False), x, k, w_crit)[:, 0]))
        off = dict(zip(oracle.DIAG_ROWS, oracle.diagnostics(_slab(n_e, ion=False), x, k, 1.01 * w_crit)[:, 0]))
        assert abs(at[name]) < 5e-9 and abs(off[name]) > 1e-3, (name, at[name], off[name])   # CODATA revisions: 1e-9


def test_p15_diagnostics_match_stix_R_and_L_with_ions(oracle):
    """Stix: R, L = 1 - sum_s wps^2 / (w (w +- eps_s W_s)), eps_e = -1, eps_i = +1, W_s = |q_s| B / m_s; S = (R+L)/2,
    D = (R-L)/2, P = 1 - sum_s wps^2/w^2."""
    rng = np.random.default_rng(15)
    n = 40
    xs = np.stack([rng.uniform(0.5, 1.5, n), rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)])
    k = rng.normal(size=(3, n)) * 1e3
    om = 2 * np.pi * rng.uniform(20e9, 200e9, n)
    eq = _slab(4e19)
    d = dict(zip(oracle.DIAG_ROWS, oracle.diagnostics(eq, xs, k, om)))
    n_e = 4e19 * (2.0 - xs[0])
    B = 2.0 / xs[0]
    np.testing.assert_allclose(d["n_e"], n_e, rtol=1e-15)
    np.testing.assert_allclose(d["B"], B, rtol=1e-15)
    wpe2 = n_e * sc.e**2 / (sc.epsilon_0 * sc.m_e)
    wpi2 = n_e * sc.e**2 / (sc.epsilon_0 * inputs.M_D)
    We, Wi = sc.e * B / sc.m_e, sc.e * B / inputs.M_D
    R = 1 - wpe2 / (om * (om - We)) - wpi2 / (om * (om + Wi))
    L = 1 - wpe2 / (om * (om + We)) - wpi2 / (om * (om - Wi))
    tol = dict(rtol=2e-9, atol=2e-9)                               # scipy's CODATA revision vs the oracle's numerals
    np.testing.assert_allclose(d["R"], R, **tol)
    np.testing.assert_allclose(d["L"], L, **tol)
    np.testing.assert_allclose(d["S"], 0.5 * (R + L), **tol)
    np.testing.assert_allclose(d["D"], 0.5 * (R - L), **tol)
    np.testing.assert_allclose(d["P"], 1 - (wpe2 + wpi2) / om**2, **tol)
    np.testing.assert_allclose(d["n_par2"], (C * k[2] / om) ** 2, rtol=1e-13)
    # outside the domain (x <= 0): NaN rows
    bad = oracle.diagnostics(eq, np.array([[-0.1], [0.0], [0.0]]), k[:, :1], om[:1])
    assert np.isnan(bad).all()


def test_diagnostics_unmagnetised_slab(oracle):
    """Parabolic slab: no field, so Y = D = n_par^2 = 0 and S = P = R = L = 1 - X."""
    w = inputs.config(1, n_rays=8)
    k = np.ones((3, 8))
    d = dict(zip(oracle.DIAG_ROWS, oracle.diagnostics(w.eq, w.x0, k, w.omega)))
    X = 0.5 * (1 + w.x0[0] ** 2 + w.x0[1] ** 2)
    np.testing.assert_allclose(d["X"], X, rtol=1e-14)
    for name in ("S", "P", "R", "L"):
        np.testing.assert_allclose(d[name], 1 - X, rtol=1e-14)
    for name in ("B", "Y", "D", "n_par2"):
        assert (d[name] == 0).all()
