"""Pins for the oracle's full-orbit particle integrator (CPU only, PAPER.md L121 / L213).

P16  gyration in a (nearly) uniform field: Larmor radius m v_perp/(|q| B), gyro-frequency |q| B/m, sense of rotation
P17  slab B = (B0 R0/x) z^: v_z bit-for-bit constant, canonical momentum v_y + (q/m) B0 R0 ln x and kinetic energy
     conserved to integrator order (halving dt divides the drifts by ~2^4 .. 2^5)
P18  axisymmetric field: toroidal canonical momentum R v_phi + (q/m) psi(R, Z) conserved, psi = (B0 a^2/4) ln(1 + 2 rho^2)
     in closed form (reading A9); the spline grid with eps = 0 reproduces the analytic orbit
P19  grad-B drift of the guiding centre: v_d = v_perp^2/(2 W) (B x grad B)/B^2 to first order in rho_L/L
"""
import numpy as np
import scipy.constants as sc

from paper_2508_15967_b200 import inputs

QM_D = sc.e / inputs.M_D


def _slab(B0R0, ion=True):
    return dict(kind="slab_linear_br", n_ref=0.0, x_foot=2.0, L_ramp=1.0, B0=B0R0, R0=1.0, ion_mass=inputs.M_D, ion_charge=1.0)


def test_p16_larmor_gyration_in_a_nearly_uniform_field(oracle):
    """x0 = 1e6 m in B = B0 R0/x with B0 R0 = 2e6 T m: B = 2 T with a gradient length of 1e6 m (non-uniformity 1e-8 over
    a Larmor radius).  A deuteron with v_perp = 1e6 m/s, v_par = 3e5 m/s gyrates on a circle of radius v_perp/W at
    W = q B/m, clockwise seen along +B for q > 0: v_x + i v_y = v_perp exp(-i W t)."""
    eq = _slab(2e6)
    B = 2.0
    W = QM_D * B
    vp, vz = 1.0e6, 3.0e5
    x0 = np.array([[1e6], [0.0], [0.0]])
    v0 = np.array([[vp], [0.0], [vz]])
    T = 2 * np.pi / W
    n_steps, stride = 4000, 50
    dt = 2 * T / n_steps                                      # two gyrations, 2000 steps each
    out = oracle.orbit(eq, x0, v0, QM_D, n_steps, dt, stride, traj=True)
    t = np.arange(n_steps // stride + 1) * stride * dt
    rho = vp / W
    # NRL formulary: ion gyro-frequency f_ci = 1.52e3 Z B[G] / mu Hz, mu = m_i / m_p
    assert abs(W / (2 * np.pi) / (1.52e3 * 2e4 / (inputs.M_D / sc.m_p)) - 1.0) < 5e-3 and 0.0104 < rho < 0.0105
    tr = out["traj"][:, :, 0]
    np.testing.assert_allclose(tr[:, 3], vp * np.cos(W * t), atol=vp * 1e-7)
    np.testing.assert_allclose(tr[:, 4], -vp * np.sin(W * t), atol=vp * 1e-7)
    np.testing.assert_array_equal(tr[:, 5], vz)
    np.testing.assert_allclose(tr[:, 0] - 1e6, rho * np.sin(W * t), atol=rho * 1e-6)
    np.testing.assert_allclose(tr[:, 1], rho * (np.cos(W * t) - 1.0), atol=rho * 1e-6)
    np.testing.assert_allclose(tr[:, 2], vz * t, rtol=1e-12)
    assert (out["status"] == 0).all() and np.abs(out["drift"]).max() < 1e-12
    # an electron (q/m < 0) turns the other way, 3670 times faster
    qm_e = -sc.e / sc.m_e
    We = abs(qm_e) * B
    oe = oracle.orbit(eq, x0, v0, qm_e, 400, 0.25 * 2 * np.pi / We / 400, 400, traj=True)     # a quarter turn
    np.testing.assert_allclose(oe["traj"][1, 3:5, 0], [0.0, vp], atol=vp * 1e-6)


def test_p17_slab_invariants_and_order(oracle):
    w = inputs.orbit_config(3, n=64, n_steps=800)
    B0R0 = w.eq["B0"] * w.eq["R0"]
    py0 = w.v0[1] + w.charge_over_mass * B0R0 * np.log(w.x0[0])
    errs = []
    for refine in (1, 2):
        out = oracle.orbit(w.eq, w.x0, w.v0, w.charge_over_mass, 800 * refine, 2e-9 / refine, 200 * refine, traj=True)
        tr = out["traj"]
        np.testing.assert_array_equal(tr[:, 5], np.broadcast_to(w.v0[2], tr[:, 5].shape))     # dv_z/dt == 0 exactly
        py = tr[:, 4] + w.charge_over_mass * B0R0 * np.log(tr[:, 0])
        e_py = np.abs(py - py0).max() / np.abs(w.v0).max()
        e_en = np.abs(out["drift"]).max()
        errs.append((e_py, e_en))
        assert (out["status"] == 0).all()
        # drift output is what it says
        np.testing.assert_allclose(out["drift"], (tr[:, 3:] ** 2).sum(1) / (w.v0**2).sum(0) - 1.0, atol=1e-15)
    (p1, e1), (p2, e2) = errs
    assert p1 < 1e-5 and e1 < 1e-3, (p1, e1)                  # W dt = 0.16 at 2 ns: energy drift ~ steps (W dt)^6/72
    assert 12 < p1 / p2 < 40 and 24 < e1 / e2 < 40, (p1 / p2, e1 / e2)
    # flipping the sign of the force would conserve v_y - (q/m) B0R0 ln x instead: make sure that one is NOT conserved
    wrong = tr[:, 4] - w.charge_over_mass * B0R0 * np.log(tr[:, 0])
    assert np.abs(wrong - wrong[0]).max() / np.abs(w.v0).max() > 1e-2


def _psi_analytic(x):
    t = inputs.TOKAMAK
    R = np.hypot(x[0], x[1])
    rho2 = ((R - t["R0"]) ** 2 + x[2] ** 2) / t["a"] ** 2
    return 0.25 * t["B0"] * t["a"] ** 2 * np.log1p(t["q1"] / t["q0"] * rho2) * (2.0 / t["q1"]) / t["q0"] * t["q0"]


def _p_phi(state, qm):
    x, v = state[:3], state[3:]
    R = np.hypot(x[0], x[1])
    v_phi = (-x[1] * v[0] + x[0] * v[1]) / R
    return R * v_phi + qm * _psi_analytic(x)


def test_p18_toroidal_canonical_momentum(oracle):
    w = inputs.orbit_config(4, n=48, n_steps=1000)
    assert inputs.TOKAMAK["q0"] == 1.0 and inputs.TOKAMAK["q1"] == 2.0       # psi's closed form above assumes q = 1 + 2 rho^2
    scale = np.abs(w.v0).max() * inputs.TOKAMAK["R0"]
    errs = []
    for refine in (1, 2):
        out = oracle.orbit(w.eq, w.x0, w.v0, w.charge_over_mass, 1000 * refine, w.dt / refine, 100 * refine, traj=True)
        P = np.stack([_p_phi(s, w.charge_over_mass) for s in out["traj"]])
        errs.append((np.abs(P - P[0]).max() / scale, np.abs(out["drift"]).max()))
        assert (out["status"] == 0).all()
    (p1, e1), (p2, e2) = errs
    # the two terms of P_phi are each ~ q/m psi ~ 1e7 m^2/s >> R v_phi: their sum must stay put to integrator order
    assert p1 < 1e-7 and e1 < 1e-4, (p1, e1)                  # energy: steps (W dt)^6/72 with W dt ~ 0.1
    assert 10 < p1 / p2 < 40 and 24 < e1 / e2 < 40, (p1 / p2, e1 / e2)
    # the orbit really moves in psi: R v_phi alone is not conserved
    Rv = np.stack([_p_phi(s, 0.0) for s in out["traj"]])
    assert np.abs(Rv - Rv[0]).max() / scale > 1e-3


def test_p18_grid_without_perturbation_reproduces_the_analytic_orbit(oracle):
    w = inputs.orbit_config(4, n=32, n_steps=500)
    grid = inputs.synth_grid(1005, eps=0.0)
    a = oracle.orbit(w.eq, w.x0, w.v0, w.charge_over_mass, 500, w.dt)["final"]
    b = oracle.orbit(grid, w.x0, w.v0, w.charge_over_mass, 500, w.dt)["final"]
    assert np.abs(a[:3] - b[:3]).max() < 2e-6 and np.abs(a[3:] - b[3:]).max() / np.abs(w.v0).max() < 2e-5


def test_p19_grad_B_drift(oracle):
    """Slab B = (B0 R0/x) z^ at x = 2 m, B0 R0 = 4: B = 2 T, grad B = -(B/x) x^, so B x grad B = -(B^2/x) y^ and the
    guiding centre of a q > 0 particle drifts at v_d = -v_perp^2/(2 W x) y^.  rho_L/x = 5e-3."""
    eq = _slab(4.0)
    W = QM_D * 2.0
    vp = 1.0e6
    x0 = np.array([[2.0], [0.0], [0.0]])
    v0 = np.array([[0.0], [vp], [0.0]])
    T = 2 * np.pi / W
    n_gyr, per = 40, 400
    out = oracle.orbit(eq, x0, v0, QM_D, n_gyr * per, T / per, 10, traj=True)
    tr = out["traj"][:, :, 0]
    # guiding centre: X = x - (v x b^)/W(x) with the LOCAL gyro-frequency W(x) = (q/m) B0R0/x: y_gc = y - v_x/W(x).
    # (Sampling y once per nominal period instead would alias the 0.5 % period change between x and x + rho_L.)
    y_gc = tr[:, 1] - tr[:, 3] / (QM_D * 4.0 / tr[:, 0])
    t = np.arange(tr.shape[0]) * 10 * (T / per)
    drift = np.polyfit(t, y_gc, 1)[0]
    v_d = -vp**2 / (2 * W * 2.0)
    assert v_d < 0 and abs(drift / v_d - 1.0) < 0.02, (drift, v_d)
    assert np.abs(tr[:, 0] - 2.0).max() < 2.5 * vp / W                     # x stays within a Larmor diameter
