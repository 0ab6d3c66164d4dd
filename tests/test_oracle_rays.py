"""Pins for the oracle's ray integration (CPU only): closed-form trajectories, convergence order, invariants,
cutoff positions, factorisation of the full determinant, spline-vs-analytic equilibrium, a 50-digit mpmath
re-integration and perturbation growth.  Pin numbers (P1..P12) refer to DESIGN.md.
"""
import numpy as np
import pytest
import scipy.constants as sc
from scipy.optimize import brentq

from paper_2508_15967_b200 import inputs
from helpers import paper_facts, rel_err_xk

GHZ = 2 * np.pi * 1e9
C = inputs.C_LIGHT


def _launch_trace(oracle, w, **kw):
    eq = oracle.Equilibrium(w.eq)
    k0, D0 = oracle.launch(eq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    return eq, k0, D0, oracle.trace(eq, w.disp, w.x0, k0, w.omega, w.n_steps, w.dt, **kw)


# ---------------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("disp", ["omode", "xmode"])
def test_vacuum_rays_are_straight_lines(oracle, disp):
    """P1: n_e = 0 -> x = x0 + n0 tau, k constant (RK4 is exact for a constant right-hand side)."""
    w = inputs.config(3, n_rays=64, n_steps=400)
    eq = dict(w.eq, n_ref=0.0)
    k0, D0 = oracle.launch(eq, disp, w.x0, w.dirs, w.omega)
    np.testing.assert_allclose(np.linalg.norm(k0, axis=0) * C / w.omega, 1.0, rtol=1e-15)
    out = oracle.trace(eq, disp, w.x0, k0, w.omega, 400, 1e-3, 100, traj=True)
    for m in range(5):
        tau = m * 100 * 1e-3
        np.testing.assert_allclose(out["traj"][m, :3], w.x0 + w.dirs * tau, rtol=0, atol=2e-15 * 400)
        np.testing.assert_array_equal(out["traj"][m, 3:], k0)
    assert np.nanmax(out["residual"]) < 1e-15 and (out["status"] == 0).all()


# ---------------------------------------------------------------------------------------------- P2
def test_config1_is_a_harmonic_oscillator(oracle):
    """P2 (BASELINE.json config 1's own check): on D = 0, x'' = -x/(2 L^2), so
    x = x0 cos(W tau) + (n0/W) sin(W tau), n = n0 cos(W tau) - W x0 sin(W tau), W = 1/(sqrt(2) L)."""
    w = inputs.config(1)
    assert w.n_rays == 1024 and w.n_steps == 1000 and w.dt == 1e-3
    eq, k0, D0, out = _launch_trace(oracle, w, save_stride=1, traj=True)
    assert np.abs(D0).max() < paper_facts()["launch_tolerance"]
    n0 = k0 * C / w.omega
    # launch states: |n0|^2 = 1 - X(x0, y0), direction as drawn
    X0 = 0.5 * (1 + (w.x0[0] ** 2 + w.x0[1] ** 2))
    np.testing.assert_allclose(np.sum(n0**2, axis=0), 1 - X0, rtol=1e-14)
    W = 1 / np.sqrt(2.0)
    tau = (np.arange(1001) * w.dt)[:, None, None]
    x_exact = w.x0[None] * np.cos(W * tau) + n0[None] / W * np.sin(W * tau)
    n_exact = n0[None] * np.cos(W * tau) - W * w.x0[None] * np.sin(W * tau)
    tr = out["traj"]
    assert np.abs(tr[:, :3] - x_exact).max() < 1e-12
    assert np.abs(tr[:, 3:] * C / w.omega - n_exact).max() < 1e-12
    assert np.nanmax(out["residual"]) < 1e-13
    assert (out["status"] == 0).all()
    # z stays identically zero, k_z too (nothing depends on z)
    assert (tr[:, 2] == 0).all() and (tr[:, 5] == 0).all()
    # final == last trajectory sample
    out2 = oracle.trace(eq, w.disp, w.x0, k0, w.omega, w.n_steps, w.dt, 1)
    np.testing.assert_array_equal(out2["final"], tr[-1])
    np.testing.assert_array_equal(out2["residual"], out["residual"][-1])


def test_linear_profile_omode_is_a_parabola_and_reflects_at_the_plasma_cutoff(oracle):
    """The paper's linear test profile f(x) = 0.1 x + 1 (Eq. 4) in the density: X(x) = X0 f(x) gives a
    constant force, x(tau) = x0 + n0 tau - (X0 * 0.1 / 4) tau^2 on-shell (RK4 integrates it exactly), and the ray
    turns where X = 1, the O-mode cutoff w = wpe (L157, L191)."""
    pf = paper_facts()
    slope, icpt = pf["eq4_slope"], pf["eq4_intercept"]
    w = 60 * GHZ
    n_c = sc.epsilon_0 * sc.m_e * w * w / sc.e**2          # critical density, X = 1
    X0 = 0.9
    # n_e = n_ref (x_foot - x)/L_ramp == X0 n_c (slope x + icpt)
    eq = dict(kind="slab_linear_br", n_ref=X0 * n_c, x_foot=-icpt / slope, L_ramp=-1.0 / slope, B0=2.0, R0=1.7,
              ion_mass=0.0, ion_charge=0.0)
    x0 = np.array([[0.2], [0.0], [0.0]])
    d = np.array([[1.0], [0.0], [0.0]])
    k0, D0 = oracle.launch(eq, "omode", x0, d, w)
    n0 = k0[0, 0] * C / w
    assert n0 == pytest.approx(np.sqrt(1 - X0 * (slope * 0.2 + icpt)), rel=1e-14)
    dt, ns = 1e-2, 800
    out = oracle.trace(eq, "omode", x0, k0, w, ns, dt, 1, traj=True)
    tau = np.arange(ns + 1) * dt
    acc = -0.5 * X0 * slope
    np.testing.assert_allclose(out["traj"][:, 0, 0], 0.2 + n0 * tau + 0.5 * acc * tau**2, atol=1e-13)
    np.testing.assert_allclose(out["traj"][:, 3, 0] * C / w, n0 + acc * tau, atol=1e-13)
    x_turn = out["traj"][:, 0, 0].max()
    x_cut = (1.0 / X0 - icpt) / slope                      # X(x_cut) = 1
    assert x_turn == pytest.approx(x_cut, abs=0.5 * abs(acc) * dt**2)
    assert np.nanmax(out["residual"]) < 1e-13


# ---------------------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("cfg,total", [(3, 0.6), (4, 0.8), (5, 0.4)])
def test_fourth_order_convergence(oracle, cfg, total):
    """P3: at fixed total tau, halving dt divides both max|D| and the state error by ~16.  On the spline grid
    (config 5) the right-hand side contains second derivatives of a C^2 spline, i.e. it has kinks at cell
    boundaries, so RK4 cannot show its full order there: only a steady decrease is asserted."""
    w = inputs.config(cfg, n_rays=48)
    eq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(eq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    res, fin = [], []
    for dt in (4e-3, 2e-3, 1e-3, 5e-4):
        out = oracle.trace(eq, w.disp, w.x0, k0, w.omega, int(round(total / dt)), dt, 1)
        assert (out["status"] == 0).all()
        res.append(np.nanmax(out["residual"]))
        fin.append(out["final"])
    r1, r2 = res[0] / res[1], res[1] / res[2]
    e = [np.abs(f - fin[3])[:3].max() for f in fin[:3]]
    if cfg == 5:
        assert 3 < r1 < 22 and 3 < r2 < 22, (res, r1, r2)
        assert e[0] > 3 * e[1] > 9 * e[2], e
        return
    assert 11 < r1 < 22 and 11 < r2 < 22, (res, r1, r2)
    # error(dt) - error(dt/8.. ) ~ dt^4: e0/e1 ~ (4^4-.5^4)/(2^4-.5^4) ~ 16.06, e1/e2 ~ (16-1/16)/(1-1/16) = 17
    assert 11 < e[0] / e[1] < 22 and 11 < e[1] / e[2] < 24, e


# ---------------------------------------------------------------------------------------------- P5
def test_slab_conserves_ky_kz_bit_for_bit(oracle):
    """P5: nothing depends on y or z in the linear slab, so k_y and k_z never change, exactly."""
    w = inputs.config(3, n_rays=64, n_steps=600)
    w.dirs[2] = 0.05
    w.dirs /= np.linalg.norm(w.dirs, axis=0)
    for disp in ("omode", "xmode", "cold_full"):
        x0 = w.x0.copy()
        x0[0] = 2.28                                       # inside the ramp (full determinant needs n_e > 0)
        k0, _ = oracle.launch(w.eq, disp, x0, w.dirs, w.omega, 1)
        out = oracle.trace(w.eq, disp, x0, k0, w.omega, 600, w.dt, 1)
        np.testing.assert_array_equal(out["final"][4], k0[1])
        np.testing.assert_array_equal(out["final"][5], k0[2])
        assert not np.array_equal(out["final"][3], k0[0])


@pytest.mark.parametrize("cfg", [4, 5])
def test_axisymmetry_conserves_toroidal_angular_momentum(oracle, cfg):
    """P5: x k_y - y k_x is constant to integrator order in an axisymmetric equilibrium."""
    w = inputs.config(cfg, n_rays=64, n_steps=500)
    eq, k0, D0, out = _launch_trace(oracle, w, save_stride=1)
    Lz0 = w.x0[0] * k0[1] - w.x0[1] * k0[0]
    f = out["final"]
    Lz1 = f[0] * f[4] - f[1] * f[3]
    assert np.abs(Lz1 - Lz0).max() / np.abs(k0).max() < (2e-12 if cfg == 4 else 2e-10)
    assert np.abs(Lz0).max() / np.abs(k0).max() > 0.1      # not trivially zero


# ---------------------------------------------------------------------------------------------- P6
def test_xmode_turns_at_the_right_hand_cutoff(oracle):
    """P6: a normally incident config-3 ray reverses where R(x) = S + Dx = 0 (Fig. 3: the X-mode is cut
    off at w_r), never reaching the upper hybrid layer S = 0."""
    w = inputs.config(3, n_rays=1)
    x0 = np.array([[2.3], [0.0], [0.0]])
    d = np.array([[-1.0], [0.0], [0.0]])
    k0, D0 = oracle.launch(w.eq, "xmode", x0, d, w.omega)
    out = oracle.trace(w.eq, "xmode", x0, k0, w.omega, 3000, w.dt, 1, traj=True)
    Rfun = lambda xx: np.sum(oracle.plasma(w.eq, np.array([[xx], [0.0], [0.0]]), w.omega)[2][:2, 0])
    Sfun = lambda xx: oracle.plasma(w.eq, np.array([[xx], [0.0], [0.0]]), w.omega)[2][0, 0]
    x_cut = brentq(Rfun, 2.12, 2.3)
    x_uh = brentq(Sfun, 2.0, x_cut - 1e-3)
    x_min = out["traj"][:, 0, 0].min()
    assert x_min == pytest.approx(x_cut, abs=2e-7)
    assert x_uh < x_cut < 2.3
    assert x_cut == pytest.approx(2.178591, abs=2e-6)      # SURVEY.md 8(c) P6 scratch value
    assert out["traj"][-1, 3, 0] > 0                       # heading back out
    assert np.nanmax(out["residual"]) < 1e-11


# ---------------------------------------------------------------------------------------------- P8
@pytest.mark.parametrize("mode", ["omode", "xmode"])
def test_full_determinant_factorises_for_perpendicular_propagation(oracle, mode):
    """P8: with n_par = 0, Det = (n^2 - P)(S n^2 - RL) and the ratio in the ray equations cancels the other
    factor, so COLD_FULL reproduces the OMODE / XMODE rays (same parametrisation).  OMODE here means the
    electron-only P = 1 - X_e, so the ions are switched off for that comparison."""
    w = inputs.config(3, n_rays=32)
    eq = dict(w.eq)
    if mode == "omode":
        eq["ion_mass"] = 0.0
    x0 = w.x0.copy()
    x0[0] = 2.28
    branch = 0 if mode == "omode" else 1
    k0, D0 = oracle.launch(eq, mode, x0, w.dirs, w.omega)
    k0f, D0f = oracle.launch(eq, "cold_full", x0, w.dirs, w.omega, branch)
    np.testing.assert_allclose(k0f, k0, rtol=1e-12, atol=1e-9)
    a = oracle.trace(eq, mode, x0, k0, w.omega, 2000, 2.5e-4, 1)
    b = oracle.trace(eq, "cold_full", x0, k0, w.omega, 2000, 2.5e-4, 1)
    ex, ek = rel_err_xk(b["final"], a["final"])
    assert ex < 1e-9 and ek < 1e-9, (ex, ek)
    assert np.abs(a["final"][:3] - np.stack([x0[0], x0[1], x0[2]])).max() > 0.05


# ---------------------------------------------------------------------------------------------- P9
def test_unperturbed_grid_reproduces_the_analytic_tokamak(oracle):
    """P9: config 5 with eps = 0 follows config 4's rays up to spline error."""
    w4 = inputs.config(4, n_rays=64, n_steps=500)
    g = inputs.synth_grid(seed=1, eps=0.0)
    eq4, eq5 = oracle.Equilibrium(w4.eq), oracle.Equilibrium(g)
    k0, _ = oracle.launch(eq4, "cold_full", w4.x0, w4.dirs, w4.omega, 0)
    a = oracle.trace(eq4, "cold_full", w4.x0, k0, w4.omega, 500, 1e-3, 1)
    b = oracle.trace(eq5, "cold_full", w4.x0, k0, w4.omega, 500, 1e-3, 1)
    assert (a["status"] == 0).all() and (b["status"] == 0).all()
    ex, ek = rel_err_xk(b["final"], a["final"])
    assert ex < 2e-7 and ek < 3e-6, (ex, ek)


# --------------------------------------------------------------------------------------------- P10
def test_trajectories_in_n_do_not_depend_on_omega_when_X_is_fixed(oracle):
    """P10 / reading A13: in (x, n = ck/w, tau = ct) config 1 is w-free, so two frequencies with n_ref scaled to
    keep X fixed give the same x and n -- this exercises every place w enters the oracle."""
    a = inputs.config(1, n_rays=32)
    eqa = a.eq
    wb = 35.0 * GHZ
    eqb = dict(eqa, n_ref=eqa["n_ref"] * (wb / a.omega) ** 2)
    ka, _ = oracle.launch(eqa, "omode", a.x0, a.dirs, a.omega)
    kb, _ = oracle.launch(eqb, "omode", a.x0, a.dirs, wb)
    fa = oracle.trace(eqa, "omode", a.x0, ka, a.omega, 1000, 1e-3, 1)["final"]
    fb = oracle.trace(eqb, "omode", a.x0, kb, wb, 1000, 1e-3, 1)["final"]
    np.testing.assert_allclose(fa[:3], fb[:3], rtol=0, atol=1e-14)
    np.testing.assert_allclose(fa[3:] / a.omega, fb[3:] / wb, rtol=0, atol=1e-14 / C)


# --------------------------------------------------------------------------------------------- P11
def _mp_trace(mp, eq, disp, x0, k0, omega, n_steps, dt):
    """Independent re-integration at 40 digits: D written in CARTESIAN axes (eps = S(I-bb) + P bb + i Dx [b]x,
    numeric determinant by mpmath), gradients by mpmath's high-order numerical differentiation, classical RK4."""
    t = {k: mp.mpf(float(v)) for k, v in eq.items() if isinstance(v, (int, float))}
    c, e, me, e0 = mp.mpf(sc.c), mp.mpf(sc.e), mp.mpf(inputs.M_E), mp.mpf(inputs.EPS0)
    kind = eq["kind"]

    def plasma(x, y, z):
        if kind == "slab_linear_br":
            return t["n_ref"] * (t["x_foot"] - x) / t["L_ramp"], (mp.mpf(0), mp.mpf(0), t["B0"] * t["R0"] / x)
        R = mp.sqrt(x * x + y * y)
        rho2 = ((R - t["R0"]) ** 2 + z * z) / t["a"] ** 2
        q = t["q0"] + t["q1"] * rho2
        BR, BZ, Bp = -t["B0"] * z / (q * R), t["B0"] * (R - t["R0"]) / (q * R), t["B0"] * t["R0"] / R
        return t["n_ref"] * (1 - rho2) ** t["p_exp"], (BR * x / R - Bp * y / R, BR * y / R + Bp * x / R, BZ)

    def D(x, y, z, kx, ky, kz, w):
        ne, B = plasma(x, y, z)
        n = [c * kx / w, c * ky / w, c * kz / w]
        n2 = n[0] ** 2 + n[1] ** 2 + n[2] ** 2
        Bm = mp.sqrt(B[0] ** 2 + B[1] ** 2 + B[2] ** 2)
        S, Dx, P = mp.mpf(1), mp.mpf(0), mp.mpf(1)
        for qs, ms, ns in ((-e, me, ne), (e * t["ion_charge"], t["ion_mass"], ne / t["ion_charge"])):
            X = ns * qs * qs / (e0 * ms * w * w)
            Y = qs * Bm / (ms * w)
            S -= X / (1 - Y * Y)
            Dx += Y * X / (1 - Y * Y)
            P -= X
        if disp == "xmode":
            return S * n2 - (S + Dx) * (S - Dx)
        b = [Bi / Bm for Bi in B]
        M = mp.matrix(3, 3)
        bx = [[0, -b[2], b[1]], [b[2], 0, -b[0]], [-b[1], b[0], 0]]
        for i in range(3):
            for j in range(3):
                M[i, j] = (P - S) * b[i] * b[j] + mp.mpc(0, 1) * Dx * bx[i][j] + n[i] * n[j]
                if i == j:
                    M[i, j] += S - n2
        return mp.re(mp.det(M))

    def rhs(y):
        g = []
        for j in range(7):
            tup = tuple(1 if i == j else 0 for i in range(7))
            g.append(mp.diff(D, tuple(y) + (mp.mpf(omega),), tup, h=mp.mpf(10) ** (-12) * (abs(y[j]) if j < 6 else mp.mpf(omega))))
        return [-g[3] / g[6], -g[4] / g[6], -g[5] / g[6], g[0] / g[6], g[1] / g[6], g[2] / g[6]]

    y = [mp.mpf(float(v)) for v in list(x0) + list(k0)]
    y = [v if v != 0 else mp.mpf(0) for v in y]
    h = mp.mpf(dt) / c
    for _ in range(n_steps):
        k1 = rhs(y)
        k2 = rhs([a + h / 2 * b for a, b in zip(y, k1)])
        k3 = rhs([a + h / 2 * b for a, b in zip(y, k2)])
        k4 = rhs([a + h * b for a, b in zip(y, k3)])
        y = [a + h / 6 * (p + 2 * q + 2 * r + s) for a, p, q, r, s in zip(y, k1, k2, k3, k4)]
    return np.array([float(v) for v in y])


@pytest.mark.parametrize("cfg,disp", [(3, "xmode"), (4, "cold_full")])
def test_oracle_rounding_error_is_far_below_tolerance_vs_mpmath(oracle, cfg, disp):
    """P11: the same RK4 at 40 digits, D in a different (Cartesian) formulation and gradients by numerical
    differentiation, agrees with the fp64 oracle to ~1e-13 -- a dropped term or wrong sign anywhere in the
    oracle's D, its dual-number gradients, the ray equations or the tableau would show at O(1)."""
    import mpmath as mp
    mp.mp.dps = 40
    w = inputs.config(cfg, n_rays=2)
    x0 = w.x0.copy()
    if cfg == 3:
        x0[0] = 2.25
        x0[2] = 0.0
    eq = dict(w.eq)
    k0, _ = oracle.launch(eq, disp, x0, w.dirs, w.omega, w.branch)
    if cfg == 3:
        k0[2] = 0.0
    n_steps = 25
    dt = 8e-3 if cfg == 4 else 4e-3
    out = oracle.trace(eq, disp, x0, k0, w.omega, n_steps, dt, 1)
    for i in range(2):
        # perturb zero components slightly is not needed: h scales with |y_j|, so give zeros an absolute step
        yi = _mp_trace(mp, {k: v for k, v in eq.items()}, disp, x0[:, i] + (x0[:, i] == 0) * 1e-30,
                       k0[:, i] + (k0[:, i] == 0) * 1e-30, w.omega, n_steps, dt)
        ex, ek = rel_err_xk(out["final"][:, i:i + 1], yi[:, None])
        assert ex < 1e-13 and ek < 1e-13, (ex, ek)
        assert np.linalg.norm(yi[:3] - x0[:, i]) > 0.04


# --------------------------------------------------------------------------------------------- P12
def test_perturbation_growth_is_mild(oracle):
    """P12: a 1e-13 relative perturbation of the launch state grows to < 1e-11 over config 4, so 1e-10 parity
    between two independent fp64 implementations is attainable."""
    w = inputs.config(4, n_rays=128)
    eq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(eq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    rng = np.random.default_rng(5)
    a = oracle.trace(eq, w.disp, w.x0, k0, w.omega, 1000, 1e-3, 1)["final"]
    b = oracle.trace(eq, w.disp, w.x0 * (1 + 1e-13 * rng.normal(size=w.x0.shape)),
                     k0 * (1 + 1e-13 * rng.normal(size=k0.shape)), w.omega, 1000, 1e-3, 1)["final"]
    ex, ek = rel_err_xk(b, a)
    assert ex < 1e-11 and ek < 1e-11, (ex, ek)


# ------------------------------------------------------------------------------- status / freezing
def test_rays_leaving_the_domain_freeze_with_status_1(oracle):
    """Reading A12: a ray aimed outward from rho = 0.95 hits rho_max = 0.98, is frozen there and flagged."""
    w = inputs.config(4, n_rays=16, n_steps=200)
    k0, _ = oracle.launch(w.eq, w.disp, w.x0, -w.dirs, w.omega, w.branch)
    out = oracle.trace(w.eq, w.disp, w.x0, k0, w.omega, 200, 1e-3, 20, traj=True)
    assert (out["status"] == 1).all()
    tr = out["traj"]
    np.testing.assert_array_equal(tr[-1], tr[-2])          # frozen
    assert not np.array_equal(tr[1], tr[0])                # but it did move first
    t = inputs.TOKAMAK
    rho = np.hypot(np.hypot(tr[-1, 0], tr[-1, 1]) - t["R0"], tr[-1, 2]) / t["a"]
    assert (rho > 0.95).all() and (rho < 0.985).all()


def test_non_finite_steps_freeze_with_status_2(oracle):
    """Reading A12: a step whose new state is not finite is rejected and the ray frozen with status 2.  The parabolic
    slab's domain is all of space, so (a) a NaN launch position and (b) a step so long that the second stage point
    overflows X = 0.5 (1 + r^2/L^2) both end with status 2 and the launch state back, while (c) the rays beside them in
    the same call integrate normally.  (d) The linear slab's domain is the POSITIVE condition x > 0, so there a NaN
    position is "outside": status 1."""
    w = inputs.config(1, n_rays=4, n_steps=10)
    k0, _ = oracle.launch(w.eq, w.disp, w.x0, w.dirs, w.omega)
    x0 = w.x0.copy()
    x0[1, 2] = np.nan
    out = oracle.trace(w.eq, w.disp, x0, k0, w.omega, 10, w.dt, 5, traj=True)
    assert list(out["status"]) == [0, 0, 2, 0]
    assert np.isnan(out["final"][1, 2]) and np.array_equal(out["final"][[0, 2, 3, 4, 5], 2], np.r_[x0[[0, 2], 2], k0[:, 2]])
    assert np.isnan(out["residual"][:, 2]).all() and np.isfinite(out["residual"][:, [0, 1, 3]]).all()
    ref = oracle.trace(w.eq, w.disp, w.x0, k0, w.omega, 10, w.dt, 5, traj=True)
    np.testing.assert_array_equal(out["traj"][:, :, [0, 1, 3]], ref["traj"][:, :, [0, 1, 3]])
    big = oracle.trace(w.eq, w.disp, w.x0, k0, w.omega, 3, 1e308)
    assert (big["status"] == 2).all()
    np.testing.assert_array_equal(big["final"], np.concatenate([w.x0, k0]))
    w3 = inputs.config(3, n_rays=2, n_steps=5)
    k3, _ = oracle.launch(w3.eq, w3.disp, w3.x0, w3.dirs, w3.omega)
    x3 = w3.x0.copy()
    x3[0, 0] = np.nan
    assert list(oracle.trace(w3.eq, w3.disp, x3, k3, w3.omega, 5, w3.dt)["status"]) == [1, 0]


@pytest.mark.parametrize("where", ["slab", "tokamak", "grid"])
def test_parallel_propagation_launches_on_R_and_L_and_integrates(oracle, where):
    """P7 at theta = 0 as rays (Fig. 3's w_r, w_l are the theta = 0 cut-offs, L157): launched along +-B/|B| the two branches
    of the full determinant are n^2 = R = S + Dx and n^2 = L = S - Dx, summed here in the textbook form
    1 - sum_s wps^2 / (w (w +- Ws)) from scipy.constants; such rays integrate (status 0) with |D| at integrator order:
    it stays small and falls about 16-fold when dt is halved.  In the slab (B along z^, k along z^) k_z is an ignorable
    coordinate's momentum and stays bit-for-bit constant, and by the mirror symmetry z -> -z the +B and -B rays are
    mirror images."""
    if where == "slab":
        w = inputs.config(3, n_rays=8)
        eq = oracle.Equilibrium(w.eq)
        x0 = np.stack([np.linspace(2.2, 2.28, 8), np.linspace(-0.1, 0.1, 8), np.zeros(8)])
    elif where == "tokamak":
        w = inputs.config(4, n_rays=8)
        eq, x0 = oracle.Equilibrium(w.eq), w.x0
    else:
        w = inputs.config(4, n_rays=8)
        eq, x0 = oracle.Equilibrium(inputs.synth_grid(seed=11, eps=1e-3, nR=65, nZ=65, nPsi=65)), w.x0
    ne, B, _, ins = oracle.plasma(eq, x0, w.omega)
    assert ins.all()
    Bm = np.linalg.norm(B, axis=0)
    b = B / Bm
    Rr, Ll = np.ones(8), np.ones(8)
    for q, m in ((-sc.e, sc.m_e), (sc.e, sc.physical_constants["deuteron mass"][0])):
        wp2 = ne * q * q / (sc.epsilon_0 * m)
        Rr -= wp2 / (w.omega * (w.omega + q * Bm / m))
        Ll -= wp2 / (w.omega * (w.omega - q * Bm / m))
    finals = {}
    for branch in (0, 1):
        for sign in (+1.0, -1.0):
            k0, D0 = oracle.launch(eq, "cold_full", x0, sign * b, w.omega, branch)
            n2 = np.sum((k0 * C / w.omega) ** 2, axis=0)
            err = np.minimum(np.abs(n2 - Rr), np.abs(n2 - Ll))
            assert err.max() < 1e-12 and np.abs(D0).max() < 1e-15
            if branch == 0:
                other, _ = oracle.launch(eq, "cold_full", x0, sign * b, w.omega, 1)
                n2o = np.sum((other * C / w.omega) ** 2, axis=0)
                np.testing.assert_allclose(np.sort([n2, n2o], axis=0), np.sort([Rr, Ll], axis=0), rtol=1e-12)
            _, g, _ = oracle.dispersion(eq, "cold_full", x0, k0, w.omega)
            assert np.isfinite(g).all()
            res = {}
            for dt in (2e-3, 1e-3):
                out = oracle.trace(eq, "cold_full", x0, k0, w.omega, int(round(0.2 / dt)), dt, traj=True)
                assert (out["status"] == 0).all()
                res[dt] = np.nanmax(out["residual"][1:])
                if where == "slab":
                    assert (out["traj"][:, 5] == k0[2]).all() and (out["traj"][:, 4] == 0.0).all()
            assert res[1e-3] < 1e-8
            if res[2e-3] > 1e-11:                                   # well above the rounding floor: 4th order
                assert res[2e-3] / res[1e-3] > 10.0, (where, branch, sign, res)
            finals[(branch, sign)] = out["final"]
    if where == "slab":
        for branch in (0, 1):
            mirror = finals[(branch, +1.0)] * np.array([1, 1, -1, 1, 1, -1.0])[:, None]
            np.testing.assert_array_equal(finals[(branch, -1.0)], mirror)


def test_trajectory_sampling_and_argument_checks(oracle):
    w = inputs.config(4, n_rays=8, n_steps=100)
    eq, k0, D0, full = _launch_trace(oracle, w, save_stride=1, traj=True)
    dec = oracle.trace(eq, w.disp, w.x0, k0, w.omega, 100, w.dt, 10, traj=True)
    np.testing.assert_array_equal(dec["traj"], full["traj"][::10])
    np.testing.assert_array_equal(dec["residual"], full["residual"][::10])
    np.testing.assert_array_equal(dec["traj"][0, :3], w.x0)
    with pytest.raises(ValueError):
        oracle.trace(eq, w.disp, w.x0, k0, w.omega, 100, w.dt, 7, traj=True)
    with pytest.raises(ValueError):
        oracle.trace(inputs.config(1, n_rays=4).eq, "cold_full", w.x0, k0, w.omega, 10, w.dt, 1)
