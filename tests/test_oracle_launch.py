"""Pins for the oracle's literal launch iteration (CPU only; w, x, k_y, k_z fixed, Newton on k_x, the initial
guess selects the root).

P20a  perpendicular propagation in the slab: the roots are n_x^2 = P (O) and n_x^2 = R L / S (X) with R, L, P summed here from
      scipy.constants in the textbook form 1 - sum wps^2 / (w (w +- Ws)); the guess selects root and sign; O-mode with
      k_y, k_z != 0: n_x^2 = 1 - X - n_y^2 - n_z^2
P20b  oblique propagation in the tokamak: the converged k_x is a root of the quartic det(eps + n n - n^2 I)(n_x) built with
      numpy from the independently summed S, D, P, and it is the root next to the guess
P20c  the iteration itself: max_iter = 0 returns the guess; |D| falls quadratically; points outside the domain and
      evanescent starts are flagged; a per-ray-w call equals scalar calls
"""
import numpy as np
import scipy.constants as sc

from paper_2508_15967_b200 import inputs

GHZ = 2 * np.pi * 1e9
C = inputs.C_LIGHT
M_D = sc.physical_constants["deuteron mass"][0]


def _stix_textbook(ne, Bm, w):
    Rr, Ll, P = np.ones_like(ne), np.ones_like(ne), np.ones_like(ne)
    for q, m in ((-sc.e, sc.m_e), (sc.e, M_D)):
        wp2 = ne * q * q / (sc.epsilon_0 * m)
        Om = q * Bm / m
        Rr -= wp2 / (w * (w + Om))
        Ll -= wp2 / (w * (w - Om))
        P -= wp2 / w**2
    return 0.5 * (Rr + Ll), 0.5 * (Rr - Ll), P, Rr, Ll


def _slab_points(n=24, lo=1.85):
    w = inputs.config(3, n_rays=1)
    x = np.stack([np.linspace(lo, 2.25, n), np.linspace(-0.1, 0.1, n), np.zeros(n)])
    ne = 5e19 * (2.3 - x[0]) / 0.5                       # BASELINE.json config 3, typed here
    Bm = 2.0 * 1.7 / x[0]
    return w, x, ne, Bm


def test_perpendicular_roots_are_P_and_RL_over_S(oracle):
    """P20a"""
    w, x, ne, Bm = _slab_points()
    S, Dx, P, Rr, Ll = _stix_textbook(ne, Bm, w.omega)
    eq = oracle.Equilibrium(w.eq)
    for target, disp in ((P, "cold_full"), (Rr * Ll / S, "cold_full"), (Rr * Ll / S, "xmode")):
        ok = target > 0.01
        assert ok.sum() >= 10
        for sign in (+1.0, -1.0):
            kg = np.zeros((3, x.shape[1]))
            kg[0] = sign * np.sqrt(np.where(ok, target, 1.0)) * 1.04 * w.omega / C
            k0, D, it = oracle.launch_kx(eq, disp, x, kg, w.omega)
            nx = k0[0] * C / w.omega
            np.testing.assert_allclose(nx[ok] ** 2, target[ok], rtol=2e-12)
            assert (np.sign(nx[ok]) == sign).all()
            assert (it[ok] >= 1).all() and (it[ok] <= 8).all() and (np.abs(D[ok]) < 1e-15).all()
            assert (k0[1:] == 0).all()                    # k_y, k_z are never touched


def test_omode_root_with_fixed_ky_kz(oracle):
    """P20a: D = n^2 - 1 + X  =>  n_x^2 = 1 - X - n_y^2 - n_z^2 (config 1's equilibrium)."""
    w = inputs.config(1, n_rays=64)
    rng = np.random.default_rng(7)
    x = np.stack([rng.uniform(-0.3, 0.3, 64), rng.uniform(-0.3, 0.3, 64), rng.uniform(-1, 1, 64)])
    X = 0.5 * (1 + (x[0] ** 2 + x[1] ** 2) / 1.0**2)
    ny, nz = rng.uniform(-0.3, 0.3, 64), rng.uniform(-0.3, 0.3, 64)
    nx2 = 1 - X - ny**2 - nz**2
    assert (nx2 > 0.05).all()
    kg = np.stack([0.9 * np.sqrt(nx2), ny, nz]) * w.omega / C
    k0, D, it = oracle.launch_kx(w.eq, "omode", x, kg, w.omega)
    np.testing.assert_allclose((k0[0] * C / w.omega) ** 2, nx2, rtol=1e-13)
    np.testing.assert_array_equal(k0[1:], kg[1:])
    assert (it >= 1).all() and (np.abs(D) < 1e-15).all()


def _cart_det(S, Dx, P, b, n):
    bx = np.array([[0, -b[2], b[1]], [b[2], 0, -b[0]], [-b[1], b[0], 0]])
    eps = S * (np.eye(3) - np.outer(b, b)) + P * np.outer(b, b) + 1j * Dx * bx
    return np.linalg.det(eps + np.outer(n, n) - (n @ n) * np.eye(3)).real


def test_oblique_root_is_a_root_of_the_numpy_quartic(oracle):
    """P20b"""
    t = inputs.TOKAMAK
    eq = dict(kind="tokamak_circular", **t)
    w = 110 * GHZ
    rng = np.random.default_rng(11)
    n = 40
    rho, th, ph = rng.uniform(0.2, 0.85, n), rng.uniform(0, 2 * np.pi, n), rng.uniform(0, 2 * np.pi, n)
    R, Z = t["R0"] + rho * t["a"] * np.cos(th), rho * t["a"] * np.sin(th)
    x = np.stack([R * np.cos(ph), R * np.sin(ph), Z])
    # field and density of BASELINE.json config 4 / reading A9, typed here
    q = t["q0"] + t["q1"] * rho**2
    BR, BZ, Bp = -(t["B0"] * Z / q) / R, (t["B0"] * (R - t["R0"]) / q) / R, t["B0"] * t["R0"] / R
    B = np.stack([BR * np.cos(ph) - Bp * np.sin(ph), BR * np.sin(ph) + Bp * np.cos(ph), BZ])
    Bm = np.linalg.norm(B, axis=0)
    ne = t["n_ref"] * (1 - rho**2) ** t["p_exp"]
    S, Dx, P, _, _ = _stix_textbook(ne, Bm, w)
    ny, nz = rng.uniform(-0.3, 0.3, n), rng.uniform(-0.3, 0.3, n)
    checked = 0
    for i in range(n):
        b = B[:, i] / Bm[i]
        s = np.linspace(-1.5, 1.5, 9)
        dets = [_cart_det(S[i], Dx[i], P[i], b, np.array([v, ny[i], nz[i]])) for v in s]
        coef = np.polyfit(s, dets, 4)                                     # the determinant is a quartic in n_x
        assert np.abs(np.polyval(coef, s) - dets).max() < 1e-11
        roots = np.roots(coef)
        real = np.sort(roots[np.abs(roots.imag) < 1e-9].real)
        for r in real:
            if np.abs(real - r).min(initial=9.0, where=real != r) < 0.1 or abs(r) < 0.05:
                continue                                                  # keep well separated roots only
            kg = np.array([[r * 1.02], [ny[i]], [nz[i]]]) * w / C
            k0, D, it = oracle.launch_kx(eq, "cold_full", x[:, i:i + 1], kg, w)
            assert it[0] >= 0 and abs(D[0]) < 1e-15
            assert k0[0, 0] * C / w == np.float64(r).item() or abs(k0[0, 0] * C / w - r) < 1e-9 * max(1.0, abs(r))
            checked += 1
    assert checked >= 40


def test_iteration_semantics(oracle):
    """P20c"""
    w, x, ne, Bm = _slab_points(8, lo=1.95)
    S, Dx, P, Rr, Ll = _stix_textbook(ne, Bm, w.omega)
    eq = oracle.Equilibrium(w.eq)
    kg = np.zeros((3, 8))
    kg[0] = np.sqrt(P) * 1.2 * w.omega / C
    k0, D0, it = oracle.launch_kx(eq, "cold_full", x, kg, w.omega, max_iter=0)
    np.testing.assert_array_equal(k0, kg)
    assert (it == -1).all() and (np.abs(D0) > 1e-3).all()
    # quadratic convergence: the error in n_x is squared (times a constant) by every update
    err = []
    for m in (1, 2, 3):
        k0, D, it = oracle.launch_kx(eq, "cold_full", x, kg, w.omega, max_iter=m)
        err.append(np.abs(k0[0] * C / w.omega - np.sqrt(P)))
    assert (err[0] < 0.1).all()
    assert (err[1] < 10.0 * err[0] ** 2).all() and (err[2] < 10.0 * err[1] ** 2 + 1e-15).all()
    # started on the root: no update
    kg[0] = oracle.launch_kx(eq, "cold_full", x, kg, w.omega)[0][0]
    k0, D, it = oracle.launch_kx(eq, "cold_full", x, kg, w.omega)
    assert (it == 0).all()
    np.testing.assert_array_equal(k0, kg)
    # outside the domain (x <= 0): NaN and -1
    xo = x.copy()
    xo[0, :3] = -1.0
    k0, D, it = oracle.launch_kx(eq, "cold_full", xo, kg, w.omega)
    assert np.isnan(k0[0, :3]).all() and np.isnan(D[:3]).all() and (it[:3] == -1).all() and (it[3:] == 0).all()
    # one frequency per ray == scalar calls
    ws = w.omega * np.linspace(0.9, 1.1, 8)
    kg[0] = np.sqrt(P) * 1.1 * ws / C
    kA, DA, itA = oracle.launch_kx(eq, "cold_full", x, kg, ws)
    for i in range(8):
        kB, DB, itB = oracle.launch_kx(eq, "cold_full", x[:, i:i + 1], kg[:, i:i + 1], ws[i])
        assert kA[0, i] == kB[0, 0] and DA[i] == DB[0] and itA[i] == itB[0]
