"""Host logic of the product on CPU, compiled with g++ through a small shim (tests/host_shim.cpp); no GPU, no oracle:

* the library's not-a-knot spline fit (csrc/spline_fit.cpp, run once per rt_create_equilibrium; reading A10)
  against scipy's CubicSpline / RectBivariateSpline and against the exactness properties of not-a-knot splines;
* the per-call constant folding (csrc/rt_params.h, step a0 of the hot path) against the definitions of X, Y and n
  (Eq. 6; L189) written out with scipy.constants."""
import ctypes
import subprocess
from pathlib import Path

import numpy as np
import pytest
from scipy.interpolate import CubicSpline, RectBivariateSpline

HERE = Path(__file__).resolve().parent
CSRC = HERE.parent / "paper_2508_15967_b200" / "csrc"


@pytest.fixture(scope="module")
def shim(tmp_path_factory):
    from helpers import build_host_shim
    return build_host_shim(tmp_path_factory.mktemp("spline"))


def _fit1(lib, x, y, stride=1):
    pp = np.empty((len(x) - 1, 4))
    assert lib.shim_fit_cubic(x.ctypes.data, y.ctypes.data, stride, len(x), pp.ctypes.data) == 0
    return pp


def _fit2(lib, R, Z, f):
    pp = np.empty((len(R) - 1, len(Z) - 1, 4, 4))
    assert lib.shim_fit_bicubic(R.ctypes.data, Z.ctypes.data, np.ascontiguousarray(f).ctypes.data, len(R), len(Z),
                                pp.ctypes.data) == pp.size
    return pp


@pytest.mark.parametrize("n", [4, 5, 9, 257])
def test_cubic_pieces_equal_scipy_not_a_knot(shim, n):
    rng = np.random.default_rng(n)
    x = np.linspace(0.0, 0.1977, n)
    y = np.cos(7 * x) + 0.3 * rng.standard_normal(n)
    pp = _fit1(shim, x, y)
    ref = CubicSpline(x, y, bc_type="not-a-knot").c[::-1].T          # scipy stores the highest power first
    scale = np.abs(ref).max(axis=0)
    assert (np.abs(pp - ref).max(axis=0) / scale).max() < 1e-10


def test_cubic_fit_reproduces_cubics_exactly_and_honours_the_stride(shim):
    x = np.linspace(-1.0, 2.0, 17)
    c = np.array([0.3, -1.2, 0.7, 2.1])
    y2 = np.zeros((17, 3))
    y2[:, 1] = c[0] + c[1] * x + c[2] * x**2 + c[3] * x**3
    pp = _fit1(shim, x, np.ascontiguousarray(y2[:, 1]))
    for i in range(16):                                               # Taylor coefficients of the cubic about x_i
        xi = x[i]
        tay = [c[0] + c[1] * xi + c[2] * xi**2 + c[3] * xi**3, c[1] + 2 * c[2] * xi + 3 * c[3] * xi**2,
               c[2] + 3 * c[3] * xi, c[3]]
        np.testing.assert_allclose(pp[i], tay, rtol=0, atol=2e-12)
    yy = np.ascontiguousarray(y2)
    pp_strided = np.empty((16, 4))
    assert shim.shim_fit_cubic(x.ctypes.data, yy.ctypes.data + 8, 3, 17, pp_strided.ctypes.data) == 0
    np.testing.assert_array_equal(pp_strided, pp)
    assert shim.shim_fit_cubic(x.ctypes.data, yy.ctypes.data, 1, 3, pp_strided.ctypes.data) == -1      # n < 4


def test_bicubic_pieces_against_scipy_and_polynomial_exactness(shim):
    R = np.linspace(0.95, 2.45, 33)
    Z = np.linspace(-0.75, 0.75, 29)
    RR, ZZ = np.meshgrid(R, Z, indexing="ij")
    f = np.log1p(2 * ((RR - 1.7) ** 2 + ZZ**2) / 0.36) * (1 + 1e-3 * np.cos(5 * RR) * np.sin(3 * ZZ))
    pp = _fit2(shim, R, Z, f)
    ref = RectBivariateSpline(R, Z, f, kx=3, ky=3, s=0)
    rng = np.random.default_rng(1)
    r = rng.uniform(R[0], R[-1], 4000)
    z = rng.uniform(Z[0], Z[-1], 4000)
    i = np.minimum(((r - R[0]) / (R[1] - R[0])).astype(int), len(R) - 2)
    j = np.minimum(((z - Z[0]) / (Z[1] - Z[0])).astype(int), len(Z) - 2)
    dr, dz = r - R[i], z - Z[j]
    p = np.arange(4)

    def ev(dp, dq):       # d^dp/dR^dp d^dq/dZ^dq of sum c[p][q] dR^p dZ^q
        out = np.zeros_like(r)
        for a in range(dp, 4):
            for b in range(dq, 4):
                fa = np.prod(np.arange(a, a - dp, -1)) if dp else 1.0
                fb = np.prod(np.arange(b, b - dq, -1)) if dq else 1.0
                out += pp[i, j, a, b] * fa * fb * dr ** (a - dp) * dz ** (b - dq)
        return out

    for dp, dq, tol in ((0, 0, 1e-13), (1, 0, 1e-11), (0, 1, 1e-11), (1, 1, 1e-10), (2, 0, 1e-9), (0, 2, 1e-9)):
        np.testing.assert_allclose(ev(dp, dq), ref.ev(r, z, dx=dp, dy=dq), rtol=0, atol=tol * max(1.0, np.abs(f).max()))
    # a bicubic polynomial is reproduced exactly by a not-a-knot tensor spline
    poly = 0.4 - RR + 0.5 * ZZ + 0.3 * RR * ZZ**2 - 0.2 * RR**3 * ZZ + 0.1 * RR**3 * ZZ**3
    pp = _fit2(shim, R, Z, poly)
    val = sum(pp[i, j, a, b] * dr**a * dz**b for a in range(4) for b in range(4))
    exact = 0.4 - r + 0.5 * z + 0.3 * r * z**2 - 0.2 * r**3 * z + 0.1 * r**3 * z**3
    np.testing.assert_allclose(val, exact, rtol=0, atol=5e-13)


@pytest.mark.parametrize("fp32", [0, 1])
def test_constant_folding_matches_the_definitions(shim, fp32):
    """Step a0: X = wpe^2/w^2 = xs * shape, Y^2 = beta |B|^2, n = c k / w, ion terms through mu = Z m_e / m_i; the derived
    constants of the reformulated stage (half gradients, field in units of sqrt(beta)) are consistent with them."""
    import scipy.constants as sc
    from paper_2508_15967_b200 import binding, inputs
    w = inputs.config(4, n_rays=1)
    desc, keep = binding.make_desc(w.eq)
    out = np.empty(16)
    rho_max = 0.98
    shim.shim_fold_params(ctypes.addressof(desc), rho_max, w.omega, fp32, out.ctypes.data)
    xs, xsh, beta, beta2, mu, mu2, opm, k2n, n2k, par_g, lin_gx, lin_gxh, sB0, sB0R0, tok_gxh, rmax2 = out
    t = inputs.TOKAMAK
    mD = sc.physical_constants["deuteron mass"][0]
    rtol = 2e-7 if fp32 else 1e-9                 # CODATA numerals typed in three places agree to < 1e-9
    assert xs == pytest.approx(t["n_ref"] * sc.e**2 / (sc.epsilon_0 * sc.m_e * w.omega**2), rel=rtol)
    assert beta == pytest.approx((sc.e / (sc.m_e * w.omega)) ** 2, rel=rtol)
    assert mu == pytest.approx(sc.m_e / mD, rel=rtol) and mu2 == pytest.approx(mu * mu, rel=rtol)
    assert opm == pytest.approx(1 + mu, rel=rtol)
    assert k2n == pytest.approx(sc.c / w.omega, rel=rtol) and k2n * n2k == pytest.approx(1.0, rel=rtol)
    assert xsh == pytest.approx(0.5 * xs, rel=rtol) and beta2 == pytest.approx(2 * beta, rel=rtol)
    assert sB0 == pytest.approx(np.sqrt(beta) * t["B0"], rel=rtol)
    assert sB0R0 == pytest.approx(np.sqrt(beta) * t["B0"] * t["R0"], rel=rtol)
    assert tok_gxh == pytest.approx(-t["p_exp"] * xs / t["a"] ** 2, rel=rtol)
    assert rmax2 == pytest.approx((rho_max * t["a"]) ** 2, rel=rtol)
    # slab constants
    w3 = inputs.config(3, n_rays=1)
    desc, keep = binding.make_desc(w3.eq)
    shim.shim_fold_params(ctypes.addressof(desc), 0.98, w3.omega, fp32, out.ctypes.data)
    xs3 = 5e19 * sc.e**2 / (sc.epsilon_0 * sc.m_e * w3.omega**2)
    assert out[10] == pytest.approx(-xs3 / 0.5, rel=rtol) and out[11] == pytest.approx(-0.5 * xs3 / 0.5, rel=rtol)
    w1 = inputs.config(1, n_rays=1)
    desc, keep = binding.make_desc(w1.eq)
    shim.shim_fold_params(ctypes.addressof(desc), 0.98, w1.omega, fp32, out.ctypes.data)
    assert out[0] == pytest.approx(0.5, rel=rtol) and out[9] == pytest.approx(0.5 / 1.0**2, rel=rtol)    # X = 1/2 (1 + r^2/L^2)


@pytest.mark.parametrize("tol", [2.0**-54, 2.0**-25])
@pytest.mark.parametrize("mu", [1 / 3670.48, 1 / 1836.15, 1 / 935.0, 1e-2, 0.0596, 0.3])
def test_series_cap_bounds_the_dropped_ion_terms(shim, mu, tol):
    """The hot loop replaces the ion terms of the Stix elements (Eq. 8-9) by their series in z = mu^2 Y2 for
    Y2 below a host-folded cap (rt_params.h: series_cap).  With 40-digit arithmetic: below the cap each of the four sums
    sig, sig', del, del' differs from its exact value by at most `tol` (a quarter ulp of the working precision) relative
    to the electron term it is added to, whatever that term's size on [0, cap] (its smallest magnitude is what the cap
    is folded against); and the cap is maximal: 2 % above it one of the bounds fails."""
    import mpmath as mp
    mp.mp.dps = 40
    cap = shim.shim_series_cap(mu, tol)
    assert cap > 0 and np.isfinite(cap)
    m = mp.mpf(mu)

    def worst(Y2):
        Y2 = mp.mpf(Y2)
        z = m * m * Y2
        e2 = 1 / (1 - z)
        # exact ion parts and their series (disp_coefs, SERIES)
        pairs = [(m * e2, m + m**3 * Y2, 1), (m**3 * e2**2, m**3, 2), (m * m * e2, m * m + m**4 * Y2, 1), (m**4 * e2**2, m**4, 2)]
        # smallest magnitude of the electron term e1 = 1 / (1 - Y2) (power p) over [0, Y2]: 1 / max(1, Y2 - 1)^p
        floor = 1 / max(mp.mpf(1), Y2 - 1)
        return max(abs(ex - se) / floor**p for ex, se, p in pairs)

    for f in (1e-3, 0.1, 0.5, 0.9, 0.999):
        assert worst(f * cap) <= tol, (mu, tol, f)
    assert worst(1.02 * cap) > tol
    assert mu * mu * cap < 0.5


def test_series_cap_without_ions_and_for_deuterium(shim):
    """Electrons only: the series is exact, no limit.  Deuterium in fp64: Y2 < 3.3, i.e. every frequency above 0.55 of the
    electron cyclotron frequency runs the fast loop."""
    assert shim.shim_series_cap(0.0, 2.0**-54) > 1e300
    cap = shim.shim_series_cap(1 / 3670.48, 2.0**-54)
    assert 3.2 < cap < 3.5
