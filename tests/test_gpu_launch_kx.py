"""GPU parity tests (-m gpu) for rt_launch_kx: the paper's own launch iteration (w, x, k_y, k_z fixed, Newton on
k_x from an initial guess that selects the root) through the C ABI, against the oracle's step-by-step restatement on the same
seeded inputs.  Both sides run the same iteration, so the converged k_x agree to rounding (compared relative to |k|); the
iteration counts may differ by one where |D| passes the 1e-15 tolerance within rounding of it.
"""
import numpy as np
import pytest

from paper_2508_15967_b200 import inputs
from test_gpu_parity import _dev, _host, rt  # noqa: F401  (rt is the module-scoped fixture)

pytestmark = pytest.mark.gpu
C = inputs.C_LIGHT


def _guesses(oracle, cfg, disp, n, seed, omega=None):
    """Seeded launch points of config `cfg`, on-shell k from the oracle's direction solver, k_x detuned by +-3 %."""
    w = inputs.config(cfg, n_rays=n)
    om = w.omega if omega is None else omega
    oeq = oracle.Equilibrium(w.eq)
    x0 = w.x0.copy()
    if cfg == 3:
        x0[0] -= np.linspace(0.02, 0.35, n)          # config 3 launches at the foot (vacuum): move into the ramp
    k_on, D0 = oracle.launch(oeq, disp, x0, w.dirs, om, w.branch if disp == "cold_full" else 0)
    ok = np.isfinite(k_on).all(axis=0)
    k_on[:, ~ok] = (np.asarray(om) / C * np.ones(n))[~ok] * 0.5
    rng = np.random.default_rng(seed)
    kg = k_on.copy()
    kg[0] *= 1.0 + 0.03 * rng.choice([-1.0, 1.0], n)
    return w, oeq, x0, kg, k_on, om


@pytest.mark.parametrize("cfg,disp", [(1, "omode"), (3, "xmode"), (3, "cold_full"), (3, "omode"), (4, "cold_full"),
                                      (4, "xmode"), (4, "omode"), (5, "cold_full"), (5, "omode")])
@pytest.mark.parametrize("per_ray", [False, True])
def test_launch_kx_parity(rt, oracle, cfg, disp, per_ray):
    n = 1500 if cfg != 5 else 700
    omega = None
    if per_ray:
        omega = inputs.frequency_scan(n, inputs.config(cfg, n_rays=1).omega, seed=3000 + cfg, spread=0.05)
    w, oeq, x0, kg, k_on, om = _guesses(oracle, cfg, disp, n, seed=100 + cfg, omega=omega)
    k_ref, D_ref, it_ref = oracle.launch_kx(oeq, disp, x0, kg, om)
    eq = rt.create_equilibrium(w.eq)
    k_gpu, D_gpu, it_gpu = rt.launch_kx(eq, disp, _dev(x0), _dev(kg), _dev(om) if per_ray else om)
    k_gpu, D_gpu, it_gpu = _host(k_gpu), _host(D_gpu), _host(it_gpu)
    eq.close()
    np.testing.assert_array_equal(k_gpu[1:], kg[1:])                       # k_y, k_z are copied bit for bit
    np.testing.assert_array_equal(np.isnan(k_gpu[0]), np.isnan(k_ref[0]))  # same points outside the domain
    conv = it_ref >= 0
    assert conv.mean() > 0.6, conv.mean()      # config 3 has an evanescent layer between the cut-off and the resonance
    # well-conditioned rays (the ray is not tangent to the dispersion surface along x): same root, to rounding
    kn = np.linalg.norm(k_ref, axis=0)
    good = conv & (np.abs(k_ref[0]) > 0.3 * kn)
    assert good.sum() > 0.3 * n
    assert (it_gpu[good] >= 0).all()
    # Both sides stop as soon as |D| < 1e-15, so their last iterates may differ by the width of that band,
    # 2 tol / |dD/dk_x| (large next to a cut-off, n -> 0, or the upper-hybrid resonance, S -> 0), plus rounding of k itself.
    om_n = np.broadcast_to(np.asarray(om, dtype=np.float64), (n,))
    h = 1e-6 * kn
    kp, km = k_ref.copy(), k_ref.copy()
    kp[0] += h
    km[0] -= h
    ok_pts = np.isfinite(k_ref[0])
    dDdk = np.full(n, np.nan)
    dDdk[ok_pts] = (oracle.dispersion_value(oeq, disp, x0[:, ok_pts], kp[:, ok_pts], om_n[ok_pts])
                    - oracle.dispersion_value(oeq, disp, x0[:, ok_pts], km[:, ok_pts], om_n[ok_pts])) / (2 * h[ok_pts])
    # ... and the two sides evaluate algebraically different forms of D, whose rounding noise is of the order of an ulp of
    # the largest term, max(1, n^2)^2 (reading A18): the root of either form is only defined to noise / |dD/dk_x|
    n2_ref = (kn * C / om_n) ** 2
    bound = (4e-15 + 1e-15 * np.maximum(1.0, n2_ref) ** 2) / np.abs(dDdk) + 1e-13 * kn
    assert (np.abs(k_gpu[0] - k_ref[0])[good] <= bound[good]).all()
    assert np.median(bound[good] / kn[good]) < 1e-11           # the tolerance is not vacuous
    assert (np.abs(it_gpu[good] - it_ref[good]) <= 1).all()
    assert np.abs(D_gpu[good]).max() < 1e-15 and np.abs(D_ref[good]).max() < 1e-15
    # every ray the GPU calls converged is on shell according to the ORACLE's D at the GPU's state
    cg = it_gpu >= 0
    om_arr = np.broadcast_to(np.asarray(om, dtype=np.float64), (n,))
    D_at = oracle.dispersion_value(oeq, disp, x0[:, cg], k_gpu[:, cg], om_arr[cg])
    n2 = (np.linalg.norm(k_gpu[:, cg], axis=0) * C / om_arr[cg]) ** 2
    # D is a cancellation residue of terms of size up to n^4 (reading A18): 64 ulp of that scale (n^2 reaches 10^2 next to
    # config 3's upper-hybrid resonance)
    assert (np.abs(D_at) < 1.5e-14 * np.maximum(1.0, n2) ** 2).all()


def test_launch_kx_semantics_and_errors(rt, oracle):
    w, oeq, x0, kg, k_on, om = _guesses(oracle, 4, "cold_full", 257, seed=9)
    eq = rt.create_equilibrium(w.eq)
    xd, kd = _dev(x0), _dev(kg)
    # max_iter = 0: the guess comes back, nothing has converged
    k0, D, it = rt.launch_kx(eq, "cold_full", xd, kd, om, max_iter=0)
    np.testing.assert_array_equal(_host(k0), kg)
    assert (_host(it) == -1).all() and (np.abs(_host(D)) > 1e-9).all()
    # started on shell: zero updates, state unchanged up to the k <-> n round trip
    k1, D1, it1 = rt.launch_kx(eq, "cold_full", xd, _dev(k_on), om)
    assert (_host(it1) <= 1).all() and np.abs(_host(k1) - k_on).max() / np.abs(k_on).max() < 1e-14
    # a looser tolerance needs fewer updates; in-place operation (k0 aliasing k_guess) is allowed by the ABI
    _, _, it_loose = rt.launch_kx(eq, "cold_full", xd, kd, om, tol=1e-6)
    _, _, it_tight = rt.launch_kx(eq, "cold_full", xd, kd, om)
    assert (_host(it_loose) <= _host(it_tight)).all() and (_host(it_loose) < _host(it_tight)).any()
    # points outside the domain (rho > rho_max): NaN, -1, on both sides
    xo = x0.copy()
    xo[:, :5] *= 1.5
    k2, D2, it2 = rt.launch_kx(eq, "cold_full", _dev(xo), kd, om)
    kr, Dr, itr = oracle.launch_kx(oeq, "cold_full", xo, kg, om)
    assert np.isnan(_host(k2)[0, :5]).all() and np.isnan(_host(D2)[:5]).all() and (_host(it2)[:5] == -1).all()
    assert np.isnan(kr[0, :5]).all() and (itr[:5] == -1).all()
    # empty input and argument errors
    import torch
    e = torch.empty((3, 0), dtype=torch.float64, device="cuda")
    k3, D3, it3 = rt.launch_kx(eq, "cold_full", e, e, om)
    assert k3.shape == (3, 0)
    with pytest.raises(rt.RtError):
        rt.launch_kx(eq, "cold_full", xd, kd, om, max_iter=-1)
    with pytest.raises(rt.RtError):
        rt.launch_kx(eq, "cold_full", xd, kd, om, tol=0.0)
    with pytest.raises(rt.RtError):
        rt.launch_kx(eq, "cold_full", xd, kd, -1.0)
    eq.close()
    par = rt.create_equilibrium(inputs.config(1, n_rays=4).eq)
    with pytest.raises(rt.RtError):
        rt.launch_kx(par, "xmode", xd, kd, om)                 # no magnetic field on the parabolic slab
    par.close()
