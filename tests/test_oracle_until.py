"""Pins for the oracle's convergence workflow ``trace_until`` (CPU only; "chaining calls to evaluation and
reduction kernels until a tolerance is met", L76 reduction kernels; SURVEY 8(f)-2 "stop-when-all-frozen").

P21a  vacuum rays aimed out of the tokamak domain are straight lines: the step at which each one freezes, hence the chunk
      at which the whole ensemble is frozen, and the frozen positions follow from the exit parameter of a straight line
      through the torus rho = rho_max (root found here with brentq on the exact geometry)
P21b  config 1 never stops (its domain is all of space): max_chunks chunks run, and the result is the plain trace of
      chunk_steps * max_chunks steps bit for bit (hence the harmonic oscillator of pin P2)
P21c  the tolerance criterion: the stopping chunk is the first sample of the plain trace's |D| history above tol
P21d  a mixed ensemble (half frozen, half active) runs to max_chunks and reports the active count; max_chunks = 0
"""
import numpy as np
import pytest
from scipy.optimize import brentq

from paper_2508_15967_b200 import inputs

C = inputs.C_LIGHT


def test_p21a_vacuum_rays_freeze_at_the_computed_chunk(oracle):
    t = inputs.TOKAMAK
    w = inputs.config(4, n_rays=96)
    eq = dict(w.eq, n_ref=0.0)                                  # vacuum: O-mode rays are straight lines with |n| = 1
    d = -w.dirs                                                 # outward
    k0, D0 = oracle.launch(eq, "omode", w.x0, d, w.omega)
    np.testing.assert_allclose(np.linalg.norm(k0, axis=0) * C / w.omega, 1.0, rtol=1e-15)
    dt, chunk = 1e-3, 7

    def rho(i, tau):
        p = w.x0[:, i] + d[:, i] * tau
        return np.hypot(np.hypot(p[0], p[1]) - t["R0"], p[2]) / t["a"]

    s_freeze = np.empty(96, dtype=np.int64)
    for i in range(96):
        tau_exit = brentq(lambda tau: rho(i, tau) - t["rho_max"], 0.0, 0.3, xtol=1e-15)
        assert abs(tau_exit / dt - round(tau_exit / dt)) > 1e-6       # not on a step boundary: the count is robust
        # step s (0-based) evaluates its last stage at tau = (s + 1) dt; the ray is frozen in the first step that reaches
        # the exit, after s_freeze completed steps
        s_freeze[i] = int(np.ceil(tau_exit / dt)) - 1
    chunks_expected = int(s_freeze.max() // chunk) + 1
    out = oracle.trace_until(eq, "omode", w.x0, k0, w.omega, chunk, 1000, dt)
    assert (out["chunks"], out["reason"], out["n_active"]) == (chunks_expected, 1, 0)
    assert (out["status"] == 1).all()
    np.testing.assert_allclose(out["final"][:3], w.x0 + d * (s_freeze * dt), rtol=0, atol=1e-13)
    np.testing.assert_array_equal(out["final"][3:], k0)
    # one chunk earlier at least one ray was still active
    early = oracle.trace_until(eq, "omode", w.x0, k0, w.omega, chunk, chunks_expected - 1, dt)
    assert early["reason"] == 0 and early["n_active"] >= 1 and early["chunks"] == chunks_expected - 1


def test_p21b_config1_never_stops_and_equals_the_plain_trace(oracle):
    w = inputs.config(1, n_rays=64)
    k0, _ = oracle.launch(w.eq, w.disp, w.x0, w.dirs, w.omega)
    out = oracle.trace_until(w.eq, w.disp, w.x0, k0, w.omega, 50, 12, w.dt)
    assert (out["chunks"], out["reason"], out["n_active"]) == (12, 0, 64)
    ref = oracle.trace(w.eq, w.disp, w.x0, k0, w.omega, 600, w.dt)
    np.testing.assert_array_equal(out["final"], ref["final"])
    np.testing.assert_array_equal(out["residual"], ref["residual"])
    assert out["max_D"] == ref["residual"].max()
    W, tau = 1 / np.sqrt(2.0), 600 * w.dt                       # pin P2's closed form
    n0 = k0 * C / w.omega
    np.testing.assert_allclose(out["final"][:3], w.x0 * np.cos(W * tau) + n0 / W * np.sin(W * tau), rtol=0, atol=1e-12)


def test_p21c_tolerance_stops_at_the_first_chunk_above_it(oracle):
    w = inputs.config(3, n_rays=48)
    k0, _ = oracle.launch(w.eq, w.disp, w.x0, w.dirs, w.omega)
    dt, chunk = 2e-3, 50                                        # a coarse step: |D| grows over the first chunks
    hist = np.nanmax(oracle.trace(w.eq, w.disp, w.x0, k0, w.omega, 600, dt, chunk, traj=True)["residual"], axis=1)[1:]
    m = 2
    assert hist[:m].max() * 1.05 < hist[m]                      # chunk m's value stands clear of everything before it
    tol = 0.5 * (hist[:m].max() + hist[m])
    out = oracle.trace_until(w.eq, w.disp, w.x0, k0, w.omega, chunk, 12, dt, tol)
    assert (out["chunks"], out["reason"]) == (m + 1, 2) and out["max_D"] == hist[m] and out["n_active"] == 48
    ref = oracle.trace(w.eq, w.disp, w.x0, k0, w.omega, (m + 1) * chunk, dt)
    np.testing.assert_array_equal(out["final"], ref["final"])
    # tol = inf: the criterion is off
    assert oracle.trace_until(w.eq, w.disp, w.x0, k0, w.omega, chunk, 12, dt)["chunks"] == 12


def test_p21d_mixed_ensemble_and_degenerate_calls(oracle):
    w = inputs.config(4, n_rays=32)
    w.dirs[:, ::2] *= -1.0                                      # every other ray leaves the domain and freezes
    eq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(eq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    out = oracle.trace_until(eq, w.disp, w.x0, k0, w.omega, 25, 8, w.dt)
    assert (out["chunks"], out["reason"], out["n_active"]) == (8, 0, 16)
    assert (out["status"][::2] == 1).all() and (out["status"][1::2] == 0).all()
    ref = oracle.trace(eq, w.disp, w.x0, k0, w.omega, 200, w.dt)
    np.testing.assert_array_equal(out["final"], ref["final"])   # frozen rays stay frozen across chunks
    np.testing.assert_array_equal(out["status"], ref["status"])
    zero = oracle.trace_until(eq, w.disp, w.x0, k0, w.omega, 25, 0, w.dt)
    assert zero["chunks"] == 0 and zero["n_active"] == 32
    np.testing.assert_array_equal(zero["final"], np.concatenate([w.x0, k0]))
    with pytest.raises(ValueError):
        oracle.trace_until(eq, w.disp, w.x0, k0, w.omega, 0, 8, w.dt)
    with pytest.raises(ValueError):
        oracle.trace_until(eq, w.disp, w.x0, k0, w.omega, 25, 8, w.dt, tol=0.0)
