"""GPU parity of the convergence workflow ``rt_trace_until`` (run with -m gpu): "chaining calls to evaluation
and reduction kernels until a tolerance is met", L76; SURVEY 8(f)-2.  The loop is a CUDA-graph WHILE node whose condition is
set on the device.  Integer outputs (chunks run, active count, stop reason, status) must EQUAL the oracle's; final states
to the north-star tolerance (1e-10 / 1e-4); max |D| like every residual (64 ulp, at the same states)."""
import numpy as np
import pytest

from paper_2508_15967_b200 import inputs
from helpers import rel_err_xk
from test_gpu_parity import RES_ATOL, TOL, _dev, _host, rt  # noqa: F401

pytestmark = pytest.mark.gpu


def _case(oracle, cfg, n, outward_every=0, disp=None, eq_over=None):
    w = inputs.config(cfg, n_rays=n)
    if disp:
        w.disp = disp
    if eq_over:
        w.eq = dict(w.eq, **eq_over)
    if outward_every:
        w.dirs[:, ::outward_every] *= -1.0
    oeq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    assert np.isfinite(k0).all()
    return w, oeq, k0


@pytest.mark.parametrize("cfg,prec,chunk,max_chunks", [(4, "f64", 3, 40), (5, "f64", 4, 30), (5, "f32", 4, 30),
                                                       (3, "f64", 5, 50)])
def test_all_rays_frozen_stops_at_the_oracles_chunk(rt, oracle, cfg, prec, chunk, max_chunks):
    """Every ray aimed out of the domain: the loop stops when the last one freezes (reason 1), at the oracle's chunk."""
    n = 64 * 3 + 17
    if cfg == 3:                      # the slab's domain is x > 0: rays leave it only through the foot side...  use the
        w, oeq, k0 = _case(oracle, 4, n, disp="omode")       # analytic tokamak with the O-mode instead (another kernel)
        w.dirs *= -1.0
        k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    else:
        w, oeq, k0 = _case(oracle, cfg, n, outward_every=1)
    ref = oracle.trace_until(oeq, w.disp, w.x0, k0, w.omega, chunk, max_chunks, w.dt)
    assert ref["reason"] == 1 and 1 < ref["chunks"] < max_chunks
    eq = rt.create_equilibrium(w.eq)
    out = rt.trace_until(eq, w.disp, _dev(w.x0, prec), _dev(k0, prec), w.omega, chunk, max_chunks, w.dt)
    info = rt.until_info(out["info"])
    assert (info["chunks"], info["n_active"], info["reason"]) == (ref["chunks"], 0, 1)
    assert np.array_equal(_host(out["status"]), ref["status"])
    eq.close()


@pytest.mark.parametrize("cfg,prec", [(1, "f64"), (2, "f32"), (4, "f64"), (5, "f64")])
def test_runs_to_max_chunks_and_matches_the_plain_trace(rt, oracle, cfg, prec):
    """Nothing stops the loop: max_chunks chunks run (reason 0) and the state equals the oracle's at 1e-10 / 1e-4; a mixed
    ensemble (config 4, 5: every third ray leaves and freezes) reports the active count and keeps frozen rays frozen."""
    n, chunk, max_chunks = 128 * 2 + 9, 30, 9
    w, oeq, k0 = _case(oracle, cfg, n, outward_every=3 if cfg >= 4 else 0)
    ref = oracle.trace_until(oeq, w.disp, w.x0, k0, w.omega, chunk, max_chunks, w.dt)
    assert ref["reason"] == 0 and ref["chunks"] == max_chunks
    eq = rt.create_equilibrium(w.eq)
    x0d, k0d = _dev(w.x0, prec), _dev(k0, prec)
    out = rt.trace_until(eq, w.disp, x0d, k0d, w.omega, chunk, max_chunks, w.dt)
    info = rt.until_info(out["info"])
    assert (info["chunks"], info["n_active"], info["reason"]) == (max_chunks, ref["n_active"], 0)
    assert np.array_equal(_host(out["status"]), ref["status"])
    act = ref["status"] == 0
    ex, ek = rel_err_xk(_host(out["final"])[:, act], ref["final"][:, act])
    assert ex < TOL[prec] and ek < TOL[prec], (ex, ek)
    if (~act).any():                                    # frozen rays: same step of freezing (a one-step difference is ~1e-3)
        ex, ek = rel_err_xk(_host(out["final"])[:, ~act], ref["final"][:, ~act])
        if cfg == 4:                                    # analytic tokamak: the bar of every other ray
            bx = bk = TOL[prec]
        else:                                           # grid edge (n_e -> 0, the determinant's two roots merge): 50 x the ORACLE's
            sx = sk = 0.0                               # own sensitivity to a 1e-15 perturbation of the launch positions, capped
            for seed in (0, 1, 2):                      # at 1e-5 -- the bound test_rays_leaving_the_domain_freeze_identically derives
                x1 = w.x0 * (1.0 + 1e-15 * np.random.default_rng(seed).normal(size=w.x0.shape))
                ref1 = oracle.trace_until(oeq, w.disp, x1, k0, w.omega, chunk, max_chunks, w.dt)
                same = (~act) & (ref1["status"] == ref["status"])
                a, b = rel_err_xk(ref1["final"][:, same], ref["final"][:, same])
                sx, sk = max(sx, a), max(sk, b)
            bx, bk = min(1e-5, max(TOL[prec], 50 * sx)), min(1e-5, max(TOL[prec], 50 * sk))
        assert ex < bx and ek < bk, (ex, ek, bx, bk)
        # ... and frozen means frozen bit for bit: they froze in the first few chunks, so a run that stops 4 chunks earlier
        # leaves them in exactly the same state (their k rows do not go through the k <-> n exchange again)
        early = rt.trace_until(eq, w.disp, x0d, k0d, w.omega, chunk, max_chunks - 4, w.dt)
        fz = np.flatnonzero(~act)
        assert np.array_equal(_host(early["status"]), ref["status"])
        assert np.array_equal(_host(out["final"])[:, fz], _host(early["final"])[:, fz])
    # max |D| is the maximum of the residual row the call wrote, and that row is D at the states it wrote
    res = _host(out["residual"])
    assert info["max_D"] == np.nanmax(res)
    D_at = np.abs(oracle.dispersion_value(oeq, w.disp, _host(out["final"])[:3], _host(out["final"])[3:], w.omega))
    ok = np.isfinite(D_at)
    assert np.array_equal(np.isfinite(res), ok) and np.abs(res[ok] - D_at[ok]).max() <= RES_ATOL[prec]
    eq.close()


def test_tolerance_stops_at_the_oracles_chunk(rt, oracle):
    """Config 3 at a coarse step: |D| grows chunk by chunk; tol sits between two consecutive chunk maxima of the ORACLE's
    history, well clear of both, so both sides must stop at the same chunk with reason 2."""
    w, oeq, k0 = _case(oracle, 3, 200)
    dt, chunk = 2e-3, 50
    hist = np.nanmax(oracle.trace(oeq, w.disp, w.x0, k0, w.omega, 600, dt, chunk, traj=True)["residual"], axis=1)[1:]
    m = next(j for j in range(1, len(hist)) if hist[j] > 1.05 * hist[:j].max())
    tol = 0.5 * (hist[:m].max() + hist[m])
    ref = oracle.trace_until(oeq, w.disp, w.x0, k0, w.omega, chunk, 12, dt, tol)
    assert (ref["chunks"], ref["reason"]) == (m + 1, 2)
    eq = rt.create_equilibrium(w.eq)
    out = rt.trace_until(eq, w.disp, _dev(w.x0), _dev(k0), w.omega, chunk, 12, dt, tol)
    info = rt.until_info(out["info"])
    assert (info["chunks"], info["reason"], info["n_active"]) == (m + 1, 2, 200)
    assert abs(info["max_D"] - ref["max_D"]) < 1e-3 * ref["max_D"]
    ex, ek = rel_err_xk(_host(out["final"]), ref["final"])
    assert ex < 1e-10 and ek < 1e-10
    eq.close()


def test_degenerate_calls_and_argument_errors(rt, oracle):
    import torch
    w, oeq, k0 = _case(oracle, 4, 70)
    eq = rt.create_equilibrium(w.eq)
    x0d, k0d = _dev(w.x0), _dev(k0)
    out = rt.trace_until(eq, w.disp, x0d, k0d, w.omega, 10, 0, w.dt)                     # max_chunks = 0
    info = rt.until_info(out["info"])
    assert (info["chunks"], info["n_active"], info["reason"]) == (0, 70, 0)
    assert np.array_equal(_host(out["final"])[:3], w.x0)
    np.testing.assert_allclose(_host(out["final"])[3:], k0, rtol=1e-15)
    one = rt.trace_until(eq, w.disp, x0d, k0d, w.omega, 40, 1, w.dt)                     # one chunk == rt_trace
    plain = rt.trace(eq, w.disp, x0d, k0d, w.omega, 40, w.dt)
    assert torch.equal(one["final"], plain["final"]) and torch.equal(one["status"], plain["status"])
    assert torch.equal(one["residual"], plain["residual"])
    # fp32: the chunk kernel is the scalar trace_kernel<float> (resuming), the plain call the packed trace_kernel_x2 -- the same
    # IEEE operations on each ray, so one chunk must reproduce the plain call (to rounding: the compiler may contract a
    # multiply-add pair of the scalar code that stays two packed instructions)
    x32, k32 = x0d.float().contiguous(), k0d.float().contiguous()
    one32 = rt.trace_until(eq, w.disp, x32, k32, w.omega, 40, 1, w.dt)
    plain32 = rt.trace(eq, w.disp, x32, k32, w.omega, 40, w.dt)
    assert torch.equal(one32["status"], plain32["status"])
    assert float(((one32["final"] - plain32["final"]).abs() / plain32["final"].abs().amax(dim=1, keepdim=True)).max()) < 2e-6
    e = torch.empty((3, 0), dtype=torch.float64, device="cuda")                          # zero rays: as the oracle's loop over an
    z = rt.until_info(rt.trace_until(eq, w.disp, e, e.clone(), w.omega, 10, 5, w.dt)["info"])   # empty ensemble (one chunk, then
    assert (z["chunks"], z["n_active"], z["reason"]) == (1, 0, 1)                        # "every ray frozen"); see the test below
    for bad in (dict(chunk_steps=0), dict(max_chunks=-1), dict(tol=0.0), dict(tol=float("nan"))):
        kw = dict(chunk_steps=10, max_chunks=3, tol=float("inf"))
        kw.update(bad)
        with pytest.raises(rt.RtError):
            rt.trace_until(eq, w.disp, x0d, k0d, w.omega, kw["chunk_steps"], kw["max_chunks"], w.dt, kw["tol"])
    eq.close()


def test_the_call_returns_before_the_loop_has_finished(rt, oracle):
    """No host synchronisation anywhere in the workflow: on a side stream the call returns while the graph is still
    running (an event recorded right after it has not completed yet), and the result is the same as on the default stream."""
    import torch
    n = 1 << 19
    w = inputs.config(4, n_rays=n)
    eq = rt.create_equilibrium(w.eq)
    x0d = _dev(w.x0)
    k0d, _ = rt.launch(eq, w.disp, x0d, _dev(w.dirs), w.omega, w.branch)
    ref = rt.trace_until(eq, w.disp, x0d, k0d, w.omega, 100, 10, w.dt)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        out = rt.trace_until(eq, w.disp, x0d, k0d, w.omega, 100, 10, w.dt)
        ev = torch.cuda.Event()
        ev.record(side)
    assert not ev.query()                       # ~20 ms of device work is still in flight when the call has returned
    ev.synchronize()
    assert torch.equal(out["final"], ref["final"]) and torch.equal(out["info"][:4], ref["info"][:4])
    assert rt.until_info(out["info"])["chunks"] == 10
    eq.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_edge_contracts_equal_the_oracles(rt, oracle, prec):
    """The two corners where the loop does not run as usual, against oracle.trace_until (not against typed values):
    max_chunks = 0 reports the launch state and makes NO stop test -- reason 0 ("max_chunks reached") even when max |D| at
    launch already exceeds tol; an empty ensemble with max_chunks > 0 goes through the loop once (1 chunk, no active ray,
    reason 1), with max_chunks = 0 not at all."""
    import torch
    n = 64 + 13
    w, oeq, k0 = _case(oracle, 4, n)
    k0 = k0 * 1.001                                   # off the dispersion surface: |D| ~ 1e-5 at launch, above tol
    tol = 1e-6
    eq = rt.create_equilibrium(w.eq)
    ref = oracle.trace_until(oeq, w.disp, w.x0, k0, w.omega, 10, 0, w.dt, tol)
    assert (ref["chunks"], ref["n_active"], ref["reason"]) == (0, n, 0) and ref["max_D"] > 10 * tol
    out = rt.trace_until(eq, w.disp, _dev(w.x0, prec), _dev(k0, prec), w.omega, 10, 0, w.dt, tol)
    info = rt.until_info(out["info"])
    assert (info["chunks"], info["n_active"], info["reason"]) == (ref["chunks"], ref["n_active"], ref["reason"])
    assert abs(info["max_D"] - ref["max_D"]) <= (1e-12 if prec == "f64" else 1e-3) * ref["max_D"] + RES_ATOL[prec]
    assert np.array_equal(_host(out["status"]), ref["status"])
    launch_state = _host(torch.cat([_dev(w.x0, prec), _dev(k0, prec)]))      # x rows as given; k rows go through k -> n -> k
    assert np.array_equal(_host(out["final"])[:3], launch_state[:3])
    assert np.allclose(_host(out["final"])[3:], launch_state[3:], rtol=4 * (2.2e-16 if prec == "f64" else 1.2e-7), atol=0)
    assert np.allclose(_host(out["final"]), ref["final"], rtol=4 * (2.2e-16 if prec == "f64" else 1.2e-7), atol=0)
    # one chunk from the same launch state does stop on the tolerance (reason 2): the test is made after a chunk, never before
    ref1 = oracle.trace_until(oeq, w.disp, w.x0, k0, w.omega, 10, 3, w.dt, tol)
    info1 = rt.until_info(rt.trace_until(eq, w.disp, _dev(w.x0, prec), _dev(k0, prec), w.omega, 10, 3, w.dt, tol)["info"])
    assert (ref1["chunks"], ref1["reason"]) == (1, 2)
    assert (info1["chunks"], info1["n_active"], info1["reason"]) == (ref1["chunks"], ref1["n_active"], ref1["reason"])
    # no rays
    e = torch.empty((3, 0), dtype=torch.float64 if prec == "f64" else torch.float32, device="cuda")
    for max_chunks in (0, 1, 5):
        ref0 = oracle.trace_until(oeq, w.disp, np.empty((3, 0)), np.empty((3, 0)), w.omega, 10, max_chunks, w.dt, tol)
        got0 = rt.until_info(rt.trace_until(eq, w.disp, e, e.clone(), w.omega, 10, max_chunks, w.dt, tol)["info"])
        assert (got0["chunks"], got0["n_active"], got0["reason"], got0["max_D"]) == \
               (ref0["chunks"], ref0["n_active"], ref0["reason"], ref0["max_D"]), max_chunks
    assert (ref0["chunks"], ref0["reason"]) == (1, 1)
    eq.close()
