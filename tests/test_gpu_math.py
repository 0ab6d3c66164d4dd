"""GPU unit test of the hot loop's own reciprocal, reciprocal square root and square root (csrc/rt_math.cuh: rt_rcp, rt_rsqrt,
rt_sqrt_fast; run with -m gpu), through the measurement hook ``rt_math_probe``.  No output of the path shows these routines
in isolation -- 1/R from rt_rsqrt feeds every term of the tokamak and grid stages -- so their rounding error is measured here,
against 64-bit-mantissa ``numpy.longdouble`` arithmetic (x86-64; error 2^-64, i.e. 1/2000 of the fp64 rounding measured).

Bounds, derived from the code BEFORE measuring (u = 2^-53 for fp64; the Newton step's truncation error 5 e^3 / 16 with a seed
error |e| <= 2^-19 adds less than 1 %):
  rt_rcp     r + r (e + e^2): e is exact to u |e|, the last FMA rounds once                             -> (1 + 2^-6) u
  rt_rsqrt   y * fma(e, p, 1): x y is rounded before e is formed (half of it survives: u/2), the
             correction factor is rounded to 1 + delta (u) and the product once more (u)                -> 2.5 u, + 1 %
  rt_sqrt    g * fma(e, p, 1), g = x y: the same three roundings                                        -> 2.5 u, + 1 %
(the earlier form of the last step, fma(y e, p, y), rounded once: 1.5 u; the factored form saves one instruction in a loop
bound by the FP64 pipe, and 2.5 u = 2.8e-16 is 5 orders below the 1e-10 parity bar).  fp32 uses the bare MUFU seeds, whose
error PTX states: rcp.approx.ftz.f32 1 ulp (2^-23), rsqrt.approx.ftz.f32 2^-22.4; sqrt = x * rsqrt adds one rounding (2^-24).
The measured maxima are printed (pytest -s) and recorded in DESIGN.md section 7.
"""
import numpy as np
import pytest

from test_gpu_parity import rt  # noqa: F401

pytestmark = pytest.mark.gpu

U64, U32 = 2.0 ** -53, 2.0 ** -24
BOUND = {("f64", "rcp"): (1 + 2.0 ** -6) * U64, ("f64", "rsqrt"): 2.5 * U64 * 1.01, ("f64", "sqrt"): 2.5 * U64 * 1.01,
         ("f32", "rcp"): 2.0 ** -23, ("f32", "rsqrt"): 2.0 ** -22.4, ("f32", "sqrt"): 2.0 ** -22.4 + U32}


def _arguments(dtype):
    """The hot loop's arguments are normal and O(1): major radii, 1 - rho^2, squared field strengths ...  2^21 log-uniform
    draws over [1e-3, 1e3], plus the neighbourhoods of powers of two and four (where a result's ulp changes size)."""
    rng = np.random.default_rng(20250815)
    x = np.exp(rng.uniform(np.log(1e-3), np.log(1e3), 1 << 21))
    edges = np.concatenate([p * (1.0 + np.arange(-512, 513) * (2.0 ** -52 if dtype == np.float64 else 2.0 ** -23))
                            for p in (0.25, 0.5, 1.0, 2.0, 4.0, 16.0)])
    return np.ascontiguousarray(np.concatenate([x, edges]).astype(dtype))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("fn", ["rcp", "rsqrt", "sqrt"])
def test_relative_error_of_the_hot_loops_reciprocals_and_roots(rt, prec, fn):
    import torch
    if np.finfo(np.longdouble).nmant < 63:
        pytest.skip("numpy.longdouble is not the 80-bit x87 type on this machine")
    x = _arguments(np.float64 if prec == "f64" else np.float32)
    got = rt.math_probe(fn, torch.from_numpy(x).cuda()).cpu().numpy()
    xl = x.astype(np.longdouble)
    ref = {"rcp": lambda: 1 / xl, "rsqrt": lambda: 1 / np.sqrt(xl), "sqrt": lambda: np.sqrt(xl)}[fn]()
    rel = np.abs((got.astype(np.longdouble) - ref) / ref).astype(np.float64)
    worst = float(rel.max())
    print(f"\n{prec} {fn}: max relative error {worst:.3e} = {worst / (U64 if prec == 'f64' else U32):.3f} u "
          f"(bound {BOUND[prec, fn]:.3e}), mean {float(rel.mean()):.3e}")
    assert np.isfinite(got).all()
    assert worst <= BOUND[prec, fn], (worst, BOUND[prec, fn])


def test_probe_argument_checks(rt):
    import torch
    x = torch.ones(8, dtype=torch.float64, device="cuda")
    with pytest.raises(rt.RtError):
        rt.math_probe(3, x)
    with pytest.raises(ValueError):
        rt.math_probe("rcp", x.cpu())
    assert rt.math_probe("rsqrt", x[:0].contiguous()).numel() == 0
    assert torch.equal(rt.math_probe("sqrt", 4.0 * x), 2.0 * x)
