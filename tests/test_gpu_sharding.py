"""Partition invariance on ONE GPU (run with -m gpu): the ray-range partition of an ensemble (strong scaling
by splitting the ensemble over devices) changes nothing -- tracing the ranges
``sharding.ray_range(n, r, world)`` of one seeded ensemble in separate calls and concatenating gives, bit for bit, the
result of the single call.  This is what makes `bench.py --scaling strong` a measurement of the same computation; no
second GPU is needed to check it."""
import numpy as np
import pytest

from paper_2508_15967_b200 import inputs, sharding
from test_gpu_parity import _dev, rt  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,prec,world", [(4, "f64", 3), (5, "f32", 3), (2, "f64", 5)])
def test_ray_range_partition_is_bit_identical_to_the_single_call(rt, cfg, prec, world):
    import torch
    n, steps = 10007, 120                         # a prime: ragged ranges, rows that are not 16-byte aligned
    w = inputs.config(cfg, n_rays=n, n_steps=steps)
    eq = rt.create_equilibrium(w.eq)
    x0d = _dev(w.x0)
    k0d, _ = rt.launch(eq, w.disp, x0d, _dev(w.dirs), w.omega, w.branch)
    if prec == "f32":
        x0d, k0d = x0d.float().contiguous(), k0d.float().contiguous()
    stride = 40
    whole = rt.trace(eq, w.disp, x0d, k0d, w.omega, steps, w.dt, stride, traj=True)
    parts = []
    for r in range(world):
        b, e = sharding.ray_range(n, r, world)
        parts.append(rt.trace(eq, w.disp, x0d[:, b:e].contiguous(), k0d[:, b:e].contiguous(), w.omega, steps, w.dt, stride,
                              traj=True))
    torch.cuda.synchronize()
    assert sum(p["status"].numel() for p in parts) == n
    for key, axis in (("traj", 2), ("final", 1), ("residual", 1), ("status", 0)):
        cat = torch.cat([p[key] for p in parts], dim=axis)
        a, b = whole[key].cpu().numpy(), cat.cpu().numpy()
        assert a.shape == b.shape and np.array_equal(a, b, equal_nan=True), key
    eq.close()
