"""Tests of ``rt_trace_host_noalloc`` (the two GPU tests run with -m gpu; the file name makes pytest collect it last, so a
failure here cannot hide another test behind ``-x``).

Who needs that entry point: a program that cannot let a library allocate device memory in the middle of its run --
because it holds the whole GPU in a memory pool of its own, because it cannot stand the device-wide stall of a cudaMalloc /
cudaFree, or because its device memory is fixed before it starts.  ``rt_trace_host`` stages the rays in buffers from
cudaMalloc; ``rt_trace_host_noalloc`` stages them in a 64 MiB array that is part of the library image
(``RT_NOALLOC_SCRATCH_BYTES``) and makes no allocation at all.

What is checked: the new entry point against the existing path (``rt_trace_host``; both run the same kernels, so the
comparison is bit for bit, well inside the 1e-10 / 1e-4 the parity tests allow) on TWO calls in a row that share the array --
the second with other rays, another size, another precision and another set of outputs, so that anything the first call left
behind would show; that the calls allocate no device memory; and that a call beyond the limit is refused with a message
that names it.  The test does not depend on what ran before it: it passes alone in a fresh process (where its first call is
the one that looks the array's address up) and after the other GPU tests.
"""
import numpy as np
import pytest

from paper_2508_15967_b200 import inputs
from test_gpu_parity import TOL, _dev, rt  # noqa: F401
from helpers import rel_err_xk



def _launch_states(rt, w, eq, prec):
    x0d = _dev(w.x0)
    k0d, _ = rt.launch(eq, w.disp, x0d, _dev(w.dirs), w.omega, w.branch)
    dt = np.float64 if prec == "f64" else np.float32
    return x0d.cpu().numpy().astype(dt), k0d.cpu().numpy().astype(dt)


def _same(a: dict, b: dict, prec):
    assert a.keys() == b.keys()
    for key in a:
        x, y = np.asarray(a[key]), np.asarray(b[key])
        assert x.shape == y.shape and x.dtype == y.dtype, key
        assert np.array_equal(x, y, equal_nan=True), key
    # the same statement at the tolerance of the parity tests (implied by the equality above; kept so that the bar is written here)
    ex, ek = rel_err_xk(a["final"], b["final"])
    assert ex <= TOL[prec] and ek <= TOL[prec]


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_allocating_path(rt):
    import torch
    # call 1: config 4 (full determinant, analytic tokamak), fp64, trajectory + every output; 1003 rays: ragged sections
    w1 = inputs.config(4, n_rays=1003, n_steps=60)
    eq1 = rt.create_equilibrium(w1.eq)
    x1, k1 = _launch_states(rt, w1, eq1, "f64")
    # call 2: config 2 (O-mode, linear slab), fp32 (the packed two-rays-per-thread kernel), fewer rays (an odd number), final
    # state only, no status: every section of the array sits somewhere else and holds call 1's bytes when it starts
    w2 = inputs.config(2, n_rays=777, n_steps=45)
    eq2 = rt.create_equilibrium(w2.eq)
    x2, k2 = _launch_states(rt, w2, eq2, "f32")
    ref1 = rt.trace_host(eq1, w1.disp, x1, k1, w1.omega, 60, w1.dt, 20, traj=True)
    ref2 = rt.trace_host(eq2, w2.disp, x2, k2, w2.omega, 45, w2.dt, traj=False, status=False)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    got1 = rt.trace_host_noalloc(eq1, w1.disp, x1, k1, w1.omega, 60, w1.dt, 20, traj=True)
    got2 = rt.trace_host_noalloc(eq2, w2.disp, x2, k2, w2.omega, 45, w2.dt, traj=False, status=False)
    free_after = torch.cuda.mem_get_info()[0]
    assert got1["traj"].shape == (4, 6, 1003) and got1["status"].dtype == np.int32 and "status" not in got2
    _same(got1, ref1, "f64")
    _same(got2, ref2, "f32")
    assert np.isfinite(got1["final"]).all() and np.isfinite(got2["final"]).all()
    # the two calls took no device memory (all inputs here are numpy arrays: nothing else allocates in between)
    assert free_after >= free_before, (free_before, free_after)
    # and once more, call 1 after call 2, through CPU torch tensors on a side stream
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        got3 = rt.trace_host_noalloc(eq1, w1.disp, torch.from_numpy(x1), torch.from_numpy(k1), w1.omega, 60, w1.dt, 20, traj=True)
    _same({k: v.numpy() for k, v in got3.items()}, ref1, "f64")
    eq1.close()
    eq2.close()


@pytest.mark.gpu
def test_a_call_beyond_the_static_array_is_refused(rt):
    w = inputs.config(1, n_rays=1024, n_steps=1000)                 # BASELINE.json config 1, all 1001 samples, fp64: 55 MiB
    eq = rt.create_equilibrium(w.eq)
    x0, k0 = _launch_states(rt, w, eq, "f64")
    fits = rt.trace_host_noalloc(eq, w.disp, x0, k0, w.omega, 1000, w.dt, 1, traj=True)
    ref = rt.trace_host(eq, w.disp, x0, k0, w.omega, 1000, w.dt, 1, traj=True)
    _same(fits, ref, "f64")
    n = 1300                                                          # 1300 x 7019 values x 8 bytes = 70 MiB > 64 MiB
    x0b, k0b = (np.ascontiguousarray(np.concatenate([a, a[:, :n - 1024]], axis=1)) for a in (x0, k0))
    with pytest.raises(rt.RtError) as err:
        rt.trace_host_noalloc(eq, w.disp, x0b, k0b, w.omega, 1000, w.dt, 1, traj=True)
    assert err.value.code == rt.RT_ERR_INVALID
    assert "RT_NOALLOC_SCRATCH_BYTES" in str(err.value) and str(rt.NOALLOC_SCRATCH_BYTES) in str(err.value)
    # the same rays fit without the trajectory, and the refusal has left the library usable
    small = rt.trace_host_noalloc(eq, w.disp, x0b, k0b, w.omega, 1000, w.dt, 1, traj=False)
    assert np.array_equal(small["final"][:, :1024], fits["final"]) and np.array_equal(small["status"][:1024], fits["status"])
    # no rays: nothing to do, and no complaint
    empty = rt.trace_host_noalloc(eq, w.disp, x0[:, :0], k0[:, :0], w.omega, 10, w.dt)
    assert empty["final"].shape == (6, 0)
    eq.close()


def test_the_size_limit_is_checked_before_cuda_is_touched():
    """No GPU needed: the refusal of a call that does not fit comes from the argument checks, so a caller learns about
    it on any machine, with nothing enqueued (the header's value, the binding's and the message's are one number)."""
    import ctypes
    import re
    from pathlib import Path
    from paper_2508_15967_b200 import binding
    from paper_2508_15967_b200 import build as rt_build
    rt_build.build()
    lib = binding.load()
    header = (Path(__file__).resolve().parent.parent / "include" / "rt.h").read_text()
    shift = re.search(r"#define RT_NOALLOC_SCRATCH_BYTES \((\d+)ll << (\d+)\)", header)
    assert int(shift.group(1)) << int(shift.group(2)) == binding.NOALLOC_SCRATCH_BYTES == 64 << 20
    eq = binding.create_equilibrium(inputs.config(1, n_rays=4).eq)
    P = ctypes.c_void_p
    buf = np.zeros(8)                                       # never read: the calls below are refused before any copy
    call = lambda n, steps, prec=0, traj=None: lib.rt_trace_host_noalloc(
        eq.handle, 0, prec, P(buf.ctypes.data), P(buf.ctypes.data), 1e11, n, steps, 1e-3, 1, traj, P(buf.ctypes.data), None,
        None, None)
    per_ray = 6 * 8 + 6 * 8                                 # x0, k0 and out_final in fp64
    n_max = (64 << 20) // per_ray // 32 * 32                # rows of 32 k rays are whole multiples of 256 bytes: no padding
    assert call(n_max + 32, 4) == binding.RT_ERR_INVALID
    msg = lib.rt_last_error().decode()
    assert "RT_NOALLOC_SCRATCH_BYTES" in msg and str(64 << 20) in msg and str((n_max + 32) * per_ray) in msg
    assert call(1500, 1000, traj=P(buf.ctypes.data)) == binding.RT_ERR_INVALID      # 69 MiB of trajectory
    assert call(1 << 40, 4) == binding.RT_ERR_INVALID and call(4, 1 << 62, traj=P(buf.ctypes.data)) == binding.RT_ERR_INVALID
    assert call(-1, 4) == binding.RT_ERR_INVALID and call(0, 4) == binding.RT_OK
    assert lib.rt_trace_host_noalloc(None, 0, 0, None, None, 1e11, 8, 4, 1e-3, 1, None, None, None, None, None) == binding.RT_ERR_INVALID
    eq.close()
