"""CPU-only checks of the C-ABI library: it builds, loads, exports every symbol the headers under include/ declare, validates its
arguments before touching CUDA, and has no CPU fallback (compute calls fail loudly without a device)."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

from paper_2508_15967_b200 import binding, inputs
from paper_2508_15967_b200 import build as rt_build

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    rt_build.build()
    return binding.load()


def _declared_symbols():
    """Every function declared by a header under include/ (rt.h: the ray-tracing interface; rt_bench.h: measurement)."""
    names = set()
    for header in sorted((ROOT / "include").glob("*.h")):
        text = re.sub(r"/\*.*?\*/", "", header.read_text(), flags=re.S)
        names |= set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", text))
    return sorted(names)


def test_library_exports_every_declared_symbol(lib):
    declared = _declared_symbols()
    assert sorted(binding.SYMBOLS) == declared
    for name in declared:
        assert getattr(lib, name) is not None
    assert "sm_100a" in binding.version()


def test_library_embeds_sm_100a_sass_only():
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not Path(cuobjdump).exists():
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", str(binding.LIB_PATH)], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_desc_struct_matches_header_field_order():
    text = (ROOT / "include" / "rt.h").read_text()
    body = re.search(r"typedef struct rt_equilibrium_desc \{(.*?)\} rt_equilibrium_desc;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        decl = re.sub(r"^(const\s+)?(int32_t|double)\s*\*?", "", decl)
        names += [n.strip().lstrip("*") for n in decl.split(",")]
    assert names == [f[0] for f in binding.EquilibriumDesc._fields_]


def test_create_validates_descriptors(lib):
    ok = inputs.config(4, n_rays=4).eq
    eq = binding.create_equilibrium(ok)          # analytic kinds need no device
    eq.close()
    for bad in (dict(ok, a=0.0), dict(ok, B0=0.0), dict(ok, q0=0.0), dict(ok, rho_max=1.5), dict(ok, kind=7), dict(ok, a=ok["R0"]),
                dict(ok, ion_mass=-1.0), dict(ok, ion_charge=0.0), dict(ok, n_ref=float("nan")),
                dict(inputs.config(1, n_rays=4).eq, L=0.0), dict(inputs.config(3, n_rays=4).eq, L_ramp=0.0)):
        with pytest.raises(binding.RtError) as e:
            binding.create_equilibrium(bad)
        assert e.value.code == binding.RT_ERR_INVALID
    g = inputs.synth_grid(seed=3, nR=3, nZ=9, nPsi=9)
    with pytest.raises(binding.RtError) as e:
        binding.create_equilibrium(g)
    assert e.value.code == binding.RT_ERR_INVALID


def test_trace_argument_checks_come_before_cuda(lib):
    eq = binding.create_equilibrium(inputs.config(1, n_rays=4).eq)
    P = ctypes.c_void_p
    buf = np.zeros((3, 8))
    call = lambda **kw: lib.rt_trace_host(eq.handle, kw.get("disp", 0), kw.get("prec", 0), P(buf.ctypes.data),
                                          P(buf.ctypes.data), kw.get("omega", 1e11), kw.get("n", 8), kw.get("steps", 4),
                                          1e-3, kw.get("stride", 1), kw.get("traj", None), None, None, None)
    assert call(disp=1) == binding.RT_ERR_UNSUPPORTED and b"parabolic" in lib.rt_last_error()
    assert call(disp=9) == binding.RT_ERR_INVALID
    assert call(prec=5) == binding.RT_ERR_INVALID
    assert call(omega=0.0) == binding.RT_ERR_INVALID
    assert call(n=-1) == binding.RT_ERR_INVALID
    assert call(stride=0) == binding.RT_ERR_INVALID
    assert call(steps=5, stride=2, traj=P(buf.ctypes.data)) == binding.RT_ERR_INVALID
    assert call(n=0) == binding.RT_OK
    # host pointers are rejected by rt_trace (no CPU fallback), whether or not a device is present
    rc = lib.rt_trace(eq.handle, 0, 0, P(buf.ctypes.data), P(buf.ctypes.data), 1e11, 8, 4, 1e-3, 1, None, None, None, None, None)
    assert rc in (binding.RT_ERR_INVALID, binding.RT_ERR_CUDA)
    assert lib.rt_trace(None, 0, 0, None, None, 1e11, 8, 4, 1e-3, 1, None, None, None, None, None) == binding.RT_ERR_INVALID
    eq.close()


def test_orbit_and_diagnostics_argument_checks_come_before_cuda(lib):
    P = ctypes.c_void_p
    buf = np.zeros((3, 8))
    slab = binding.create_equilibrium(inputs.config(3, n_rays=4).eq)
    par = binding.create_equilibrium(inputs.config(1, n_rays=4).eq)
    call = lambda eq=slab, **kw: lib.rt_orbit(eq.handle if eq else None, kw.get("prec", 0), P(buf.ctypes.data),
                                              P(buf.ctypes.data), kw.get("qm", 4.8e7), kw.get("n", 8), kw.get("steps", 4),
                                              1e-9, kw.get("stride", 1), kw.get("traj", None), None, None, None, None)
    assert call(eq=par) == binding.RT_ERR_UNSUPPORTED and b"parabolic" in lib.rt_last_error()
    assert call(eq=None) == binding.RT_ERR_INVALID
    assert call(prec=3) == binding.RT_ERR_INVALID
    assert call(qm=float("inf")) == binding.RT_ERR_INVALID
    assert call(n=-2) == binding.RT_ERR_INVALID
    assert call(stride=0) == binding.RT_ERR_INVALID
    assert call(steps=5, stride=2, traj=P(buf.ctypes.data)) == binding.RT_ERR_INVALID
    assert call(n=0) == binding.RT_OK
    assert call() in (binding.RT_ERR_INVALID, binding.RT_ERR_CUDA)          # host pointers: no CPU fallback
    assert lib.rt_diagnostics(None, None, None, 1e11, None, 8, None, None) == binding.RT_ERR_INVALID
    assert lib.rt_diagnostics(slab.handle, None, None, -1.0, None, 8, None, None) == binding.RT_ERR_INVALID
    assert lib.rt_diagnostics(slab.handle, None, None, 1e11, None, 0, None, None) == binding.RT_OK
    assert lib.rt_trace_w(slab.handle, 1, 0, None, None, None, 0, 4, 1e-3, 1, None, None, None, None, None) == binding.RT_OK
    assert lib.rt_trace_w(slab.handle, 7, 0, None, None, None, 8, 4, 1e-3, 1, None, None, None, None, None) == binding.RT_ERR_INVALID
    assert lib.rt_launch_w(slab.handle, 1, 2, None, None, None, 8, None, None, None) == binding.RT_ERR_INVALID
    kx = lambda eq=slab, disp=2, omega=1e11, n=8, it=50, tol=1e-15: lib.rt_launch_kx(
        eq.handle if eq else None, disp, P(buf.ctypes.data), P(buf.ctypes.data), omega, None, n, it, tol,
        P(buf.ctypes.data), None, None, None)
    assert kx(eq=None) == binding.RT_ERR_INVALID
    assert kx(eq=par, disp=1) == binding.RT_ERR_UNSUPPORTED
    assert kx(omega=0.0) == binding.RT_ERR_INVALID
    assert kx(n=-1) == binding.RT_ERR_INVALID
    assert kx(it=-1) == binding.RT_ERR_INVALID and kx(it=1001) == binding.RT_ERR_INVALID
    assert kx(tol=0.0) == binding.RT_ERR_INVALID and kx(tol=float("nan")) == binding.RT_ERR_INVALID
    assert kx(n=0) == binding.RT_OK
    assert kx() in (binding.RT_ERR_INVALID, binding.RT_ERR_CUDA)            # host pointers: no CPU fallback
    until = lambda eq=slab, disp=1, omega=1e11, n=8, chunk=10, chunks=5, tol=float("inf"), info=P(buf.ctypes.data): \
        lib.rt_trace_until(eq.handle if eq else None, disp, 0, P(buf.ctypes.data), P(buf.ctypes.data), omega, n, chunk, chunks,
                           1e-3, tol, P(buf.ctypes.data), P(buf.ctypes.data), P(buf.ctypes.data), info, None)
    assert until(eq=None) == binding.RT_ERR_INVALID
    assert until(eq=par) == binding.RT_ERR_UNSUPPORTED
    assert until(omega=-1.0) == binding.RT_ERR_INVALID
    assert until(chunk=0) == binding.RT_ERR_INVALID and until(chunks=-1) == binding.RT_ERR_INVALID
    assert until(tol=0.0) == binding.RT_ERR_INVALID and until(tol=float("nan")) == binding.RT_ERR_INVALID
    assert until(n=-1) == binding.RT_ERR_INVALID
    assert until(info=None) == binding.RT_ERR_INVALID                      # out_info is required even for zero rays
    assert until() in (binding.RT_ERR_INVALID, binding.RT_ERR_CUDA)         # host pointers: no CPU fallback
    slab.close()
    par.close()


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    eq = binding.create_equilibrium(inputs.config(1, n_rays=4).eq)
    buf = np.zeros((3, 8))
    out = np.zeros((6, 8))
    P = ctypes.c_void_p
    rc = lib.rt_trace_host(eq.handle, 0, 0, P(buf.ctypes.data), P(buf.ctypes.data), 1e11, 8, 4, 1e-3, 1, None,
                           P(out.ctypes.data), None, None)
    assert rc == binding.RT_ERR_CUDA
    rate = ctypes.c_double()
    assert lib.rt_fma_peak(0, 10.0, ctypes.byref(rate), None) == binding.RT_ERR_CUDA
    assert lib.rt_fma_peak_shape(0, 1, 2, 10.0, ctypes.byref(rate), None) == binding.RT_ERR_CUDA
    assert lib.rt_fma_peak_shape(0, 5, 2, 10.0, ctypes.byref(rate), None) == binding.RT_ERR_INVALID     # packed: fp32 only
    assert lib.rt_fma_peak_shape(1, 7, 2, 10.0, ctypes.byref(rate), None) == binding.RT_ERR_INVALID
    assert lib.rt_fma_peak_shape(0, 0, 9, 10.0, ctypes.byref(rate), None) == binding.RT_ERR_INVALID
    with pytest.raises(binding.RtError):
        binding.create_equilibrium(inputs.synth_grid(seed=3, nR=9, nZ=9, nPsi=9))   # grid tables live on the device
    eq.close()


def test_product_never_imports_the_oracle():
    for path in list((ROOT / "paper_2508_15967_b200").rglob("*.py")) + list((ROOT / "paper_2508_15967_b200").rglob("*.cu*")) \
            + list((ROOT / "paper_2508_15967_b200").rglob("*.cpp")) + list((ROOT / "paper_2508_15967_b200").rglob("*.h")):
        text = path.read_text()
        assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), path
        assert "rt_oracle" not in text and "librt_oracle" not in text, path
    for path in (ROOT / "oracle").glob("*"):
        if path.suffix in (".py", ".cpp", ".h"):
            assert "paper_2508_15967_b200.binding" not in path.read_text() and "csrc" not in path.read_text().replace(
                "paper_2508_15967_b200/csrc", ""), path


def test_flop_tables_match_the_compiled_kernels(lib):
    """bench.py's algorithmic-flop and FP-instruction tables are counted from the SASS of the trace kernels
    (sass_count.py); a kernel change that alters the counts must update the tables."""
    import bench
    import sass_count
    if sass_count.cuobjdump() is None:
        pytest.skip("cuobjdump not available")
    counted = sass_count.count_kernels()
    for (cfg, prec), flops in bench.FLOPS_PER_RAY_STEP.items():
        eq, disp = bench.KERNEL_OF_CONFIG[cfg]
        got = counted[(prec, eq, disp)]
        assert got["flops"] == flops, (cfg, prec, got)
        assert got["instr"] == bench.FP_INSTR_PER_RAY_STEP[(cfg, prec)], (cfg, prec, got)
        assert got["rf3"] == bench.FP_RF3_PER_RAY_STEP[(cfg, prec)], (cfg, prec, got)
        assert got["executed"] == bench.FLOPS_EXECUTED_PER_RAY_STEP[(cfg, prec)], (cfg, prec, got)
    for prec, c in bench.ORBIT_COUNTS.items():
        got = counted[(prec, *bench.ORBIT_KERNEL)]
        assert (got["flops"] - c.get("compensation", 0), got["instr"], got["rf3"], got["executed"]) == \
               (c["flops"], c["instr"], c["rf3"], c["executed"]), (prec, got)
    # spills would show up as local-memory traffic: no trace kernel may execute a local load / store inside a ray-step,
    # and what ptxas parks outside the step loop (store staging: once per ray) stays below 64 bytes
    assert all(r["local"] == 0 for r in counted.values()), {k: r["local"] for k, r in counted.items() if r["local"]}
    report_path = ROOT / "paper_2508_15967_b200" / "librt_b200.ptxas.txt"
    if not report_path.exists():
        rt_build.build(force=True)
    report = report_path.read_text()
    blocks = report.split("Compiling entry function")
    traces = [b for b in blocks if "trace_kernel" in b.split("\n")[0]]
    # 13 (equilibrium, dispersion) pairs x 2 precisions x {one w, per-ray w, one w resuming from a status array
    # (rt_trace_until's chunk kernel)}, where the 10 plain fp32 kernels of the analytic equilibria are the packed
    # trace_kernel_x2 instead of trace_kernel<float, ...>
    assert len(traces) == 78
    assert sum("trace_kernel_x2" in b.split("\n")[0] for b in traces) == 11
    import re
    spilled = [max(int(x) for x in re.findall(r"(\d+) bytes spill stores", b)) for b in traces]
    assert max(spilled) <= 64, spilled


def test_no_trace_or_orbit_kernel_spills(lib):
    """north_star: "register spills at zero".  Every instantiation of the step-loop kernels -- trace_kernel (per-ray frequency and
    resume variants included), trace_kernel_x2, orbit_kernel -- in the ptxas report the build writes beside the library."""
    report = binding.LIB_PATH.parent / "librt_b200.ptxas.txt"
    if not report.exists() or report.stat().st_mtime < binding.LIB_PATH.stat().st_mtime - 600:
        rt_build.build(force=True)
    rows = re.findall(r"Function properties for (_ZN2rt(?:12trace_kernel|15trace_kernel_x2|12orbit_kernel)I\w+)\n\s*(\d+) bytes stack "
                      r"frame, (\d+) bytes spill stores, (\d+) bytes spill loads", report.read_text())
    assert len(rows) >= 60, len(rows)
    spilled = {name: (int(a), int(b), int(c)) for name, a, b, c in rows if int(a) or int(b) or int(c)}
    assert not spilled, spilled
