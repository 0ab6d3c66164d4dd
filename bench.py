#!/usr/bin/env python
"""bench.py -- ray-steps/s of the batched RF ray tracer on B200 (BASELINE.json's metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--precision f64] [--impl ours|reference]
                    [--scaling weak|strong]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path over one batch: one ``rt_trace`` call that loads the launch states, runs all
RK4 steps of every ray and writes the config's outputs.  The default workload is BASELINE.json
config 4 -- the configuration the north-star target is quoted on (2^20 rays x 1000 steps, full Stix determinant,
analytic tokamak, fp64, trajectories decimated every 10 steps).  Inputs are seeded and synthetic (inputs.py) and are
resident in HBM when the timed region starts; launch wave vectors come from the library's own ``rt_launch`` kernel.

`value`        = (rays all ranks traced) * n_steps * K / (max-over-ranks device time of K steps).  ``--scaling weak``
                 (default): every rank traces its own full-size seeded batch; ``--scaling strong``: ONE seeded ensemble of
                 the config's size is split into contiguous ray ranges, rank r traces ``sharding.ray_range(n, r, world)``
                 (the paper's own multi-device experiment).  No collective on the data path either way.
`e2e`          = the same metric through ``rt_trace_host`` with pinned HOST buffers (H2D + kernel + D2H per step)
`roofline`     = bound "alu": algorithmic flops per launch / mean kernel time (CUDA events on the launch stream) against
                 2 x the DFMA (FFMA) rate measured by ``rt_fma_peak`` in this process
`cpu_baseline` = the CPU oracle, as it stands, on a bounded sample of the same workload (rank 0, N = 1 only)
``--impl reference`` times the oracle alone (the reference arm of this tier).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_2508_15967_b200 import inputs  # noqa: E402

METRIC = "ray_steps_per_s"
UNIT = "ray-steps/s"

# Algorithmic flops per ray-step: adds + multiplies + divisions + square roots of the hand-derived
# formulation, one RK4 step = 4 right-hand sides + the tableau; a fused multiply-add counts 2, a division or square root 1
# (its Newton refinement is NOT counted).  FP_INSTR_PER_RAY_STEP is what the FP64 / FP32 pipe actually issues per
# ray-step (FMA, MUL, ADD, SETP instructions, refinements included).  Both tables are counted from the compiled kernels by
# tests/sass_count.py and pinned to it by tests/test_abi.py::test_flop_tables_match_the_compiled_kernels.
FLOPS_PER_RAY_STEP = {(1, "f64"): 115, (2, "f64"): 115, (3, "f64"): 243, (4, "f64"): 707, (5, "f64"): 1200,
                      (1, "f32"): 117, (2, "f32"): 117, (3, "f32"): 246, (4, "f32"): 711, (5, "f32"): 1200}
# FLOPS_EXECUTED_PER_RAY_STEP: flops as the kernel executes them (2 per fused multiply-add, 1 per multiply / add, Newton
# refinements included) -- SURVEY.md section 8(d)'s own numerator, what ncu's op_dfma / op_dmul / op_dadd counters add up to.
FLOPS_EXECUTED_PER_RAY_STEP = {(1, "f64"): 135, (2, "f64"): 135, (3, "f64"): 303, (4, "f64"): 843, (5, "f64"): 1288,
                               (1, "f32"): 113, (2, "f32"): 113, (3, "f32"): 234, (4, "f32"): 687, (5, "f32"): 1184}
FP_INSTR_PER_RAY_STEP = {(1, "f64"): 75, (2, "f64"): 75, (3, "f64"): 193, (4, "f64"): 553, (5, "f64"): 820,
                         (1, "f32"): 70, (2, "f32"): 70, (3, "f32"): 174, (4, "f32"): 484, (5, "f32"): 775}
# FP_RF3_PER_RAY_STEP: how many of those instructions read THREE DISTINCT registers from the register file.  Such an instruction
# occupies the FP64 pipe for 3 cycles instead of 2 (scalar FP32: 1.56 slots instead of 1; packed f32x2: 3 cycles instead of 2) -- measured by
# rt_fma_peak_shape, shapes 2 / 6 (profiles/r2_fma_peak_shapes.md) -- so the pipe time of a ray-step is
# (instr + RF3_EXTRA * rf3) issue slots of the FMA microbenchmark; `pipe_model_frac` is that time over the measured kernel
# time.  The fp32 kernels of the analytic equilibria (configs 1-4) are the packed two-rays-per-thread
# kernels (trace_kernel_x2); their counts are per ray (a packed instruction = one slot per ray).
FP_RF3_PER_RAY_STEP = {(1, "f64"): 27, (2, "f64"): 27, (3, "f64"): 37, (4, "f64"): 134, (5, "f64"): 312,
                       (1, "f32"): 32, (2, "f32"): 32, (3, "f32"): 42, (4, "f32"): 143, (5, "f32"): 258}
RF3_EXTRA = {"f64": 0.5, "f32": 0.563, "f32x2": 0.507}   # shape 0 / shape 2 - 1: 63.9 / 42.7, 123.2 / 78.8; packed 127.9 / 84.9
PACKED = {(c, "f32") for c in (1, 2, 3, 4, 5)}           # (config, precision) pairs that run trace_kernel_x2
# The second ensemble workload (rt_orbit on config 4's tokamak): the same three counts per PARTICLE-step, from
# sass_count.py's orbit_kernel rows (pinned by the same test).
# fp32: 12 of the executed adds are the compensated position update (rt_kernels.cuh: orbit_step), not work of the method:
# sass_count's flop count includes them, the algorithmic figure here does not.
ORBIT_COUNTS = {"f64": dict(flops=238, instr=184, rf3=50, executed=286),
                "f32": dict(flops=238, instr=174, rf3=49, executed=242, compensation=12)}
ORBIT_KERNEL = (2, "orbit")
# (equilibrium kind, dispersion kind) of rt_math.cuh behind each config: the key sass_count.py reports under
KERNEL_OF_CONFIG = {1: (0, 0), 2: (0, 0), 3: (1, 1), 4: (2, 2), 5: (3, 2)}
# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of each kernel from the committed `ncu --set full`
# captures of this build: profiles/r2_cfg4_f64_ncu_g.md (headline), profiles/r2_other_configs_ncu_g.md (the others)
NCU_DRAM_BYTES = {(4, "f64"): 5.986e9, (2, "f64"): 6.64e7, (2, "f32"): 2.55e7, (3, "f64"): 1.26e7, (4, "f32"): 2.964e9,
                  (5, "f64"): 1.832e9, (5, "f32"): 9.14e8, ("orbit4", "f64"): 5.976e9}

WORKLOAD_NAMES = {
    1: "cfg1: O-mode, parabolic slab, 1024 rays x 1000 steps, full trajectory",
    2: "cfg2: O-mode, parabolic slab, 2^20 rays x 2000 steps, final state + |D|",
    3: "cfg3: X-mode, e+D, B0R0/R slab with linear density ramp, 2^18 rays x 3000 steps, final state + |D|",
    4: "cfg4: full Stix determinant, e+D, analytic circular tokamak, 2^20 rays x 1000 steps, trajectory every 10 steps + |D|",
    5: "cfg5: full Stix determinant, e+D, 257x257 bicubic-spline R-Z grid, 2^24 rays x 500 steps, final state + |D|",
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--n-rays", type=int, default=None, help="override the config's ray count (debugging only)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the secondary per-config table")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons while the timed region runs (nvidia-smi, the profiling recipe's line)."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        # "under load": samples at or above half the maximum power seen
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        thr = 0.5 * max(pw)
        load = [s for s, p in zip(sm, pw) if p >= thr] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ CPU oracle legs
def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    import platform
    return platform.processor() or platform.machine()


def host_cores() -> int:
    """All host cores this process may run on (torchrun exports OMP_NUM_THREADS=1, which omp_get_max_threads() would obey;
    under torchrun only rank 0 runs the oracle, so the cores are its own)."""
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def oracle_rate(cfg: int, target_s: float, n_threads: int = 0):
    """Time the CPU oracle, as it stands, on a bounded sample of config `cfg`: the first n rays of the seeded launch set
    at the config's full step count, n sized from a short calibration so the run takes about `target_s` seconds.
    n_threads = 0: every host core; 1: the single-thread leg."""
    import oracle
    oracle.build()
    cores = max(host_cores(), oracle.max_threads()) if n_threads <= 0 else n_threads
    n_steps = inputs.FULL_SIZES[cfg][1]
    probe_n = 64 * cores if cores > 1 else 16    # enough rays that every thread of the dynamic schedule (chunks of 16) is busy
    w = inputs.config(cfg, n_rays=probe_n, n_steps=n_steps)
    oeq = oracle.Equilibrium(w.eq)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    oracle.trace(oeq, w.disp, w.x0, k0, w.omega, max(1, n_steps // 10), w.dt, n_threads=cores)   # thread start-up
    t0 = time.perf_counter()
    oracle.trace(oeq, w.disp, w.x0, k0, w.omega, n_steps, w.dt, n_threads=cores)
    t_probe = time.perf_counter() - t0
    n = int(max(probe_n, min(inputs.FULL_SIZES[cfg][0], probe_n * target_s / max(t_probe, 1e-6))))
    n = max(cores, n // cores * cores)
    w = inputs.config(cfg, n_rays=n, n_steps=n_steps)
    k0, _ = oracle.launch(oeq, w.disp, w.x0, w.dirs, w.omega, w.branch)
    stride = w.save_stride if w.save_stride > 0 else 1

    def run_once():
        t0 = time.perf_counter()
        oracle.trace(oeq, w.disp, w.x0, k0, w.omega, n_steps, w.dt, stride, traj=w.save_stride > 0, n_threads=cores)
        return time.perf_counter() - t0

    return run_once, n, n_steps, cores


def cpu_baseline(cfg: int, target_s: float = 12.0, single_thread_s: float = 6.0) -> dict:
    """the oracle timed (a) on every host core and (b) on one thread (single_thread_s = 0: leg (a) only), core
    count and CPU model stated.  The single-thread leg is reported in scalar keys beside the all-cores ones."""
    run_once, n, n_steps, cores = oracle_rate(cfg, target_s=target_s)
    t = run_once()
    out = {"value": n * n_steps / t, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": round(t, 2),
           "sample": f"first {n} rays of config {cfg}'s seeded launch set x {n_steps} steps (fp64, OpenMP over rays)",
           "cpu_model": cpu_model()}
    if single_thread_s > 0:
        run1, n1, _, _ = oracle_rate(cfg, target_s=single_thread_s, n_threads=1)
        t1 = run1()
        out.update({"single_thread_value": n1 * n_steps / t1, "single_thread_seconds": round(t1, 2),
                    "single_thread_sample": f"first {n1} rays of the same launch set x {n_steps} steps, one thread"})
    return out


def workload_config(cfg: int, scaling: str) -> dict:
    """The `config` object of the JSON line: the same keys and values on both arms (the reference arm times a bounded
    sample of this workload; what the sample was is said under `cpu_baseline.sample`)."""
    n_rays, n_steps = inputs.FULL_SIZES[cfg]
    return {"workload": WORKLOAD_NAMES[cfg], "n_rays": n_rays, "n_steps": n_steps, "rays_per_gpu": "n_rays (weak: one "
            "seeded batch per rank)" if scaling == "weak" else "n_rays / n_gpus (strong: contiguous ranges of one ensemble)",
            "l2": "flushed between steps (256 MiB memset)", "sharding": "independent rays, no collective"}


def run_reference(args) -> int:
    """--impl reference: the oracle timed on the host cores, same metric / config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    cfg = args.config
    run_once, n, n_steps, cores = oracle_rate(cfg, target_s=3.0)
    for _ in range(args.warmup):
        run_once()
    t = sum(run_once() for _ in range(args.steps))
    value = n * n_steps * args.steps / t
    sample = f"first {n} rays of config {cfg}'s seeded launch set x {n_steps} steps per step (fp64, OpenMP over rays)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, args.scaling),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ the CUDA arm
class Job:
    """One config resident on the current device: equilibrium handle, launch states, preallocated outputs.
    ray_range = (begin, end): trace only that contiguous range of the seeded ensemble (strong scaling)."""

    def __init__(self, rt, torch, cfg: int, prec: str, n_rays, seed: int, scan: bool = False, ray_range=None):
        self.rt, self.torch, self.cfg, self.prec = rt, torch, cfg, prec
        self.w = w = inputs.config(cfg, n_rays=n_rays, seed=seed)
        b, e = ray_range if ray_range is not None else (0, w.n_rays)
        self.n = e - b
        self.eq = rt.create_equilibrium(w.eq)
        dt = torch.float64 if prec == "f64" else torch.float32
        x0 = torch.from_numpy(np.ascontiguousarray(w.x0[:, b:e])).cuda()
        # scan: a frequency scan, one w per ray (rt_launch_w / rt_trace_w); else the config's single frequency
        self.omega = torch.from_numpy(inputs.frequency_scan(w.n_rays, w.omega, seed)[b:e].copy()).cuda() if scan else w.omega
        k0, D0 = rt.launch(self.eq, w.disp, x0, torch.from_numpy(np.ascontiguousarray(w.dirs[:, b:e])).cuda(), self.omega,
                           w.branch)
        if not bool(torch.isfinite(k0).all()):
            raise RuntimeError("rt_launch returned non-finite launch states for a bench workload")
        self.launch_residual = float(D0.abs().max()) if self.n else 0.0
        self.x0, self.k0 = x0.to(dt).contiguous(), k0.to(dt).contiguous()
        self.traj = w.save_stride > 0
        self.stride = w.save_stride if self.traj else 1
        self.out = {}
        self.es = 8 if prec == "f64" else 4

    @property
    def ray_steps(self) -> int:
        return self.n * self.w.n_steps

    def step(self):
        w = self.w
        return self.rt.trace(self.eq, w.disp, self.x0, self.k0, self.omega, w.n_steps, w.dt, self.stride, traj=self.traj,
                             out=self.out)

    def parity_sample(self, n_sampled: int = 192) -> dict:
        """The launch state (the bytes the kernel read), final state and status of `n_sampled` rays of the LAST timed step --
        first / last rays, a warp boundary and seeded draws, as tests/test_gpu_parity.py samples them -- copied to the host for
        `sampled_parity` (which runs after every GPU measurement is done: the oracle is never called inside a timed region)."""
        torch = self.torch
        rng = np.random.default_rng(4242 + self.cfg)
        n = self.n
        idx = np.unique(np.concatenate([np.arange(min(8, n)), np.arange(max(0, n - 8), n), np.array([127, 128, 129]) % n,
                                        rng.integers(0, n, n_sampled - 19)]))
        d = torch.from_numpy(idx).cuda()
        host = lambda t: t.cpu().numpy().astype(np.float64)
        return {"kind": "rays", "cfg": self.cfg, "x0": host(self.x0[:, d]), "k0": host(self.k0[:, d]),
                "omega": host(self.omega[d]) if torch.is_tensor(self.omega) else self.omega,
                "final": host(self.out["final"][:, d]), "status": self.out["status"][d].cpu().numpy()}

    def host_buffers(self):
        torch, w = self.torch, self.w
        x0h, k0h = self.x0.cpu().pin_memory(), self.k0.cpu().pin_memory()
        n, dt = self.n, self.x0.dtype
        n_saved = w.n_steps // self.stride + 1
        out = {"final": torch.empty((6, n), dtype=dt, pin_memory=True),
               "residual": torch.empty((n_saved, n) if self.traj else (n,), dtype=dt, pin_memory=True),
               "status": torch.empty((n,), dtype=torch.int32, pin_memory=True)}
        if self.traj:
            out["traj"] = torch.empty((n_saved, 6, n), dtype=dt, pin_memory=True)
        h2d = x0h.numel() * self.es + k0h.numel() * self.es
        d2h = sum(t.numel() * t.element_size() for t in out.values())
        return x0h, k0h, out, h2d, d2h

    def step_host(self, x0h, k0h, out):
        w = self.w
        return self.rt.trace_host(self.eq, w.disp, x0h, k0h, w.omega, w.n_steps, w.dt, self.stride, traj=self.traj, out=out)

    def close(self):
        self.out = {}
        self.eq.close()


class OrbitJob:
    """The second ensemble workload: rt_orbit on inputs.orbit_config(4), 2^20 particles x 1000 steps,
    trajectories every 10 steps.  Same interface as Job as far as time_steps needs it."""

    def __init__(self, rt, torch, prec: str):
        self.rt, self.torch, self.prec = rt, torch, prec
        self.w = w = inputs.orbit_config(4)
        self.eq = rt.create_equilibrium(w.eq)
        dt = torch.float64 if prec == "f64" else torch.float32
        self.x0 = torch.from_numpy(w.x0).to(dt).cuda().contiguous()
        self.v0 = torch.from_numpy(w.v0).to(dt).cuda().contiguous()
        self.out = {}

    @property
    def ray_steps(self) -> int:
        return self.w.n * self.w.n_steps

    def step(self):
        w = self.w
        return self.rt.orbit(self.eq, self.x0, self.v0, w.charge_over_mass, w.n_steps, w.dt, w.save_stride, traj=True,
                             out=self.out)

    def parity_sample(self, n_sampled: int = 192) -> dict:
        torch, n = self.torch, self.w.n
        idx = np.unique(np.concatenate([np.arange(8), np.arange(n - 8, n), [127, 128, 129],
                                        np.random.default_rng(4242).integers(0, n, n_sampled - 19)]))
        d = torch.from_numpy(idx).cuda()
        host = lambda t: t.cpu().numpy().astype(np.float64)
        return {"kind": "orbits", "x0": host(self.x0[:, d]), "k0": host(self.v0[:, d]), "final": host(self.out["final"][:, d]),
                "status": self.out["status"][d].cpu().numpy()}

    def close(self):
        self.out = {}
        self.eq.close()


def sampled_parity(sample: dict) -> dict:
    """the sampled rays of one timed launch against the CPU oracle, from the very launch states the
    kernel read (fp32 runs: the fp32-rounded ones).  Errors are per-ray 2-norms relative to the oracle's (reading A15),
    maxima over the rays that end active on both sides; a ray whose status differs is counted, not measured."""
    import oracle
    oracle.build()
    if sample["kind"] == "orbits":
        w = inputs.orbit_config(4, n=8)
        ref = oracle.orbit(oracle.Equilibrium(w.eq), sample["x0"], sample["k0"], w.charge_over_mass, w.n_steps, w.dt)
    else:
        w = inputs.config(sample["cfg"], n_rays=8)
        ref = oracle.trace(oracle.Equilibrium(w.eq), w.disp, sample["x0"], sample["k0"], sample["omega"], w.n_steps, w.dt)
    got, same = sample["final"], sample["status"] == ref["status"]
    ok = same & (ref["status"] == 0)
    rel = lambda a, b: float((np.linalg.norm(a - b, axis=0) / np.linalg.norm(b, axis=0)).max()) if a.shape[1] else 0.0
    second = "max_rel_err_v" if sample["kind"] == "orbits" else "max_rel_err_k"
    return {"max_rel_err_x": rel(got[:3, ok], ref["final"][:3, ok]), second: rel(got[3:, ok], ref["final"][3:, ok]),
            "status_mismatches": int((~same).sum()), "n_sampled": int(same.size), "n_compared": int(ok.sum())}


def time_steps(torch, job: Job, steps: int, warmup: int, flush, barrier=None):
    """W warm-up steps, then exactly K steps bracketed by barrier + synchronize; L2 is flushed between steps by
    overwriting a buffer larger than L2.  Returns (total ms over the bracket, mean kernel ms from per-step events)."""
    for _ in range(warmup):
        job.step()
        flush.zero_()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for a, b in ev:
        a.record()
        job.step()
        b.record()
        flush.zero_()
    t1.record()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    return t0.elapsed_time(t1), statistics.fmean(a.elapsed_time(b) for a, b in ev)


def fractions(counts: dict, units: float, kernel_ms: float, fma_rate: float, flavour: str) -> dict:
    """The fractions of DESIGN.md section 6 for one kernel launch of `units` ray-steps (particle-steps);
    flavour = 'f64' | 'f32' | 'f32x2' selects the cost of a three-register instruction.
    roofline_frac  algorithmic flops (a division or square root = 1) against 2 x the FMA rate -- the strict figure;
    frac_executed  flops as executed against the same peak (SURVEY.md section 8(d)'s formula; what ncu's counters give);
    frac_ceiling   the largest roofline_frac THIS instruction stream allows: flops / (2 x pipe slots), a multiply or add
                   filling half of its slot, a three-register instruction taking a slot and a half;
    pipe_frac, pipe_model_frac  pipe slots issued (plain / with the three-register cost) against the FMA rate."""
    per_s = units / (kernel_ms * 1e-3)
    slots = counts["instr"] + RF3_EXTRA[flavour] * counts["rf3"]
    return {"roofline_frac": counts["flops"] * per_s / (2.0 * fma_rate),
            "frac_executed": counts["executed"] * per_s / (2.0 * fma_rate), "frac_ceiling": counts["flops"] / (2.0 * slots),
            "pipe_frac": counts["instr"] * per_s / fma_rate, "pipe_model_frac": slots * per_s / fma_rate}


def kernel_resources(kernel: str) -> dict:
    """Registers and spill bytes of one kernel instantiation, parsed from the ptxas report the build writes beside the
    library (librt_b200.ptxas.txt); `kernel` is the mangled-name prefix.  SURVEY 8(d) item (4)."""
    import re
    from paper_2508_15967_b200 import build as rt_build
    try:
        text = (rt_build.LIB.parent / "librt_b200.ptxas.txt").read_text()
    except OSError:
        return {"registers": None, "spill_bytes": None}
    m = re.search(r"Function properties for " + re.escape(kernel) + r"\w*\n\s*(\d+) bytes stack frame, (\d+) bytes spill stores, "
                  r"(\d+) bytes spill loads\nptxas info\s*: Used (\d+) registers", text)
    if not m:
        return {"registers": None, "spill_bytes": None}
    return {"registers": int(m.group(4)), "spill_bytes": int(m.group(2)) + int(m.group(3)), "stack_bytes": int(m.group(1))}


def trace_kernel_symbol(cfg: int, prec: str, scan: bool = False) -> str:
    """Mangled-name prefix of the kernel rt_trace / rt_trace_w launches for a config (rt_api.cu: launch_trace)."""
    e, d = KERNEL_OF_CONFIG[cfg]
    if (cfg, prec) in PACKED and not scan:
        return f"_ZN2rt15trace_kernel_x2ILi{e}ELi{d}EEE"
    return f"_ZN2rt12trace_kernelI{'d' if prec == 'f64' else 'f'}Li{e}ELi{d}ELb{int(scan)}ELb0EEE"


def flavour(cfg: int, prec: str) -> str:
    return "f32x2" if (cfg, prec) in PACKED else prec


def rank_plan(scaling: str, cfg: int, n_rays: int, rank: int, world: int):
    """What rank `rank` of `world` traces: (seed of the ensemble it draws, (begin, end) ray range of it, or None = all).
    strong: ONE seeded ensemble, contiguous ranges; weak: every rank its own full-size batch."""
    from paper_2508_15967_b200 import sharding
    if scaling == "strong":
        return 1000 + cfg, sharding.ray_range(n_rays, rank, world)
    return sharding.rank_seed(1000 + cfg, rank), None


def run_ours(args) -> int:
    import torch
    if not torch.cuda.is_available():
        print("bench.py: no CUDA device -- the product has no CPU fallback", file=sys.stderr)
        return 2
    from paper_2508_15967_b200 import binding as rt
    from paper_2508_15967_b200 import build as rt_build
    from paper_2508_15967_b200 import sharding
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if rank == 0:
        rt_build.build()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    rt.load()
    barrier = (lambda: dist.barrier()) if dist else None
    cfg, prec = args.config, args.precision
    n_rays = args.n_rays if args.n_rays else inputs.FULL_SIZES[cfg][0]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB of L2
    seed, span = rank_plan(args.scaling, cfg, n_rays, rank, world)
    job = Job(rt, torch, cfg, prec, n_rays, seed, ray_range=span)

    peak_before, _ = rt.fma_peak(prec, 200.0)
    sampler = ClockSampler(local)
    launches0 = rt.launch_count()
    sampler.start()
    total_ms, kernel_ms = time_steps(torch, job, args.steps, args.warmup, flush, barrier)
    clocks = sampler.stop()
    launches = rt.launch_count() - launches0 - args.warmup
    peak_after, peak_mhz = rt.fma_peak(prec, 200.0)

    want_oracle = rank == 0 and world == 1 and not args.no_cpu_baseline
    headline_sample = job.parity_sample() if want_oracle else None
    # a reduction over the last step's outputs: the run's own correctness summary (max |D|, status counts)
    red = rt.reduce(job.out["residual"].reshape(-1)).cpu().tolist()[:3] + rt.reduce(None, job.out["status"]).cpu().tolist()[3:]

    total_ms_max = sharding.max_over_ranks(total_ms, dist, "cuda")
    all_ray_steps = sharding.sum_over_ranks(float(job.ray_steps), dist, "cuda")
    value = all_ray_steps * args.steps / (total_ms_max * 1e-3)

    e2e = None
    if not args.no_e2e:
        x0h, k0h, hout, h2d, d2h = job.host_buffers()
        job.step_host(x0h, k0h, hout)                                       # warm-up (allocates the pipeline workspace)
        k_e2e = max(1, args.steps)
        torch.cuda.synchronize()
        if barrier:
            barrier()
        w0 = time.perf_counter()
        for _ in range(k_e2e):
            job.step_host(x0h, k0h, hout)
        torch.cuda.synchronize()
        t_e2e = sharding.max_over_ranks(time.perf_counter() - w0, dist, "cuda")
        e2e = {"value": all_ray_steps * k_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": k_e2e, "ms_per_step": 1e3 * t_e2e / k_e2e,
               "pcie_gb_per_s": (h2d + d2h) * k_e2e / t_e2e / 1e9,       # both directions, copies overlapped with the kernel
               "api": "rt_trace_host (pinned host buffers, 2-stream chunk pipeline)"}
        del x0h, k0h, hout

    counts = {"flops": FLOPS_PER_RAY_STEP[(cfg, prec)], "instr": FP_INSTR_PER_RAY_STEP[(cfg, prec)],
              "rf3": FP_RF3_PER_RAY_STEP[(cfg, prec)], "executed": FLOPS_EXECUTED_PER_RAY_STEP[(cfg, prec)]}
    fr = fractions(counts, job.ray_steps, kernel_ms, peak_after, flavour(cfg, prec))
    launch_residual = job.launch_residual
    peak = 2.0 * peak_after
    roofline = {"bound": "alu", "achieved": fr["roofline_frac"] * peak / 1e12, "peak": peak / 1e12, "unit": "TFLOP/s",
                "frac": fr["roofline_frac"], "traffic": NCU_DRAM_BYTES.get((cfg, prec)),
                "kernel": "rt::trace_kernel_x2 (packed f32x2, two rays per thread)" if (cfg, prec) in PACKED
                else f"rt::trace_kernel<{'double' if prec == 'f64' else 'float'}>",
                "kernel_ms": kernel_ms, "flops_per_ray_step": counts["flops"], "fp_instr_per_ray_step": counts["instr"],
                "fp_rf3_per_ray_step": counts["rf3"], "flops_executed_per_ray_step": counts["executed"],
                "frac_executed": fr["frac_executed"], "frac_ceiling": fr["frac_ceiling"],
                "pipe_frac": fr["pipe_frac"], "pipe_model_frac": fr["pipe_model_frac"],
                "peak_source": f"rt_fma_peak({prec}) measured in this process after the timed region: "
                               f"{peak_after / 1e12:.3f} T{'D' if prec == 'f64' else 'F'}FMA/s at {peak_mhz:.0f} MHz "
                               f"(before: {peak_before / 1e12:.3f})"}
    extra = None
    if rank == 0 and world == 1 and not args.no_extra and not args.n_rays:
        job.close()
        del job
        torch.cuda.empty_cache()
        extra, samples = [], []
        # the last tuple entry: a divisor of the config's ray count -- the per-rank size of a strong-scaling run over that many
        # GPUs, timed on this one GPU (rays never communicate, so this IS the per-rank time)
        table = [(1, "f64", False, 1), (1, "f32", False, 1), (2, "f64", False, 1), (2, "f32", False, 1), (3, "f64", False, 1),
                 (3, "f32", False, 1), (4, "f32", False, 1), (5, "f64", False, 1), (5, "f32", False, 1), (4, "f64", True, 1), (4, "f32", True, 1)]
        table += [(c, "f64", False, d) for c in (4, 5) for d in (2, 4, 8)]
        for c, p, scan, div in table:
            if (c, p) == (cfg, prec) and not scan and div == 1:
                continue
            j = Job(rt, torch, c, p, inputs.FULL_SIZES[c][0] // div, 1000 + c, scan=scan)
            _, kms = time_steps(torch, j, 3, 1, flush)
            pk, _ = rt.fma_peak(p, 100.0)
            cn = {"flops": FLOPS_PER_RAY_STEP[(c, p)], "instr": FP_INSTR_PER_RAY_STEP[(c, p)], "rf3": FP_RF3_PER_RAY_STEP[(c, p)],
                  "executed": FLOPS_EXECUTED_PER_RAY_STEP[(c, p)]}
            name = f"cfg{c}" + (" with one frequency per ray (rt_trace_w, w_i = w0 (1 +- 10 %))" if scan else "")
            if div > 1:
                name += f" at n_rays / {div} = {j.n} rays (the per-rank size of a {div}-GPU strong-scaling run, on one GPU)"
            if c == 1:
                name += " -- 1024 rays = 16 blocks on 148 SMs: latency-bound, the fractions say how empty the chip is"
            extra.append({"workload": name, "dtype": p, "n_rays": j.n, "value": j.ray_steps / (kms * 1e-3), "unit": UNIT,
                          "kernel_ms": kms, "traffic": NCU_DRAM_BYTES.get((c, p)) if not scan and div == 1 else None,
                          **kernel_resources(trace_kernel_symbol(c, p, scan)),
                          **fractions(cn, j.ray_steps, kms, pk, flavour(c, p) if not scan else p)})
            samples.append(j.parity_sample() if want_oracle and div == 1 else None)
            j.close()
            del j
            torch.cuda.empty_cache()
        for p in ("f64", "f32"):      # the second ensemble workload: full orbits, rt_orbit
            j = OrbitJob(rt, torch, p)
            _, kms = time_steps(torch, j, 3, 1, flush)
            pk, _ = rt.fma_peak(p, 100.0)
            extra.append({"workload": "orbits: 10 keV deuterons in config 4's tokamak, 2^20 particles x 1000 steps, trajectory "
                                      "every 10 steps + energy drift (rt_orbit)", "dtype": p,
                          "value": j.ray_steps / (kms * 1e-3), "unit": "particle-steps/s", "kernel_ms": kms,
                          "kernel": "rt::orbit_kernel", "traffic": NCU_DRAM_BYTES.get(("orbit4", p)),
                          **kernel_resources(f"_ZN2rt12orbit_kernelI{'d' if p == 'f64' else 'f'}Li2EEE"),
                          **fractions(ORBIT_COUNTS[p], j.ray_steps, kms, pk, p)})
            samples.append(j.parity_sample() if want_oracle else None)
            j.close()
            del j
            torch.cuda.empty_cache()

    # every GPU measurement is done: now the oracle legs (the only place this arm calls oracle/)
    cpu, parity = None, None
    if want_oracle:
        cpu = cpu_baseline(cfg)
        parity = sampled_parity(headline_sample)
        if extra:
            per_cfg = {}                   # the oracle timed on a ~3 s sample of each other config too, all cores
            for row, smp in zip(extra, samples):
                if smp is None:
                    continue
                row["parity"] = sampled_parity(smp)
                if smp["kind"] == "rays":
                    c = smp["cfg"]
                    if c not in per_cfg:
                        per_cfg[c] = cpu_baseline(c, target_s=3.0, single_thread_s=0.0)
                    row["cpu_baseline"] = per_cfg[c]

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": total_ms_max / args.steps, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
                "dtype": prec, "data": "synthetic", "config": workload_config(cfg, args.scaling),
                "run": {"launch_states": "rt_launch kernel, max |D0| = %.1e" % launch_residual,
                        "rays_this_rank": n_rays if args.scaling == "weak" else list(sharding.ray_range(n_rays, rank, world))},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
                "roofline": {**roofline, **kernel_resources(trace_kernel_symbol(cfg, prec))},
                "checks": {"max_abs_D": red[0], "mean_abs_D": red[1] / max(red[2], 1.0), "status_counts": red[3:6],
                           "parity": parity},
                "cpu_baseline": cpu, "other_configs": extra}
        print(json.dumps(line))
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main() -> int:
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
