"""Count the floating-point work of one ray-step (particle-step) in the compiled ``trace_kernel`` and ``orbit_kernel``
instantiations (``cuobjdump -sass``).

    python tests/sass_count.py            # table for every trace kernel in librt_b200.so

A ray-step is one pass through the body of the kernel's step loop (the loops that hold FP-pipe instructions are nested:
sample loop > step loop, and for the grid equilibrium > the rolled stage loop, which runs 4 times per step).
Reported per kernel:

* ``instr``     FP-pipe instructions per ray-step (DFMA + DMUL + DADD + DSETP, or the FP32 analogues) -- what the FP64
                (FP32) pipe has to issue, the quantity the kernels are optimised for;
* ``rf3``       how many of them read THREE DISTINCT registers from the register file (constants, immediates, RZ and operands
                served by the operand-reuse cache -- flagged ``.reuse`` in the same slot of the preceding instruction --
                do not count).  Such an instruction occupies the FP64 pipe for 3 cycles instead of 2 (FP32: 1.56
                instead of 1; ``rt_fma_peak_shape`` shape 2, profiles/r2_fma_peak_shapes.md), so the pipe time of a
                ray-step is 2 instr + rf3 cycles per warp and scheduler;
* ``executed``  flops as executed, a fused multiply-add counted as 2;
* ``mufu``      MUFU seeds (reciprocals and reciprocal square roots), ``rsqrt`` of them square roots;
* f32, analytic equilibria: the kernels that run are ``trace_kernel_x2`` (two rays per thread, packed f32x2 arithmetic).
                Their loop body advances two rays; the counts are reported PER RAY: a packed FFMA2 / FMUL2 / FADD2 is one
                pipe slot per ray (it occupies the FMA pipe for two cycles and does the operation for both rays), a scalar
                FP instruction or MUFU seed (they serve ONE of the two rays: per-half domain tests, and the per-ray spline
                look-ups of the grid equilibrium's packed kernel) half a slot; likewise for ``rf3``.  ``rf3`` counts packed instructions with three distinct register
                operands: 3 pipe cycles instead of 2 (84.9 against 127.9 FMA per clock per SM, ``rt_fma_peak_shape`` shapes 6 / 5);
* ``local``     local-memory (spill) instructions executed per ray-step: must be 0.  ptxas may still report a few bytes
                of spill for values parked once before the step loop and reloaded after it (the store staging);
* ``flops``     the ALGORITHMIC flops bench.py uses for ``roofline.achieved``: every division and square root counted as
                ONE flop.  In fp64 a reciprocal executes 3 FMAs (6 flops) and a reciprocal square root 2 MUL + 3 FMA
                (8 flops) of Newton refinement after the seed, so flops = executed - 5 rcp - 7 rsqrt; in fp32 the seed
                is used as is, so flops = executed + mufu.  The two precisions agree on this figure to within 1 %.

This is a measuring tool; nothing in the product path imports it.  ``tests/test_abi.py`` checks
bench.py's ``FLOPS_PER_RAY_STEP`` table against it, so the table cannot go stale when the kernels change.
"""
from __future__ import annotations

import re
import shutil
import subprocess
from collections import Counter
from pathlib import Path

LIB = Path(__file__).resolve().parent.parent / "paper_2508_15967_b200" / "librt_b200.so"
_INS = re.compile(r"\s+/\*([0-9a-f]+)\*/\s+(?:@!?U?P\w+\s+)?([A-Z0-9_.]+)(.*?);")
_FP = {"d": ("DFMA", "DMUL", "DADD", "DSETP"), "f": ("FFMA", "FMUL", "FADD", "FSETP")}
_FP2 = ("FFMA2", "FMUL2", "FADD2")       # packed f32x2: one instruction serves both rays of a thread


def cuobjdump() -> str | None:
    for cand in (shutil.which("cuobjdump"), "/usr/local/cuda/bin/cuobjdump"):
        if cand and Path(cand).exists():
            return cand
    return None


def _parse(body: str):
    out = []
    for line in body.splitlines():
        m = _INS.match(line)
        if m:
            out.append((int(m.group(1), 16), m.group(2), m.group(3)))
    return out


def _target(rest: str):
    m = re.search(r"0x([0-9a-f]+)", rest)
    return int(m.group(1), 16) if m else None


def _count(ins, lo, hi):
    return Counter(op.split(".")[0] for a, op, _ in ins if lo <= a < hi), \
        sum(1 for a, op, _ in ins if lo <= a < hi and op.startswith("MUFU.RSQ"))


_REG = re.compile(r"[-|~]*R(\d+)")


def _rf3(ins, lo, hi, fp_ops):
    """FP-pipe instructions in [lo, hi) whose three source operands are all read from the register file."""
    n3, reuse = 0, {}
    for a, op, rest in ins:
        if not (lo <= a < hi):
            continue
        ops = [o.strip() for o in rest.split(",")]
        base = op.split(".")[0]
        srcs = ops[2:] if base.endswith("SETP") else ops[1:]
        if base in fp_ops:
            regs = set()                                    # distinct registers read from the register file: the same
            for slot, o in enumerate(srcs):                 # register in two slots is read once (measured: fma(b, b, acc)
                m = _REG.match(o)                           # runs at the full rate)
                if m and reuse.get(slot) != m.group(1):
                    regs.add(m.group(1))
            n3 += len(regs) >= 3
        reuse = {}
        for slot, o in enumerate(ops[1:]):
            m = _REG.match(o)
            if m and ".reuse" in o:
                reuse[slot] = m.group(1)
    return n3


def _step_region(ins, fp_ops):
    """(step loop, stage loop or None) of a trace / orbit kernel as address ranges [lo, hi).

    Loop nest of the kernel = its backward branches.  The loops that hold FP-pipe instructions: the sample loop, inside it
    the step loop -- for the magnetised dispersion functions TWO step loops side by side, the hot one (ion terms by their
    series, rt_math.cuh: disp_coefs) and the rarely entered exact one, which holds more FP instructions -- and, when the
    stages are rolled (grid equilibrium), a stage loop inside each step loop.  The small loops of the store staging and of
    the cell-cache refill hold no FP instruction and are ignored.  Returned: the step loop with the fewest FP instructions
    (the hot one)."""
    loops = set()
    for a, op, rest in ins:
        if op.startswith("BRA"):
            t = _target(rest)
            if t is not None and t < a:
                loops.add((t, a + 16))
    nfp = {l: sum(1 for b, o, _ in ins if l[0] <= b < l[1] and o.split(".")[0] in fp_ops) for l in loops}
    fpl = sorted((l for l in loops if nfp[l] > 0), key=lambda l: l[0] - l[1])            # largest first
    if not fpl:
        return None
    inside = lambda a, b: b[0] <= a[0] and a[1] <= b[1] and a != b
    outer = fpl[0]
    if len(fpl) == 1:
        return outer, None                                   # no sample loop distinguishable: the one loop is the step loop
    assert all(inside(l, outer) for l in fpl[1:]), "FP loops outside the sample loop"
    steps = [l for l in fpl[1:] if not any(inside(l, m) for m in fpl[1:])]               # maximal loops inside the sample loop
    nmufu = lambda l: sum(1 for b, o, _ in ins if l[0] <= b < l[1] and o.startswith("MUFU"))
    step = min(steps, key=lambda l: (nfp[l] + nmufu(l), l[0]))        # fp32: the series saves a MUFU seed, not an FP instruction
    stages = [l for l in fpl[1:] if inside(l, step)]
    assert len(stages) <= 1, "more than one FP loop inside the step loop"
    return step, (stages[0] if stages else None)


def count_kernels(lib: Path = LIB) -> dict:
    """{(precision 'f64'|'f32', eq_kind, disp_kind | 'orbit'): {'instr', 'rf3', 'executed', 'mufu', 'rsqrt', 'flops',
    'local'}} per ray-step (particle-step for the orbit kernels)."""
    exe = cuobjdump()
    if exe is None:
        raise RuntimeError("cuobjdump not found")
    sass = subprocess.run([exe, "-sass", str(lib)], capture_output=True, text=True, check=True).stdout
    res = {}
    for fn in re.split(r"\n\s*Function : ", sass):
        m = re.match(r"_ZN2rt12trace_kernelI([df])Li(\d)ELi(\d)ELb0ELb0E", fn)      # the plain single-frequency kernels
        mo = re.match(r"_ZN2rt12orbit_kernelI([df])Li(\d)EE", fn)                   # the second workload (rt_orbit)
        m2 = re.match(r"_ZN2rt15trace_kernel_x2ILi(\d)ELi(\d)EE", fn)              # fp32, two rays per thread (packed)
        if not m and not mo and not m2:
            continue
        packed = bool(m2)
        if m:
            prec, eq, disp = m.group(1), int(m.group(2)), int(m.group(3))
        elif mo:
            prec, eq, disp = mo.group(1), int(mo.group(2)), "orbit"
        else:
            prec, eq, disp = "f", int(m2.group(1)), int(m2.group(2))
        ins = _parse(fn)
        fp_ops = _FP[prec] + (_FP2 if packed else ())
        sel = _step_region(ins, fp_ops)
        if sel is None:
            continue
        region, stage = sel
        rolled = stage is not None
        c, rsq = _count(ins, *region)
        tot = Counter(c)

        def rf3_of(ops):                                    # the stage loop (rolled stages) runs 4 times per step
            return _rf3(ins, *region, ops) + (3 * _rf3(ins, *stage, ops) if rolled else 0)
        rf3 = rf3_of(fp_ops)
        if rolled:
            ci, rsqi = _count(ins, *stage)
            for k, v in ci.items():
                tot[k] += 3 * v
            rsq += 3 * rsqi
        fma, mul, add, setp = _FP[prec]
        local = tot["STL"] + tot["LDL"]                     # spill traffic executed per ray-step (must be 0)
        if packed:
            # the loop body advances TWO rays: a packed instruction is one pipe slot per ray; a scalar FP instruction
            # (per-half domain tests, |x|) and a MUFU seed serve one ray each, i.e. half a slot per ray
            n2 = tot["FFMA2"] + tot["FMUL2"] + tot["FADD2"]
            n1 = tot[fma] + tot[mul] + tot[add] + tot[setp]
            executed = 2 * tot["FFMA2"] + tot["FMUL2"] + tot["FADD2"] + (2 * tot[fma] + tot[mul] + tot[add] + 1) // 2
            mufu, rsq = tot["MUFU"] // 2, rsq // 2
            res[("f32", eq, disp)] = dict(instr=n2 + (n1 + 1) // 2, executed=executed, mufu=mufu, rsqrt=rsq,
                                          flops=executed + mufu, local=local,
                                          rf3=rf3_of(_FP2) + (rf3_of(_FP[prec]) + 1) // 2, packed=True)
            continue
        executed = 2 * tot[fma] + tot[mul] + tot[add]
        mufu = tot["MUFU"]
        flops = executed - 5 * (mufu - rsq) - 7 * rsq if prec == "d" else executed + mufu
        res[("f64" if prec == "d" else "f32", eq, disp)] = dict(instr=tot[fma] + tot[mul] + tot[add] + tot[setp],
                                                                executed=executed, mufu=mufu, rsqrt=rsq, flops=flops,
                                                                local=local, rf3=rf3, packed=False)
    return res


if __name__ == "__main__":
    names = {0: "parabolic", 1: "linear", 2: "tokamak", 3: "grid", 4: "tokamak_pow"}
    disps = {0: "O", 1: "X", 2: "full"}
    print("(f32 analytic rows: trace_kernel_x2, two rays per thread, packed FFMA2 / FMUL2 / FADD2; counts are per ray)")
    print(f"{'kernel':34s} {'instr':>6s} {'rf3':>5s} {'executed':>9s} {'mufu':>5s} {'rsqrt':>6s} {'flops':>6s} {'local':>6s}")
    for (prec, eq, disp), r in sorted(count_kernels().items(), key=lambda kv: (kv[0][2] == "orbit", kv[0][0], kv[0][1], str(kv[0][2]))):
        name = f"orbit_kernel<{prec}, {names[eq]:11s}>      " if disp == "orbit" else f"trace_kernel<{prec}, {names[eq]:11s}, {disps[disp]:4s}>"
        print(f"{name} {r['instr']:6d} {r['rf3']:5d} {r['executed']:9d} {r['mufu']:5d} "
              f"{r['rsqrt']:6d} {r['flops']:6d} {r['local']:6d}")
