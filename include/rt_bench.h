/* rt_bench.h -- measurement entry points of librt_b200.so (NOT part of the ray-tracing interface of rt.h).
 *
 * bench.py reports the hot path against a roofline whose denominator is measured in the same process ("a
 * microbenchmark of >= 8 independent dependent-chain DFMA (resp. FFMA) accumulators per thread ... reporting FMA/s and the
 * SM clock observed").  rt_fma_peak is that microbenchmark; rt_fma_peak_shape runs it at other instruction shapes and
 * occupancies, the evidence behind DESIGN.md section 6's operand-port model of the FP64 / FP32 pipe.  Both are
 * synchronous, allocate and free their own scratch, and use the current device.  rt_math_probe exposes the hot loop's
 * reciprocal / square-root routines to a unit test.  Return codes as in rt.h. */
#ifndef RT_B200_RT_BENCH_H
#define RT_B200_RT_BENCH_H

#include "rt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measured roofline denominator: run >= min_ms milliseconds of independent dependent-chain FMA accumulators (DFMA
 * for RT_F64, FFMA for RT_F32) on every SM and report the sustained rate.  Synchronous.
 *   fma_per_s     HOST out: fused multiply-adds per second (flop/s = 2x)
 *   sm_clock_mhz  HOST out: average SM clock over the run derived from clock64()/globaltimer; or NULL */
int rt_fma_peak(int precision, double min_ms, double* fma_per_s, double* sm_clock_mhz);

/* The same microbenchmark with its instruction shape and occupancy exposed (evidence for DESIGN.md section 6's
 * "practical ceiling of the pipe"; rt_fma_peak is shape 0 -- for RT_F32 shape 5 -- with 4 blocks per SM).
 *   shape          0: acc = acc * a + acc (two distinct source registers);  1: acc = acc * a + b, a and b shared by all
 *                  chains (three distinct sources, two of them served by the operand-reuse cache);  2: acc_j = acc_j *
 *                  a_j + b_j with per-chain a_j, b_j (every instruction reads three registers from the register file);
 *                  3: shape 0 plus 4 independent MUFU reciprocal seeds per 16 FMAs (the seeds are not counted);
 *                  4: shape 0 with one chain per thread (rate = warps per scheduler / dependent-issue latency);
 *                  fp32 only: 5 / 6 = shapes 0 / 2 issued as packed f32x2 instructions (FFMA2: two fused multiply-adds per
 *                  instruction and lane; rates are always reported in fused multiply-adds, not instructions).
 *                  rt_fma_peak(RT_F32) is shape 5, the best the FP32 FMA pipe delivers
 *   blocks_per_sm  1..8 blocks of 256 threads per SM, i.e. 2..16 warps per scheduler
 * Errors: RT_ERR_INVALID for an unknown precision / shape (5 and 6 exist for RT_F32 only) / blocks_per_sm outside [1, 8] / min_ms outside (0, 10000]
 * / fma_per_s NULL (all checked before the first CUDA call); RT_ERR_CUDA when no device is usable. */
int rt_fma_peak_shape(int precision, int shape, int blocks_per_sm, double min_ms, double* fma_per_s,
                      double* sm_clock_mhz);

/* Unit-test hook: the hot loop's own reciprocal, reciprocal square root and square root (a MUFU seed plus one Newton
 * step in fp64, the bare seed in fp32; csrc/rt_math.cuh) applied to an array, so that their rounding error can be measured
 * directly (tests/test_gpu_math.py; DESIGN.md section 7 has the bounds).  Asynchronous on `cuda_stream`, allocates nothing.
 *   fn   0: 1/x    1: 1/sqrt(x)    2: sqrt(x)
 *   x    DEVICE [n] of `precision`;   out  DEVICE [n] of `precision`
 * Errors: RT_ERR_INVALID (unknown precision / fn, n < 0, a NULL, misaligned or host pointer), RT_ERR_CUDA. */
int rt_math_probe(int precision, int fn, const void* x, int64_t n, void* out, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* RT_B200_RT_BENCH_H */
