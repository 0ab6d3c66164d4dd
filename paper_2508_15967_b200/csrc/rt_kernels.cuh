// rt_kernels.cuh -- the CUDA kernels of the hot path (sm_100a).
//
//   trace_kernel   one thread per ray; loads (x0, k0) once, runs all n_steps classical RK4 steps
//                  with the state, the stage slopes and every intermediate of D's gradient in registers, and writes
//                  decimated SoA trajectory samples / the final state / |D| / status (steps a1-a6 of DESIGN.md).
//   orbit_kernel   the second ensemble workload: full-orbit particles, same structure as trace_kernel.
//   rhs_kernel     one stage evaluation per point (diagnostics and gradient parity tests).
//   launch_kernel  launch conditions: closed-form |n| on D = 0 plus Newton polish.
//   launch_kx_kernel  the paper's own launch iteration: k_y, k_z fixed, Newton on k_x from an initial guess.
//   reduce_kernel  max / sum of |D| and status counts (PAPER.md L76 reduction kernels).
//   fma_peak_kernel  the roofline denominator: independent FMA chains.
#pragma once

#include <stdint.h>

#include <type_traits>

#include "rt_math.cuh"

namespace rt {

// Launch shapes.  The trace kernels are bound by the FP64 (FP32) pipe, not by memory and not by latency: 4 warps per
// scheduler saturate the FP64 pipe even without instruction-level parallelism (8-cycle dependent-issue latency, one
// instruction per 2 cycles), and every shape between 12 and 18 warps per SM runs within 0.3 % of the others as long as it
// does not spill (profiles/r1_tuning.md).  So the register cap (`__maxnreg__`) is simply the smallest one without spills
// inside the step, with 64-thread blocks so that the register file divides evenly:
//   fp64, analytic equilibria   120 registers -> 8 blocks = 16 warps per SM
//   fp64, linear slab, O / X     72 registers -> 14 blocks = 28 warps per SM (the stage is a short chain through three
//                                reciprocals: config 3 11.52 ms at 120 registers, 10.88 ms at 72; spills at 64)
//   fp64, grid equilibrium      128 registers -> 8 blocks = 16 warps per SM (the profile pieces live in 16 of them)
//   fp32, scalar kernels         72 registers -> 14 blocks = 28 warps per SM (the grid kernel's LDS latency likes warps:
//                                321 ms at 72 registers, 344 ms at 128); the packed fp32 kernels: TraceShape2 below
// The grid equilibrium keeps ONE copy of the stage code (stage loop not unrolled: unrolled it needs >= 168 registers and
// is slower at every cap, profiles/r1_tuning.md).  The diagnostic kernels (rhs, launch, diag) use plain 128-thread blocks.
constexpr int AUX_BLOCK = 128;
template <class T, int EQ> struct TraceShape { static constexpr int BLOCK = 64, MAXNREG = 72; };
template <int EQ> struct TraceShape<double, EQ> { static constexpr int BLOCK = 64, MAXNREG = 120; };
template <> struct TraceShape<double, EQ_GRID> { static constexpr int BLOCK = 64, MAXNREG = 128; };
// register cap of trace_kernel<T, EQ, DISP>: the class's, except for the short O- / X-mode stages over the linear slab
template <class T, int EQ, int DISP>
constexpr int trace_maxnreg() {
  return (sizeof(T) == 8 && EQ == EQ_LINEAR && DISP != DISP_FULL) ? 72 : TraceShape<T, EQ>::MAXNREG;
}

// extra registers of the per-ray-frequency (PW) kernels, which hold the frequency-dependent constants per thread: 16, and 24
// for the fp64 full determinant over the analytic equilibria (at 136 the tokamak instantiation spilled 8 bytes in its
// prologue; 144 registers are the same 7 blocks per SM)
template <class T, int EQ, int DISP>
constexpr int pw_extra_regs() {
  return (sizeof(T) == 8 && DISP == DISP_FULL && EQ != EQ_GRID) ? 24 : 16;
}

template <class T>
struct TraceArgs {
  const T* x0;
  const T* k0;
  T* traj;
  T* fin;
  T* res;
  int32_t* status;
  long long n_rays;     // rays in this launch == row pitch of every buffer
  long long n_steps;
  long long stride;
  T h;                  // step in tau = c t
  T hh, h3, h6;         // h/2, h/3, h/6: the tableau's step factors, folded on the host (constant bank operands)
  const double* omega;  // per-ray frequencies [n_rays] (PW kernels only), rad/s
  double omega_ref;     // the frequency the Params were folded at
  const int32_t* status_in;   // resume (rt_trace_until's chunks): each ray's status at entry, or NULL = every ray starts
                              // active.  May alias `status`; x0 / k0 may then alias the rows of `fin` (in-place chunk).
};

// One classical RK4 step (reading A7): stage abscissae (0, 1/2, 1/2, 1), weights (1, 2, 2, 1)/6, written so that every
// update is one fused multiply-add: acc = y + h/6 k1 + h/3 k2 + h/3 k3, y_new = acc + h/6 k4 (42 FMAs per step).
// Returns 0 accepted, 1 a stage point left the domain (step rejected), 2 the new state is not finite (rejected).
// The analytic equilibria run the four stages fully unrolled (the compiler schedules across stages); the grid
// equilibrium keeps ONE copy of the right-hand-side code (smaller instruction footprint and fewer live registers around
// the gathers).  Components of the right-hand side that are structurally zero (slabs: dn_y/dtau = dn_z/dtau = 0,
// parabolic: dn_z/dtau = 0) are skipped, which also keeps them bit-for-bit constant.
template <int EQ>
RT_DEV constexpr bool rhs_component_active(int j) {
  return !((EQ == EQ_LINEAR && j >= 4) || (EQ == EQ_PARABOLIC && j == 5));
}

// rk4_stages: the four stages of one step from y; writes the candidate new state to ys and returns whether every stage
// point was inside the domain (per lane for the packed fp32 kernels).  rk4_step applies the acceptance rule (A12).
// SERIES: the ion terms by their series (rt_math.cuh: disp_coefs); `fast` is cleared if a stage point lies outside the
// series' range (Y2 >= Params::y2cap), and the step then has to be repeated with SERIES = false.
template <class T, int EQ, int DISP, bool SERIES, class Gather>
RT_DEV typename Lane<T>::mask rk4_stages(const Params<T>& P, T h, T hh, T h3, T h6, const T* y, T* ys, Gather& gather,
                                         typename Lane<T>::mask& fast) {
  T k[6], acc[6], r;                 // the slope of a stage is r k (ray_rhs): r is folded into the step-size factors
  typename Lane<T>::mask ok = rt_true<T>();
  if (EQ == EQ_GRID) {
#pragma unroll
    for (int j = 0; j < 6; ++j) { k[j] = T(0); acc[j] = y[j]; }
    T ar = T(0);                     // a_st r_{st-1}
#pragma unroll 1
    for (int st = 0; st < 4; ++st) {
#pragma unroll
      for (int j = 0; j < 6; ++j) ys[j] = rt_fma(ar, k[j], y[j]);
      ok = rt_and(ray_rhs<T, EQ, DISP, SERIES>(P, ys, k, r, gather, fast), ok);
      const T wr = ((st == 0 || st == 3) ? h6 : h3) * r;
      ar = ((st == 2) ? h : hh) * r;
#pragma unroll
      for (int j = 0; j < 6; ++j) acc[j] = rt_fma(wr, k[j], acc[j]);
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) ys[j] = acc[j];
  } else {
#pragma unroll
    for (int j = 0; j < 6; ++j) { ys[j] = y[j]; acc[j] = y[j]; }
    ok = ray_rhs<T, EQ, DISP, SERIES>(P, y, k, r, gather, fast);
    T wr = h6 * r, ar = hh * r;
#pragma unroll
    for (int j = 0; j < 6; ++j)
      if (rhs_component_active<EQ>(j)) { acc[j] = rt_fma(wr, k[j], y[j]); ys[j] = rt_fma(ar, k[j], y[j]); }
    ok = rt_and(ray_rhs<T, EQ, DISP, SERIES>(P, ys, k, r, gather, fast), ok);
    wr = h3 * r; ar = hh * r;
#pragma unroll
    for (int j = 0; j < 6; ++j)
      if (rhs_component_active<EQ>(j)) { acc[j] = rt_fma(wr, k[j], acc[j]); ys[j] = rt_fma(ar, k[j], y[j]); }
    ok = rt_and(ray_rhs<T, EQ, DISP, SERIES>(P, ys, k, r, gather, fast), ok);
    wr = h3 * r; ar = h * r;
#pragma unroll
    for (int j = 0; j < 6; ++j)
      if (rhs_component_active<EQ>(j)) { acc[j] = rt_fma(wr, k[j], acc[j]); ys[j] = rt_fma(ar, k[j], y[j]); }
    ok = rt_and(ray_rhs<T, EQ, DISP, SERIES>(P, ys, k, r, gather, fast), ok);
    wr = h6 * r;
#pragma unroll
    for (int j = 0; j < 6; ++j) ys[j] = rhs_component_active<EQ>(j) ? rt_fma(wr, k[j], acc[j]) : y[j];
  }
  return ok;
}

// One step with the acceptance rule.  SERIES: returns -1, with y untouched, if a stage point lay outside the range of the ion
// terms' series; the caller then repeats this step (and finishes its stretch of steps) with SERIES = false.
template <class T, int EQ, int DISP, bool SERIES, class Gather>
RT_DEV int rk4_step(const Params<T>& P, T h, T hh, T h3, T h6, T* y, Gather& gather) {
  T ys[6];
  bool fast = true;
  const bool ok = rk4_stages<T, EQ, DISP, SERIES>(P, h, hh, h3, h6, y, ys, gather, fast);
  if (SERIES && DISP != DISP_O && !fast) return -1;
  if (!ok) return 1;
  bool fin = true;
#pragma unroll
  for (int j = 0; j < 6; ++j) fin = fin && rt_finite(ys[j]);
  if (!fin) return 2;
#pragma unroll
  for (int j = 0; j < 6; ++j) y[j] = ys[j];
  return 0;
}

template <class T, int EQ, int DISP, class Gather>
RT_DEV T abs_residual(const Params<T>& P, const T* y, Gather& gather) {
  typename Lane<T>::mask inside;
  const T D = ray_D<T, EQ, DISP>(P, y, &inside, gather);
  return rt_select(inside, rt_abs(D), rt_nan<T>());
}

#ifdef __CUDACC__

// Shared-memory cell cache of the grid equilibrium.  A ray moves ~1 mm per RK4 step through 5.9 mm cells, so the 16
// psi pieces (one 128-B line in fp64) and the 8 profile pieces it needs are the same for many consecutive stages.  Read
// straight from global memory, every 128-bit load of a warp touches 32 different lines and the L1 data pipe saturates
// (99.8 % `l1tex__data_pipe_lsu_wavefronts`, FP64 pipe 43 %: round-1 capture, profiles/README.md "history").  Here each thread keeps its
// current cell's pieces in its own column of a [chunk][thread] shared array -- 16-byte chunks, consecutive threads in
// consecutive chunks, so a warp's LDS.128 is 4 conflict-free wavefronts -- and refills the column from global memory
// only when its cell index changes.  The column is private to the thread: no barrier is needed.
template <class T> struct Vec16;
template <> struct Vec16<double> { typedef double2 type; };
template <> struct Vec16<float> { typedef float4 type; };
RT_DEV void unpack4(const double2* s, int row, int pitch, double* c) {
  const double2 a = s[(2 * row) * pitch], b = s[(2 * row + 1) * pitch];
  c[0] = a.x; c[1] = a.y; c[2] = b.x; c[3] = b.y;
}
RT_DEV void unpack4(const float4* s, int row, int pitch, float* c) {
  const float4 a = s[row * pitch];
  c[0] = a.x; c[1] = a.y; c[2] = a.z; c[3] = a.w;
}

// ASYNC_PROF: the profile pieces' refill as cp.async too (worth it only where other work separates request and wait)
template <class T, int BLOCK, bool ASYNC_PROF = false>
struct GatherCached {
  typedef typename Vec16<T>::type V;
  // fp64: the 8 pieces of the two 1-D profiles stay in REGISTERS while the psi-cell is unchanged (about ten stages), so a
  // stage reads only the 16 psi pieces from shared memory (8 instead of 12 LDS.128: config 5 fp64 543 -> 535 ms).  fp32:
  // they stay in shared memory -- the fp32 kernel is issue-bound and the register copies cost more than the two LDS.128
  // they replace (289 -> 301 ms, profiles/r2_tuning.md).
  static constexpr bool PROF_REGS = sizeof(T) == 8;
  static constexpr int PSI_CHUNKS = 16 * sizeof(T) / 16, PROF_CHUNKS = PROF_REGS ? 0 : 8 * sizeof(T) / 16;
  static constexpr int CHUNKS = PSI_CHUNKS + PROF_CHUNKS;
  V* col;                  // this thread's column: chunk j at col[j * BLOCK]
  int cell, pcell;         // cached cell indices (-1: nothing cached)
  T prof[PROF_REGS ? 8 : 1];
  // refill: global -> shared directly (cp.async, 16 bytes per chunk), no staging through registers and no separate STS;
  // wait() before the column is read.  A thread's copies all land in its own column: no barrier is needed.
  // (both requests return whether a copy was issued that wait() has to cover)
  RT_DEV bool psi_request(const Params<T>& P, int c) {
    if (c != cell) {
      const V* g = reinterpret_cast<const V*>(P.psi_pp + (size_t)c * 16);
      const unsigned dst = (unsigned)__cvta_generic_to_shared(col);
#pragma unroll
      for (int j = 0; j < PSI_CHUNKS; ++j)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + (unsigned)(j * BLOCK * sizeof(V))), "l"(g + j) : "memory");
      cell = c;
      return true;
    }
    return false;
  }
  RT_DEV bool prof_request(const Params<T>& P, int c) {
    if (c != pcell) {
      if (PROF_REGS) {
        ld4(P.prof_pp + (size_t)c * 8, prof);
        ld4(P.prof_pp + (size_t)c * 8 + 4, prof + 4);
      } else if (ASYNC_PROF) {
        const V* g = reinterpret_cast<const V*>(P.prof_pp + (size_t)c * 8);
        const unsigned dst = (unsigned)__cvta_generic_to_shared(col + PSI_CHUNKS * BLOCK);
#pragma unroll
        for (int j = 0; j < PROF_CHUNKS; ++j)
          asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + (unsigned)(j * BLOCK * sizeof(V))), "l"(g + j) : "memory");
      } else {           // scalar fp32 kernels: load + store (the wait follows at once; cp.async here: 282 -> 305 ms)
        const V* g = reinterpret_cast<const V*>(P.prof_pp + (size_t)c * 8);
#pragma unroll
        for (int j = 0; j < PROF_CHUNKS; ++j) col[(PSI_CHUNKS + j) * BLOCK] = __ldg(g + j);
      }
      pcell = c;
      return !PROF_REGS && ASYNC_PROF;
    }
    return false;
  }
  RT_DEV void wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }
  RT_DEV void psi_row(const Params<T>&, int, int p, T* c) const { unpack4(col, p, BLOCK, c); }
  RT_DEV void prof_row(const Params<T>&, int, int which, T* c) const {
    if (PROF_REGS) {
#pragma unroll
      for (int j = 0; j < 4; ++j) c[j] = prof[4 * which + j];
    } else {
      unpack4(col + PSI_CHUNKS * BLOCK, which, BLOCK, c);
    }
  }
};

// the packed fp32 kernel of the grid equilibrium: one scalar cell cache per ray of the thread (rt_math.cuh: grid_values_per_ray)
template <int BLOCK> struct GatherPair { GatherCached<float, BLOCK, true> a, b; };
template <int BLOCK> struct gather_is_pair<GatherPair<BLOCK>> { static constexpr bool value = true; };

template <class T, int EQ> struct TraceGather { typedef GatherDirect type; };
template <class T> struct TraceGather<T, EQ_GRID> { typedef GatherCached<T, TraceShape<T, EQ_GRID>::BLOCK> type; };

// Per-ray frequency (w is a per-ray kernel input).  The per-call constants are folded at
// the reference frequency w_ref; a ray with its own w sees X and Y^2 scaled by lam^2 and n = c k/w by lam, lam = w_ref/w.
// The thread-local copy below overrides exactly the w-dependent fields; everything else stays in the constant bank.
template <class T>
RT_DEV Params<T> params_at_frequency(const Params<T>& P, double lam) {
  Params<T> Q = P;
  const double l2 = lam * lam;
  Q.xs = T(P.xs * l2); Q.beta = T(P.beta * l2); Q.beta2 = T(P.beta2 * l2);
  Q.par_g = T(P.par_g * l2); Q.lin_gx = T(P.lin_gx * l2); Q.two_xs_a2 = T(P.two_xs_a2 * l2);
  Q.xsh = T(P.xsh * l2); Q.lin_gxh = T(P.lin_gxh * l2); Q.tok_gxh = T(P.tok_gxh * l2);
  Q.sB0 = T(P.sB0 * lam); Q.sB0R0 = T(P.sB0R0 * lam);
  Q.k2n = T(P.k2n * lam); Q.n2k = T(P.n2k / lam);
  return Q;
}

// Output staging: 128-bit coalesced stores (DESIGN.md section 6 "Trajectory stores").  A saved sample is 6 state rows
// (+ 1 residual row) of consecutive rays.  Each thread drops its 7 values into its column of a [7][BLOCK] shared array;
// after a warp barrier lane l reads 16-byte chunks along the rows (conflict-free) and writes them with one 128-bit
// store each, so a warp emits 4 (fp64) / 2 (fp32) STG.128 wavefront groups of 512 contiguous bytes per row pair instead
// of 7 STG.64 / STG.32.  Requires the row pitch N to be a multiple of 16 / sizeof(T) (rows stay 16-byte aligned); other
// N fall back to scalar stores.  The staging slice is private to the warp: __syncwarp() is the only barrier.
template <class T, int BLOCK>
struct RowStore {
  typedef typename Vec16<T>::type V;
  static constexpr int VEC = 16 / sizeof(T), CPR = 32 / VEC;    // elements per chunk, chunks per row per warp
  T* stage;              // this warp's slice: row r at stage[r * BLOCK + lane]
  long long N, i0;       // row pitch; first ray of this warp
  int lane;
  bool vec;
  // rows6: row 0 of a [6][N] block or NULL; res_row: a [N] row or NULL
  RT_DEV void store(T* rows6, T* res_row, const T* v, T r, bool valid) const {
    if (!vec) {
      if (!valid) return;
      if (rows6) {
#pragma unroll
        for (int c = 0; c < 6; ++c) rows6[c * N + i0 + lane] = v[c];
      }
      if (res_row) res_row[i0 + lane] = r;
      return;
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) stage[c * BLOCK + lane] = v[c];
    stage[6 * BLOCK + lane] = r;
    __syncwarp();
    const int first = rows6 ? 0 : 6 * CPR, last = res_row ? 7 * CPR : 6 * CPR;
    for (int q = first + lane; q < last; q += 32) {
      const int row = q / CPR, col = (q % CPR) * VEC;
      if (i0 + col < N) {
        const V val = *reinterpret_cast<const V*>(stage + row * BLOCK + col);
        T* dst = (row < 6) ? rows6 + row * N : res_row;
        *reinterpret_cast<V*>(dst + i0 + col) = val;
      }
    }
    __syncwarp();
  }
};

// RESUME: the chunk kernel of rt_trace_until -- each ray's status at entry comes from A.status_in (a separate
// instantiation, so that the plain kernels' register allocation is untouched).
template <class T, int EQ, int DISP, bool PW, bool RESUME = false>
__global__ void __maxnreg__((trace_maxnreg<T, EQ, DISP>() + (PW ? pw_extra_regs<T, EQ, DISP>() : 0) + (RESUME ? 8 : 0)))
trace_kernel(const __grid_constant__ Params<T> P0, const __grid_constant__ TraceArgs<T> A) {
  constexpr int BLOCK = TraceShape<T, EQ>::BLOCK;
  const long long N = A.n_rays;
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool valid = i < N;
  typename TraceGather<T, EQ>::type gather;
  if constexpr (EQ == EQ_GRID) {
    typedef GatherCached<T, BLOCK> GC;
    __shared__ typename GC::V cache[GC::CHUNKS * BLOCK];
    gather.col = cache + threadIdx.x;
    gather.cell = -1; gather.pcell = -1;
  }
  __shared__ __align__(16) T stage[7 * BLOCK];
  Params<T> Pw;                                    // PW only: this ray's own copy of the w-dependent constants
  bool bad_w = false;                              // PW only: w_i not positive and finite defines no ray (reading A20):
  if constexpr (PW) {                              // status 2, never advanced, launch state back bit for bit, |D| = NaN
    const double wi = valid ? A.omega[i] : A.omega_ref;
    bad_w = !(wi > 0.0 && wi < __longlong_as_double(0x7ff0000000000000LL));
    Pw = params_at_frequency(P0, bad_w ? 1.0 : A.omega_ref / wi);
    if (bad_w) { Pw.k2n = T(1); Pw.n2k = T(1); }
  }
  const Params<T>& P = PW ? Pw : P0;
  T y[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    y[c] = valid ? A.x0[c * N + i] : T(0);
    y[3 + c] = valid ? A.k0[c * N + i] * P.k2n : T(0);          // n = c k / w  (Eq. 6)
  }
  int status = valid ? (bad_w ? 2 : 0) : 3;        // 3: padding lane of the last block, never stored
  if (RESUME && status == 0) status = A.status_in[i];
  // Everything the store needs is recomputed here from threadIdx / the kernel arguments, so that nothing of it stays
  // live across the step loop (the loop is register-bound).
  auto save = [&](T* rows6, T* res_row) {
    RowStore<T, BLOCK> out;
    out.lane = threadIdx.x & 31;
    out.stage = stage + (threadIdx.x & ~31);
    out.N = A.n_rays;
    out.i0 = (long long)blockIdx.x * BLOCK + (threadIdx.x & ~31);
    out.vec = (A.n_rays % RowStore<T, BLOCK>::VEC) == 0;
    T v[6];
#pragma unroll
    for (int c = 0; c < 3; ++c) { v[c] = y[c]; v[3 + c] = y[3 + c] * P.n2k; }
    // Resume mode: a ray that was already frozen at entry has never been advanced; its k rows go back bit for bit
    // (re-read here; out_status is only written after the last store) instead of through the round trip k -> n -> k, so
    // a frozen ray stays frozen however many chunks follow.  Nothing of this is live across the step loop.
    if (RESUME) {
      const long long ii = (long long)blockIdx.x * BLOCK + threadIdx.x;
      if (ii < A.n_rays && A.status_in[ii] != 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) v[3 + c] = A.k0[c * A.n_rays + ii];
      }
    }
    T r = res_row ? abs_residual<T, EQ, DISP>(P, y, gather) : T(0);
    if (PW && bad_w) r = rt_nan<T>();
    out.store(rows6, res_row, v, r, out.i0 + out.lane < A.n_rays);
  };
  // Sample m = state after m * stride steps (sample 0 = launch state).  The inner loop holds the step and nothing else.
  const long long n_outer = A.traj ? A.n_steps / A.stride : 1, n_inner = A.traj ? A.stride : A.n_steps;
  if (A.traj) save(A.traj, A.res);
  for (long long m = 1; m <= n_outer; ++m) {
    long long s = 0;
#pragma unroll 1
    for (; s < n_inner; ++s)                        // the hot loop: ion terms by their series
      if (status == 0) {
        const int st = rk4_step<T, EQ, DISP, true>(P, A.h, A.hh, A.h3, A.h6, y, gather);
        if (st < 0) break;                         // a stage point outside the series' range (Y2 >= Params::y2cap)
        status = st;
      }
    if (DISP != DISP_O) {
#pragma unroll 1
      for (; s < n_inner; ++s)                      // the rest of this stretch exactly (rare: nothing in BASELINE's configs)
        if (status == 0) status = rk4_step<T, EQ, DISP, false>(P, A.h, A.hh, A.h3, A.h6, y, gather);
    }
    if (A.traj) save(A.traj + m * 6 * A.n_rays, A.res ? A.res + m * A.n_rays : nullptr);
  }
  if (A.fin || (!A.traj && A.res)) save(A.fin, A.traj ? nullptr : A.res);
  if (A.status && valid) A.status[i] = status;
}

// ---- fp32, two rays per thread: packed f32x2 arithmetic (rt_math.cuh: f32x2) ------------------------------------------
// Thread t of a block traces rays 2 (block * BLOCK + t) and the next one, one in each half of every f32x2 value; a warp
// owns 64 consecutive rays.  Same formulas per ray as trace_kernel<float, ...> (the IEEE fp32 operation on each half), and a
// ray's result does not depend on which half or thread it rides in -- but the two kernels are NOT bit-identical to each
// other: where the scalar code has a multiply followed by an add the compiler may contract the pair into one FFMA, while
// the packed code keeps the two instructions it was written with (measured: one 40-step chunk differs by <= 2e-6 relative,
// tests/test_gpu_until.py).  So an fp32 result depends on the entry point: rt_trace / rt_trace_host run this kernel, rt_trace_w
// and rt_trace_until the scalar one (include/rt.h says so at rt_trace_until).  What changes here is the instruction stream:
// one FFMA2 / FMUL2 / FADD2 issue slot serves two rays, and MUFU seeds, domain tests and table look-ups are done per half.
// A lane whose ray is frozen keeps computing on its frozen state and is masked out of every update.
// The packed kernels exist for every dispersion function over the analytic equilibria and for the full determinant over the
// grid equilibrium.  Over the grid the spline look-ups are NOT packed (rt_math.cuh: grid_values_per_ray): each ray of the
// thread has its own scalar shared-memory cell cache and its look-ups run in scalar arithmetic, the nine results are packed
// and everything after them runs packed -- fully packed look-ups were measured and dropped (profiles/r2_tuning.md: pairing
// every spline piece with the other ray's costs ~100 register moves per stage).
template <int EQ> struct TraceShape2 { static constexpr int BLOCK = 64, MAXNREG = 128; };
// the slabs' short stages like more warps (config 2 fp32 6.00 -> 5.86 ms at 80 registers, config 3 fp32 4.90 -> 4.76 ms at 96)
template <> struct TraceShape2<EQ_PARABOLIC> { static constexpr int BLOCK = 64, MAXNREG = 80; };
template <> struct TraceShape2<EQ_LINEAR> { static constexpr int BLOCK = 64, MAXNREG = 96; };

template <int EQ, int DISP>
__global__ void __maxnreg__((TraceShape2<EQ>::MAXNREG))
trace_kernel_x2(const __grid_constant__ Params<float> P0, const __grid_constant__ TraceArgs<float> A) {
  typedef f32x2 T;
  constexpr int BLOCK = TraceShape2<EQ>::BLOCK, RAYS = 2 * BLOCK;
  const Params<T>& P = static_cast<const Params<T>&>(reinterpret_cast<const Params<T>&>(P0));
  const long long N = A.n_rays;
  const long long ia = ((long long)blockIdx.x * BLOCK + threadIdx.x) * 2, ib = ia + 1;
  const bool va = ia < N, vb = ib < N;
  static_assert(EQ != EQ_GRID || DISP == DISP_FULL, "grid equilibrium: the packed kernel exists for the full determinant");
  typename std::conditional<EQ == EQ_GRID, GatherPair<BLOCK>, GatherDirect>::type gather;
  if constexpr (EQ == EQ_GRID) {
    typedef GatherCached<float, BLOCK, true> GC;
    __shared__ typename GC::V cache[2 * GC::CHUNKS * BLOCK];
    gather.a.col = cache + threadIdx.x;              gather.a.cell = -1; gather.a.pcell = -1;
    gather.b.col = cache + GC::CHUNKS * BLOCK + threadIdx.x; gather.b.cell = -1; gather.b.pcell = -1;
  }
  __shared__ __align__(16) float stage[7 * RAYS];
  T y[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    y[c] = T(va ? A.x0[c * N + ia] : 0.0f, vb ? A.x0[c * N + ib] : 0.0f);
    y[3 + c] = T(va ? A.k0[c * N + ia] : 0.0f, vb ? A.k0[c * N + ib] : 0.0f) * P.k2n;      // n = c k / w  (Eq. 6)
  }
  int sa = va ? 0 : 3, sb = vb ? 0 : 3;            // 3: padding lane, never stored
  // store: each thread drops its two rays' 7 values into columns 2 lane, 2 lane + 1 of its warp's [7][64] slice; then the
  // warp writes the rows with 128-bit stores (16 chunks of 16 bytes per row).  Nothing of this is live across the step loop.
  auto save = [&](float* rows6, float* res_row) {
    const int lane = threadIdx.x & 31;
    float* st = stage + (threadIdx.x & ~31) * 2;                                   // this warp's slice: row r at st[r * RAYS]
    const long long i0 = ((long long)blockIdx.x * BLOCK + (threadIdx.x & ~31)) * 2;  // first ray of this warp
    const long long NN = A.n_rays;
    T v[7];
#pragma unroll
    for (int c = 0; c < 3; ++c) { v[c] = y[c]; v[3 + c] = y[3 + c] * P.n2k; }
    GatherDirect direct;                                                           // once per sample: straight from the tables
    v[6] = res_row ? abs_residual<T, EQ, DISP>(P, y, direct) : T(0.0f);
    if ((NN & 3) != 0) {                                                           // rows not 16-byte aligned: scalar stores
      const long long ja = i0 + 2 * lane;
#pragma unroll
      for (int c = 0; c < 7; ++c) {
        float* dst = (c < 6) ? (rows6 ? rows6 + c * NN : nullptr) : res_row;
        if (!dst) continue;
        if (ja < NN) dst[ja] = v[c].lo();
        if (ja + 1 < NN) dst[ja + 1] = v[c].hi();
      }
      return;
    }
#pragma unroll
    for (int c = 0; c < 7; ++c) *reinterpret_cast<float2*>(st + c * RAYS + 2 * lane) = make_float2(v[c].lo(), v[c].hi());
    __syncwarp();
    const int first = rows6 ? 0 : 6 * 16, last = res_row ? 7 * 16 : 6 * 16;
    for (int q = first + lane; q < last; q += 32) {
      const int row = q >> 4, col = (q & 15) * 4;
      if (i0 + col < NN) {
        const float4 val = *reinterpret_cast<const float4*>(st + row * RAYS + col);
        float* dst = (row < 6) ? rows6 + row * NN : res_row;
        *reinterpret_cast<float4*>(dst + i0 + col) = val;
      }
    }
    __syncwarp();
  };
  const long long n_outer = A.traj ? A.n_steps / A.stride : 1, n_inner = A.traj ? A.stride : A.n_steps;
  if (A.traj) save(A.traj, A.res);
  for (long long m = 1; m <= n_outer; ++m) {
    // one step of both rays with the acceptance rule (reading A12) per ray: a stage point outside the domain -> status 1,
    // a non-finite new state -> 2.  SERIES: returns false, with nothing changed, if a stage point of either ray lay outside
    // the range of the ion terms' series.
    auto step = [&](auto series) -> bool {
      constexpr bool SERIES = decltype(series)::value;
      T ys[6];
      mask2 fast = {true, true};
      const mask2 ok = rk4_stages<T, EQ, DISP, SERIES>(P, T(A.h), T(A.hh), T(A.h3), T(A.h6), y, ys, gather, fast);
      if (SERIES && DISP != DISP_O && !rt_all(fast)) return false;
      mask2 fin = {true, true};
#pragma unroll
      for (int j = 0; j < 6; ++j) fin = rt_and(fin, rt_finite(ys[j]));
      const mask2 acc = {sa == 0 && ok.a && fin.a, sb == 0 && ok.b && fin.b};
      if (acc.a && acc.b) {                        // the common case: both rays advance, no per-half selects
#pragma unroll
        for (int j = 0; j < 6; ++j) y[j] = ys[j];
      } else {
        if (sa == 0 && !acc.a) sa = ok.a ? 2 : 1;
        if (sb == 0 && !acc.b) sb = ok.b ? 2 : 1;
#pragma unroll
        for (int j = 0; j < 6; ++j) y[j] = rt_select(acc, ys[j], y[j]);
      }
      return true;
    };
    long long s = 0;
#pragma unroll 1
    for (; s < n_inner; ++s) {                     // the hot loop: ion terms by their series
      if (sa != 0 && sb != 0) break;               // both rays frozen (or padding): nothing left to do in this stretch
      if (!step(std::true_type())) break;
    }
    if (DISP != DISP_O) {
#pragma unroll 1
      for (; s < n_inner; ++s) {                   // the rest of this stretch exactly (rare)
        if (sa != 0 && sb != 0) break;
        step(std::false_type());
      }
    }
    if (A.traj) save(A.traj + m * 6 * A.n_rays, A.res ? A.res + m * A.n_rays : nullptr);
  }
  if (A.fin || (!A.traj && A.res)) save(A.fin, A.traj ? nullptr : A.res);
  if (A.status) {
    if (va) A.status[ia] = sa;
    if (vb) A.status[ib] = sb;
  }
}

// ---- second ensemble workload: full-orbit charged particles in the same equilibria -----------------
// PAPER.md L121 ("full orbit affects on particle losses"), L213 ("waves or particles ... a large ensemble of independent
// problems").  Newton-Lorentz equations dx/dt = v, dv/dt = (q/m) v x B(x), no electric field; state y = (x, v) in SI.
// B comes from the same `equilibrium` code as the rays' (its density / gradient parts are dead code here and are
// eliminated by the compiler); the slab's field is along z, so dv_z/dt = 0 is skipped and v_z stays bit-for-bit constant.
template <class T, int EQ, class Gather>
RT_DEV bool orbit_rhs(const Params<T>& P, T qm, const T* y, T* f, Gather& gather) {
  Local<T> L;
  const T* v = y + 3;
  const bool inside = equilibrium<T, EQ, DISP_FULL>(P, y, v, L, gather);
  f[0] = v[0]; f[1] = v[1]; f[2] = v[2];
  if (EQ == EQ_LINEAR) {
    const T w = qm * L.B[2];
    f[3] = w * v[1]; f[4] = -w * v[0]; f[5] = T(0);
    return inside;
  }
  const T Bx = rt_fma(L.B[0], L.cph, -L.B[1] * L.sph) * qm;
  const T By = rt_fma(L.B[0], L.sph, L.B[1] * L.cph) * qm;
  const T Bz = L.B[2] * qm;
  f[3] = rt_fma(v[1], Bz, -v[2] * By);
  f[4] = rt_fma(v[2], Bx, -v[0] * Bz);
  f[5] = rt_fma(v[0], By, -v[1] * Bx);
  return inside;
}

// One classical RK4 step of the orbit equations; same acceptance rule and return codes as rk4_step.
// fp32 (COMP): the POSITION is carried as the unevaluated sum y[0..2] + xlo[0..2].  A step moves a particle by ~1e-3 m at
// |x| ~ 2 m, so a plain fp32 update loses ~0.2 um per step; over 1000 steps that random walk reaches several um, the field
// seen by the particle is off by dB/B = dR/R ~ 3e-6, and the gyro-phase (~100 rad) by ~2e-4 -- the velocity error that
// bench.py's sampled parity showed (2.2e-4, over north_star's 1e-4).  So the step's increment is summed on its own and
// added to (y, xlo) with a Fast2Sum (|y| >> |increment| for positions): 12 FADD per step.  Velocities rotate through zero
// and their rounding only random-walks the phase (~2e-6): they keep the plain update.  fp64 is untouched (xlo unused).
template <class T, int EQ, class Gather>
RT_DEV int orbit_step(const Params<T>& P, T qm, T h, T* y, T* xlo, Gather& gather) {
  constexpr bool COMP = sizeof(T) == 4;
  const T hh = T(0.5) * h, h6 = h * T(1.0 / 6.0), h3 = h * T(1.0 / 3.0);
  constexpr int NA = (EQ == EQ_LINEAR) ? 5 : 6;          // active components (slab: v_z is constant)
  T k[6], acc[6], ys[6];
#pragma unroll
  for (int j = 0; j < 6; ++j) { k[j] = T(0); acc[j] = (COMP && j < 3) ? T(0) : y[j]; ys[j] = y[j]; }
  bool ok = true;
  auto stage = [&](int st) {
    const T a = (st == 0) ? T(0) : ((st == 3) ? h : hh);
    const T w = (st == 0 || st == 3) ? h6 : h3;
#pragma unroll
    for (int j = 0; j < NA; ++j) ys[j] = rt_fma(a, k[j], y[j]);
    ok = orbit_rhs<T, EQ>(P, qm, ys, k, gather) && ok;
#pragma unroll
    for (int j = 0; j < NA; ++j) acc[j] = rt_fma(w, k[j], acc[j]);
  };
  if (EQ == EQ_GRID) {               // one copy of the stage code, as in rk4_stages
#pragma unroll 1
    for (int st = 0; st < 4; ++st) stage(st);
  } else {                           // analytic fields: the four stages unrolled (the compiler schedules across them)
#pragma unroll
    for (int st = 0; st < 4; ++st) stage(st);
  }
  if (!ok) return 1;
  T nlo[3] = {T(0), T(0), T(0)};
  if constexpr (COMP) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const T t = acc[j] + xlo[j];       // the step's increment plus what earlier steps could not represent
      const T s = y[j] + t;
      nlo[j] = t - (s - y[j]);           // Fast2Sum: exact for |y| >= |t|
      acc[j] = s;
    }
  }
  bool fin = true;
#pragma unroll
  for (int j = 0; j < 6; ++j) fin = fin && rt_finite(acc[j]);
  if (!fin) return 2;
#pragma unroll
  for (int j = 0; j < 6; ++j) y[j] = acc[j];
  if constexpr (COMP) {
#pragma unroll
    for (int j = 0; j < 3; ++j) xlo[j] = nlo[j];
  }
  return 0;
}

template <class T>
struct OrbitArgs {
  const T* x0;
  const T* v0;
  T* traj;
  T* fin;
  T* drift;             // relative kinetic-energy drift |v|^2/|v0|^2 - 1
  int32_t* status;
  long long n;
  long long n_steps;
  long long stride;
  T h;                  // time step [s]
  T qm;                 // charge over mass [C/kg]
};

template <class T, int EQ>
__global__ void __maxnreg__((TraceShape<T, EQ>::MAXNREG))
orbit_kernel(const __grid_constant__ Params<T> P, const __grid_constant__ OrbitArgs<T> A) {
  constexpr int BLOCK = TraceShape<T, EQ>::BLOCK;
  const long long N = A.n;
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool valid = i < N;
  typename TraceGather<T, EQ>::type gather;
  if constexpr (EQ == EQ_GRID) {
    typedef GatherCached<T, BLOCK> GC;
    __shared__ typename GC::V cache[GC::CHUNKS * BLOCK];
    gather.col = cache + threadIdx.x;
    gather.cell = -1; gather.pcell = -1;
  }
  __shared__ __align__(16) T stage[7 * BLOCK];
  T y[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    y[c] = valid ? A.x0[c * N + i] : T(0);
    y[3 + c] = valid ? A.v0[c * N + i] : T(1);
  }
  T xlo[3] = {T(0), T(0), T(0)};          // fp32: low parts of the position (orbit_step)
  const T inv_e0 = T(1) / rt_fma(y[3], y[3], rt_fma(y[4], y[4], y[5] * y[5]));
  int status = valid ? 0 : 3;
  auto save = [&](T* rows6, T* drift_row) {
    RowStore<T, BLOCK> out;
    out.lane = threadIdx.x & 31;
    out.stage = stage + (threadIdx.x & ~31);
    out.N = A.n;
    out.i0 = (long long)blockIdx.x * BLOCK + (threadIdx.x & ~31);
    out.vec = (A.n % RowStore<T, BLOCK>::VEC) == 0;
    const T e = rt_fma(y[3], y[3], rt_fma(y[4], y[4], y[5] * y[5]));
    out.store(rows6, drift_row, y, rt_fma(e, inv_e0, T(-1)), out.i0 + out.lane < A.n);
  };
  const long long n_outer = A.traj ? A.n_steps / A.stride : 1, n_inner = A.traj ? A.stride : A.n_steps;
  if (A.traj) save(A.traj, A.drift);
  for (long long m = 1; m <= n_outer; ++m) {
#pragma unroll 1
    for (long long s = 0; s < n_inner; ++s)
      if (status == 0) status = orbit_step<T, EQ>(P, A.qm, A.h, y, xlo, gather);
    if (A.traj) save(A.traj + m * 6 * A.n, A.drift ? A.drift + m * A.n : nullptr);
  }
  if (A.fin || (!A.traj && A.drift)) save(A.fin, A.traj ? nullptr : A.drift);
  if (A.status && valid) A.status[i] = status;
}

template <class T, int EQ, int DISP>
__global__ void __launch_bounds__(AUX_BLOCK)
rhs_kernel(const __grid_constant__ Params<T> P, const T* __restrict__ x, const T* __restrict__ k, long long n,
           T* __restrict__ D_out, T* __restrict__ rhs_out, int32_t* __restrict__ inside_out) {
  const long long i = (long long)blockIdx.x * AUX_BLOCK + threadIdx.x;
  if (i >= n) return;
  T y[6], f[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) { y[c] = x[c * n + i]; y[3 + c] = k[c * n + i] * P.k2n; }
  GatherDirect gather;
  const bool inside = ray_rhs_scaled<T, EQ, DISP>(P, y, f, gather);
  if (rhs_out) {
#pragma unroll
    for (int c = 0; c < 6; ++c) rhs_out[c * n + i] = inside ? f[c] : T(0);
  }
  if (D_out) {
    bool in2;
    const T D = ray_D<T, EQ, DISP>(P, y, &in2, gather);
    D_out[i] = in2 ? D : rt_nan<T>();
  }
  if (inside_out) inside_out[i] = inside ? 1 : 0;
}

// Launch conditions.  `dir` is passed to the equilibrium in the role of n, so L.G = dir.B.
template <int EQ, int DISP, bool PW>
__global__ void __launch_bounds__(AUX_BLOCK)
launch_kernel(const __grid_constant__ Params<double> P0, int branch, const double* __restrict__ x0,
              const double* __restrict__ dir, const double* __restrict__ omega, double omega_ref, long long n,
              double* __restrict__ k0, double* __restrict__ D_out) {
  const long long i = (long long)blockIdx.x * AUX_BLOCK + threadIdx.x;
  if (i >= n) return;
  const Params<double> P = PW ? params_at_frequency(P0, omega_ref / omega[i]) : P0;
  double x[3], d[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) { x[c] = x0[c * n + i]; d[c] = dir[c * n + i]; }
  Local<double> L;
  GatherDirect gather;
  const bool inside = equilibrium<double, EQ, DISP>(P, x, d, L, gather);
  const double X = L.X;
  double Y2 = 0.0, c2 = 0.0, n2;
  if (DISP == DISP_O) {
    n2 = 1.0 - X;
  } else {
    Y2 = P.beta * L.b2;
    const StixT<double> st = stix(P, X, Y2);
    const double RL = st.s * st.s - st.d2;
    if (DISP == DISP_X) {
      n2 = RL / st.s;
    } else {
      // Stix's biquadratic A n^4 - B n^2 + C = 0 at the angle between dir and B
      c2 = L.G * L.G / L.b2;
      const double s2 = 1.0 - c2;
      const double A = st.s * s2 + st.p * c2;
      const double Bq = RL * s2 + st.p * st.s * (1.0 + c2);
      const double Cq = st.p * RL;
      const double F = sqrt(Bq * Bq - 4.0 * A * Cq);
      const double r1 = (Bq - F) / (2.0 * A), r2 = (Bq + F) / (2.0 * A);
      const bool r1_is_O = fabs(r1 - st.p) <= fabs(r2 - st.p);      // reading A11: "O" = the root nearer to P
      n2 = (branch == 0) ? (r1_is_O ? r1 : r2) : (r1_is_O ? r2 : r1);
    }
  }
  if (!inside) n2 = rt_nan<double>();
  double sn = sqrt(n2);                                              // NaN if evanescent
  for (int it = 0; it < 8 && isfinite(sn); ++it) {
    const double v = sn * sn, u = v * c2;
    const double D = disp_value<double, DISP>(P, X, Y2, u, v);
    if (fabs(D) < 1e-15) break;
    double DX, DY2, Du, Dv;
    disp_partials<double, DISP>(P, X, Y2, u, v, DX, DY2, Du, Dv);
    const double dDds = 2.0 * sn * (Dv + c2 * Du);
    const double s_new = sn - D / dDds;
    if (!(s_new > 0.0) || !isfinite(s_new)) break;
    sn = s_new;
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) k0[c * n + i] = sn * d[c] * P.n2k;
  if (D_out) {
    const double v = sn * sn;
    D_out[i] = disp_value<double, DISP>(P, X, Y2, v * c2, v);
  }
}

// Launch conditions exactly as the paper states them: w, x, k_y, k_z fixed; k_x by Newton's method from
// the caller's initial guess (which selects the root) until |D| < tol, at most max_iter updates.  x is fixed, so the
// equilibrium is evaluated once; only n^2 and n.B change with k_x.  dD/dn_x = 2 D_v n_x + (2 G D_u / |B|^2) B_x.
// Outputs: k0 = (k_x, k_y, k_z) at the last iterate (k_y, k_z copied bit for bit), D there, iters = updates made if
// |D| < tol was reached, -1 if not; outside the domain or on a non-finite iterate k_x = D = NaN and iters = -1.
template <int EQ, int DISP, bool PW>
__global__ void __launch_bounds__(AUX_BLOCK)
launch_kx_kernel(const __grid_constant__ Params<double> P0, const double* __restrict__ x0, const double* __restrict__ kg,
                 const double* __restrict__ omega, double omega_ref, long long n, int max_iter, double tol,
                 double* __restrict__ k0, double* __restrict__ D_out, int32_t* __restrict__ iters_out) {
  const long long i = (long long)blockIdx.x * AUX_BLOCK + threadIdx.x;
  if (i >= n) return;
  const Params<double> P = PW ? params_at_frequency(P0, omega_ref / omega[i]) : P0;
  double x[3], nn[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) { x[c] = x0[c * n + i]; nn[c] = kg[c * n + i] * P.k2n; }
  Local<double> L;
  GatherDirect gather;
  const bool inside = equilibrium<double, EQ, DISP>(P, x, nn, L, gather);
  double B[3] = {0.0, 0.0, 0.0}, ib2 = 0.0, Y2 = 0.0;
  if (DISP != DISP_O) Y2 = P.beta * L.b2;
  if (DISP == DISP_FULL) {
    if (EQ == EQ_LINEAR) {
      B[2] = L.B[2];
    } else {                                  // axisymmetric kinds: (R^, phi^, Z^) components -> Cartesian
      B[0] = L.B[0] * L.cph - L.B[1] * L.sph;
      B[1] = L.B[0] * L.sph + L.B[1] * L.cph;
      B[2] = L.B[2];
    }
    ib2 = 1.0 / L.b2;
  }
  const double qnan = rt_nan<double>();
  double nx = inside ? nn[0] : qnan, D = qnan;
  int iters = -1;
  bool updated = false;                       // no update made: k_x goes back bit for bit
  for (int it = 0; it <= max_iter && inside; ++it) {
    const double v = nx * nx + nn[1] * nn[1] + nn[2] * nn[2];
    const double G = nx * B[0] + nn[1] * B[1] + nn[2] * B[2];
    const double u = G * G * ib2;
    D = disp_value<double, DISP>(P, L.X, Y2, u, v);
    if (!isfinite(D)) { nx = qnan; D = qnan; break; }
    if (fabs(D) < tol) { iters = it; break; }
    if (it == max_iter) break;
    double DX, DY2, Du, Dv;
    disp_partials<double, DISP>(P, L.X, Y2, u, v, DX, DY2, Du, Dv);
    nx -= D / (2.0 * Dv * nx + 2.0 * G * Du * ib2 * B[0]);
    updated = true;
    if (!isfinite(nx)) { nx = qnan; D = qnan; break; }
  }
  k0[i] = (updated || !inside) ? nx * P.n2k : kg[i];
  k0[n + i] = kg[n + i];
  k0[2 * n + i] = kg[2 * n + i];
  if (D_out) D_out[i] = D;
  if (iters_out) iters_out[i] = iters;
}

// Critical-surface diagnostics (cut-offs and resonances along the ray).
// Rows of out [10][n]: n_e [m^-3], |B| [T], X = wpe^2/w^2, Y = |Wce|/w, S, Dx, P (Eq. 8-10), R = S + Dx,
// L = S - Dx, n_par^2 = (n.B)^2/|B|^2.  Cut-offs: P = 0 (X = 1 for electrons only), R = 0, L = 0; resonance: S = 0 (upper
// hybrid), Y = 1 (cyclotron).  Everything is NaN outside the equilibrium's domain.  inv_alpha_ref = n_e / X at w_ref.
template <int EQ, bool PW>
__global__ void __launch_bounds__(AUX_BLOCK)
diag_kernel(const __grid_constant__ Params<double> P0, double inv_alpha_ref, const double* __restrict__ x,
            const double* __restrict__ k, const double* __restrict__ omega, double omega_ref, long long n,
            double* __restrict__ out) {
  constexpr int DISP = (EQ == EQ_PARABOLIC) ? DISP_O : DISP_FULL;
  const long long i = (long long)blockIdx.x * AUX_BLOCK + threadIdx.x;
  if (i >= n) return;
  const double lam = PW ? omega_ref / omega[i] : 1.0;
  const Params<double> P = PW ? params_at_frequency(P0, lam) : P0;
  double xx[3], nn[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) { xx[c] = x[c * n + i]; nn[c] = k[c * n + i] * P.k2n; }
  Local<double> L;
  GatherDirect gather;
  L.b2 = 0.0; L.G = 0.0;
  const bool inside = equilibrium<double, EQ, DISP>(P, xx, nn, L, gather);
  const double X = L.X, b2 = (EQ == EQ_PARABOLIC) ? 0.0 : L.b2;
  const double Y2 = P.beta * b2;
  const StixT<double> st = stix(P, X, Y2);
  const double Y = sqrt(Y2);
  const double Dx = X * Y * st.del;
  const double v[10] = {X * inv_alpha_ref / (lam * lam), sqrt(b2), X, Y, st.s, Dx, st.p, st.s + Dx, st.s - Dx,
                        (EQ == EQ_PARABOLIC) ? 0.0 : L.G * L.G / b2};
#pragma unroll
  for (int r = 0; r < 10; ++r) out[r * n + i] = inside ? v[r] : rt_nan<double>();
}

// out[0] = max |D|, out[1] = sum |D|, out[2] = #finite, out[3..5] = #status 0/1/2.  out must be zeroed beforehand.
template <class T>
__global__ void __launch_bounds__(256)
reduce_kernel(const T* __restrict__ res, const int32_t* __restrict__ status, long long n, double* __restrict__ out) {
  double mx = 0.0, sm = 0.0, cnt = 0.0, s0 = 0.0, s1 = 0.0, s2 = 0.0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    if (res) {
      const double r = (double)res[i];
      if (isfinite(r)) { mx = fmax(mx, fabs(r)); sm += fabs(r); cnt += 1.0; }
    }
    if (status) {
      const int s = status[i];
      s0 += (s == 0); s1 += (s == 1); s2 += (s == 2);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    sm += __shfl_xor_sync(0xffffffffu, sm, o);
    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    s0 += __shfl_xor_sync(0xffffffffu, s0, o);
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
  }
  if ((threadIdx.x & 31) == 0) {
    // non-negative doubles order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long*>(out), (unsigned long long)__double_as_longlong(mx));
    atomicAdd(out + 1, sm);
    atomicAdd(out + 2, cnt);
    atomicAdd(out + 3, s0);
    atomicAdd(out + 4, s1);
    atomicAdd(out + 5, s2);
  }
}

// The convergence workflow's decision step (rt_trace_until; "chaining calls to evaluation and reduction
// kernels until a tolerance is met").  Runs as the last node of the body of a CUDA-graph WHILE node, after the chunk's
// trace_kernel and reduce_kernel: one thread reads the reduction, counts the chunk, records why the loop stops and
// sets the WHILE condition on the device -- no host round trip between chunks.
//   info[0] chunks run   info[1] rays still active (status 0)   info[2] max |D| (bit pattern of a double)
//   info[3] reason: 0 max_chunks reached, 1 every ray frozen, 2 max |D| > tol        info[4..9]: reduce_kernel's out[6]
// mode: bit 0 = a chunk has just run (count it), bit 1 = set the WHILE condition (the launch inside the graph's body).
// The stop tests belong to the end of a chunk: with max_chunks == 0 no chunk runs, none is made and the reason is 0
// whatever the launch state looks like (as the oracle's loop, which is never entered then).
__global__ void until_decide_kernel(long long* __restrict__ info, double tol, long long max_chunks,
                                    cudaGraphConditionalHandle cond, int mode) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const double* red = reinterpret_cast<const double*>(info + 4);
  const long long chunks = info[0] + ((mode & 1) ? 1 : 0);
  const long long n_active = (long long)red[3];
  const double max_D = red[0];
  long long reason = 0;
  bool go = chunks < max_chunks;
  if (max_chunks > 0) {
    if (n_active == 0) { reason = 1; go = false; }
    else if (max_D > tol) { reason = 2; go = false; }
  }
  info[0] = chunks; info[1] = n_active; info[2] = __double_as_longlong(max_D); info[3] = reason;
  if (mode & 2) cudaGraphSetConditional(cond, go ? 1u : 0u);
}

// Roofline denominator: FMA_CHAINS independent accumulators per thread, each a dependent chain of fused multiply-adds.
//   SHAPE 0 (the denominator rt_fma_peak reports): acc = acc * a + acc -- two distinct source registers;
//   SHAPE 1: acc = acc * a + b with a, b shared by all chains -- three distinct sources, but consecutive instructions
//            find a and b in the operand-reuse cache;
//   SHAPE 2: acc_j = acc_j * a_j + b_j with per-chain a_j, b_j (8 chains, each used twice per round) -- three distinct
//            64-bit registers read from the register file by every instruction: what most DFMAs of real code look like;
//   SHAPE 3: shape 0 plus 4 independent MUFU reciprocal seeds per 16 FMAs (the ratio of the O-mode kernel; the full
//            determinant has 1 per 22): the seeds run on the XU pipe BESIDE the FMA pipe and cost ~2 % of the FMA rate;
//   SHAPE 4: shape 0 with ONE chain per thread: the rate is warps-per-scheduler / dependent-issue latency (8 cycles for
//            a DFMA), i.e. 4 warps per scheduler saturate the FP64 pipe without any instruction-level parallelism.
//   SHAPE 5 (fp32 only; the denominator rt_fma_peak reports for fp32): shape 0 with PACKED f32x2 accumulators -- 8 chains
//            of FFMA2, each instruction two fused multiply-adds: what the chip's FP32 FMA pipe delivers at best;
//   SHAPE 6 (fp32 only): shape 2 with packed accumulators (three distinct 64-bit register pairs per FFMA2).
// On B200 the DFMA rate is 63.7 / 58 / 42.7 per clock per SM for shapes 0 / 1 / 2: an FP64 instruction that reads three
// registers from the register file occupies the pipe for 3 cycles instead of 2 (profiles/r2_fma_peak_shapes.md).  FP32:
// 123.2 / 117 / 78.8 scalar, 127.9 / 84.9 packed (shapes 5 / 6): the same port limit, two FMAs per issue slot.
constexpr int FMA_CHAINS = 16;
constexpr int FMA_BLOCK = 256;
RT_DEV double rcp_seed(double x) { double r; asm volatile("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }
RT_DEV float rcp_seed(float x) { float r; asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
template <class T, int SHAPE>
__global__ void __launch_bounds__(FMA_BLOCK)
fma_peak_kernel(T* __restrict__ sink, long long iters, T a, T b, unsigned long long* __restrict__ clk) {
  constexpr int NC = (SHAPE == 2) ? FMA_CHAINS / 2 : (SHAPE == 4) ? 1 : FMA_CHAINS;
  T acc[NC], aj[NC], bj[NC], seed[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) seed[j] = T(1.5) + T(threadIdx.x + j);
#pragma unroll
  for (int j = 0; j < NC; ++j) {
    acc[j] = T(threadIdx.x + j) * T(1e-3);
    aj[j] = a + T(threadIdx.x + j) * T(1e-9);
    bj[j] = b + T(threadIdx.x + 2 * j) * T(1e-9);
  }
  unsigned long long t0, t1;
  const long long c0 = clock64();
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t0));
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < FMA_CHAINS; ++j) {
        const int c = j % NC;
        acc[c] = (SHAPE == 0 || SHAPE == 3 || SHAPE == 4) ? rt_fma(acc[c], a, acc[c])
                 : (SHAPE == 1) ? rt_fma(acc[c], a, b) : rt_fma(acc[c], aj[c], bj[c]);
      }
      if (SHAPE == 3) {
#pragma unroll
        for (int j = 0; j < 4; ++j) seed[j] = rcp_seed(seed[j]);
      }
    }
  }
  const long long c1 = clock64();
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t1));
  T s = T(0);
#pragma unroll
  for (int j = 0; j < NC; ++j) s += acc[j];
  if (SHAPE == 3) s += seed[0] + seed[1] + seed[2] + seed[3];
  sink[(long long)blockIdx.x * FMA_BLOCK + threadIdx.x] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) { clk[0] = (unsigned long long)(c1 - c0); clk[1] = t1 - t0; }
}

// shapes 5 / 6: the same FMA count per iteration (FMA_CHAINS x 8) issued as FMA_CHAINS / 2 packed chains
template <int SHAPE>
__global__ void __launch_bounds__(FMA_BLOCK)
fma_peak_packed_kernel(float* __restrict__ sink, long long iters, float a, float b, unsigned long long* __restrict__ clk) {
  constexpr int NC = FMA_CHAINS / 2;
  f32x2 acc[NC], aj[NC], bj[NC];
#pragma unroll
  for (int j = 0; j < NC; ++j) {
    acc[j] = f32x2(float(threadIdx.x + j) * 1e-3f, float(threadIdx.x + j + 1) * 1e-3f);
    aj[j] = f32x2(a + float(threadIdx.x + j) * 1e-9f, a - float(j) * 1e-9f);
    bj[j] = f32x2(b + float(threadIdx.x + 2 * j) * 1e-9f, b);
  }
  const f32x2 pa(a);
  unsigned long long t0, t1;
  const long long c0 = clock64();
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t0));
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < NC; ++j) acc[j] = (SHAPE == 5) ? rt_fma(acc[j], pa, acc[j]) : rt_fma(acc[j], aj[j], bj[j]);
    }
  }
  const long long c1 = clock64();
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t1));
  float s = 0.0f;
#pragma unroll
  for (int j = 0; j < NC; ++j) s += acc[j].lo() + acc[j].hi();
  sink[(long long)blockIdx.x * FMA_BLOCK + threadIdx.x] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) { clk[0] = (unsigned long long)(c1 - c0); clk[1] = t1 - t0; }
}

// Unit-test hook for the hot loop's own reciprocal / square-root routines (rt_math.cuh), which no output of the path shows
// in isolation: out[i] = f(x[i]) with f = 0 rt_rcp, 1 rt_rsqrt, 2 rt_sqrt_fast, in the precision of T.
template <class T>
__global__ void __launch_bounds__(AUX_BLOCK)
math_probe_kernel(int fn, const T* __restrict__ x, long long n, T* __restrict__ out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const T v = x[i];
  out[i] = (fn == 0) ? rt_rcp(v) : (fn == 1) ? rt_rsqrt(v) : rt_sqrt_fast(v);
}

#endif  // __CUDACC__

}  // namespace rt
