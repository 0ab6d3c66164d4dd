// rt_kernels.cuh -- the CUDA kernels of the hot path (sm_100a).
//
//   trace_kernel   one thread per ray; loads (x0, k0) once, runs all n_steps classical RK4 steps
//                  with the state, the stage slopes and every intermediate of D's gradient in registers, and writes
//                  decimated SoA trajectory samples / the final state / |D| / status (steps a1-a6 of DESIGN.md).
//   rhs_kernel     one stage evaluation per point (diagnostics and gradient parity tests).
//   launch_kernel  launch conditions: closed-form |n| on D = 0 plus Newton polish.
//   reduce_kernel  max / sum of |D| and status counts (PAPER.md L76 reduction kernels).
//   fma_peak_kernel  the roofline denominator: independent FMA chains.
#pragma once

#include <stdint.h>

#include "rt_math.cuh"

namespace rt {

// Tuning knobs (defaults chosen by measurement on B200, profiles/r1_tuning.md).
#ifndef RT_TRACE_BLOCK
#define RT_TRACE_BLOCK 128
#endif
#ifndef RT_MIN_BLOCKS
#define RT_MIN_BLOCKS 4       // <= 128 registers per thread: 16 warps per SM
#endif
#ifndef RT_GRID_ROLLED
#define RT_GRID_ROLLED 1      // grid equilibrium: one copy of the stage code (stage loop not unrolled)
#endif
constexpr int TRACE_BLOCK = RT_TRACE_BLOCK;

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

template <class T, int EQ, int DISP, class Gather>
RT_DEV int rk4_step(const Params<T>& P, T h, T* y, Gather& gather) {
  const T hh = T(0.5) * h, h6 = h * T(1.0 / 6.0), h3 = h * T(1.0 / 3.0);
  T k[6], acc[6], ys[6];
  bool ok = true;
  if (EQ == EQ_GRID && RT_GRID_ROLLED) {
#pragma unroll
    for (int j = 0; j < 6; ++j) { k[j] = T(0); acc[j] = y[j]; }
#pragma unroll 1
    for (int st = 0; st < 4; ++st) {
      const T a = (st == 0) ? T(0) : ((st == 3) ? h : hh);
      const T w = (st == 0 || st == 3) ? h6 : h3;
#pragma unroll
      for (int j = 0; j < 6; ++j) ys[j] = rt_fma(a, k[j], y[j]);
      ok = ray_rhs<T, EQ, DISP>(P, ys, k, gather) && ok;
#pragma unroll
      for (int j = 0; j < 6; ++j) acc[j] = rt_fma(w, k[j], acc[j]);
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) ys[j] = acc[j];
  } else {
#pragma unroll
    for (int j = 0; j < 6; ++j) { ys[j] = y[j]; acc[j] = y[j]; }
    ok = ray_rhs<T, EQ, DISP>(P, y, k, gather);
#pragma unroll
    for (int j = 0; j < 6; ++j)
      if (rhs_component_active<EQ>(j)) { acc[j] = rt_fma(h6, k[j], y[j]); ys[j] = rt_fma(hh, k[j], y[j]); }
    ok = ray_rhs<T, EQ, DISP>(P, ys, k, gather) && ok;
#pragma unroll
    for (int j = 0; j < 6; ++j)
      if (rhs_component_active<EQ>(j)) { acc[j] = rt_fma(h3, k[j], acc[j]); ys[j] = rt_fma(hh, k[j], y[j]); }
    ok = ray_rhs<T, EQ, DISP>(P, ys, k, gather) && ok;
#pragma unroll
    for (int j = 0; j < 6; ++j)
      if (rhs_component_active<EQ>(j)) { acc[j] = rt_fma(h3, k[j], acc[j]); ys[j] = rt_fma(h, k[j], y[j]); }
    ok = ray_rhs<T, EQ, DISP>(P, ys, k, gather) && ok;
#pragma unroll
    for (int j = 0; j < 6; ++j) ys[j] = rhs_component_active<EQ>(j) ? rt_fma(h6, k[j], acc[j]) : y[j];
  }
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
  bool inside;
  const T D = ray_D<T, EQ, DISP>(P, y, &inside, gather);
  return inside ? rt_abs(D) : rt_nan<T>();
}

#ifdef __CUDACC__

// Shared-memory cell cache of the grid equilibrium.  A ray moves ~1 mm per RK4 step through 5.9 mm cells, so the 16
// psi pieces (one 128-B line in fp64) and the 8 profile pieces it needs are the same for many consecutive stages.  Read
// straight from global memory, every 128-bit load of a warp touches 32 different lines and the L1 data pipe saturates
// (99.8 % `l1tex__data_pipe_lsu_wavefronts`, FP64 pipe 43 %: profiles/r1_cfg5_ncu.md).  Here each thread keeps its
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

template <class T, int BLOCK>
struct GatherCached {
  typedef typename Vec16<T>::type V;
  static constexpr int PSI_CHUNKS = 16 * sizeof(T) / 16, PROF_CHUNKS = 8 * sizeof(T) / 16;
  static constexpr int CHUNKS = PSI_CHUNKS + PROF_CHUNKS;
  V* col;                  // this thread's column: chunk j at col[j * BLOCK]
  int cell, pcell;         // cached cell indices (-1: nothing cached)
  RT_DEV void psi_select(const Params<T>& P, int c) {
    if (c != cell) {
      const V* g = reinterpret_cast<const V*>(P.psi_pp + (size_t)c * 16);
#pragma unroll
      for (int j = 0; j < PSI_CHUNKS; ++j) col[j * BLOCK] = __ldg(g + j);
      cell = c;
    }
  }
  RT_DEV void prof_select(const Params<T>& P, int c) {
    if (c != pcell) {
      const V* g = reinterpret_cast<const V*>(P.prof_pp + (size_t)c * 8);
#pragma unroll
      for (int j = 0; j < PROF_CHUNKS; ++j) col[(PSI_CHUNKS + j) * BLOCK] = __ldg(g + j);
      pcell = c;
    }
  }
  RT_DEV void psi_row(const Params<T>&, int, int p, T* c) const { unpack4(col, p, BLOCK, c); }
  RT_DEV void prof_row(const Params<T>&, int, int which, T* c) const { unpack4(col + PSI_CHUNKS * BLOCK, which, BLOCK, c); }
};

template <class T, int EQ> struct TraceGather { typedef GatherDirect type; };
template <class T> struct TraceGather<T, EQ_GRID> { typedef GatherCached<T, TRACE_BLOCK> type; };

template <class T, int EQ, int DISP>
__global__ void __launch_bounds__(TRACE_BLOCK, RT_MIN_BLOCKS)
trace_kernel(const __grid_constant__ Params<T> P, const __grid_constant__ TraceArgs<T> A) {
  const long long N = A.n_rays;
  const long long i = (long long)blockIdx.x * TRACE_BLOCK + threadIdx.x;
  typename TraceGather<T, EQ>::type gather;
  if constexpr (EQ == EQ_GRID) {
    typedef GatherCached<T, TRACE_BLOCK> GC;
    __shared__ typename GC::V cache[GC::CHUNKS * TRACE_BLOCK];
    gather.col = cache + threadIdx.x;
    gather.cell = -1; gather.pcell = -1;
  }
  if (i >= N) return;
  T y[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    y[c] = A.x0[c * N + i];
    y[3 + c] = A.k0[c * N + i] * P.k2n;          // n = c k / w  (Eq. 6)
  }
  int status = 0;
  long long m = 0;                                 // next trajectory sample
  if (A.traj) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      A.traj[(m * 6 + c) * N + i] = y[c];
      A.traj[(m * 6 + 3 + c) * N + i] = y[3 + c] * P.n2k;
    }
    if (A.res) A.res[m * N + i] = abs_residual<T, EQ, DISP>(P, y, gather);
    ++m;
  }
  long long countdown = A.stride;
  for (long long s = 0; s < A.n_steps; ++s) {
    if (status == 0) status = rk4_step<T, EQ, DISP>(P, A.h, y, gather);
    if (A.traj && --countdown == 0) {
      countdown = A.stride;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        A.traj[(m * 6 + c) * N + i] = y[c];
        A.traj[(m * 6 + 3 + c) * N + i] = y[3 + c] * P.n2k;
      }
      if (A.res) A.res[m * N + i] = abs_residual<T, EQ, DISP>(P, y, gather);
      ++m;
    }
  }
  if (A.fin) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      A.fin[c * N + i] = y[c];
      A.fin[(3 + c) * N + i] = y[3 + c] * P.n2k;
    }
  }
  if (!A.traj && A.res) A.res[i] = abs_residual<T, EQ, DISP>(P, y, gather);
  if (A.status) A.status[i] = status;
}

template <class T, int EQ, int DISP>
__global__ void __launch_bounds__(TRACE_BLOCK)
rhs_kernel(const __grid_constant__ Params<T> P, const T* __restrict__ x, const T* __restrict__ k, long long n,
           T* __restrict__ D_out, T* __restrict__ rhs_out, int32_t* __restrict__ inside_out) {
  const long long i = (long long)blockIdx.x * TRACE_BLOCK + threadIdx.x;
  if (i >= n) return;
  T y[6], f[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) { y[c] = x[c * n + i]; y[3 + c] = k[c * n + i] * P.k2n; }
  GatherDirect gather;
  const bool inside = ray_rhs<T, EQ, DISP>(P, y, f, gather);
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
template <int EQ, int DISP>
__global__ void __launch_bounds__(TRACE_BLOCK)
launch_kernel(const __grid_constant__ Params<double> P, int branch, const double* __restrict__ x0,
              const double* __restrict__ dir, long long n, double* __restrict__ k0, double* __restrict__ D_out) {
  const long long i = (long long)blockIdx.x * TRACE_BLOCK + threadIdx.x;
  if (i >= n) return;
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

// Roofline denominator: FMA_CHAINS independent accumulators per thread, each a dependent chain of fused multiply-adds.
// The chain is acc = acc * a + acc (two distinct source registers): with three distinct 64-bit sources the DFMA rate
// drops from 63.7 to 58.8 per clock per SM on B200 (register-bank conflicts; measured, profiles/r1_fma_peak_shapes.md).
constexpr int FMA_CHAINS = 16;
constexpr int FMA_BLOCK = 256;
template <class T>
__global__ void __launch_bounds__(FMA_BLOCK)
fma_peak_kernel(T* __restrict__ sink, long long iters, T a, unsigned long long* __restrict__ clk) {
  T acc[FMA_CHAINS];
#pragma unroll
  for (int j = 0; j < FMA_CHAINS; ++j) acc[j] = T(threadIdx.x + j) * T(1e-3);
  unsigned long long t0, t1;
  const long long c0 = clock64();
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t0));
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < FMA_CHAINS; ++j) acc[j] = acc[j] * a + acc[j];
    }
  }
  const long long c1 = clock64();
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t1));
  T s = T(0);
#pragma unroll
  for (int j = 0; j < FMA_CHAINS; ++j) s += acc[j];
  sink[(long long)blockIdx.x * FMA_BLOCK + threadIdx.x] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) { clk[0] = (unsigned long long)(c1 - c0); clk[1] = t1 - t0; }
}

#endif  // __CUDACC__

}  // namespace rt
