// rt_math.cuh -- per-stage arithmetic of the ray tracer: equilibrium -> dispersion partials -> ray RHS.
//
// Everything here is hand-derived and templated on the scalar type T (double / float), the
// equilibrium kind EQ and the dispersion kind DISP, so that each kernel instantiation contains only the arithmetic
// its combination needs.  State variables are x [m] and n = c k / w (Eq. 6); the independent
// variable is tau = c t.  In these variables the ray equations (Eq. 2-3) read
//
//      dx/dtau = -(dD/dn) / W ,    dn/dtau = +(dD/dx) / W ,    W = w dD/dw at fixed (x, k).
//
// D depends on (x, n, w) only through four scalars:
//      X  = wpe^2/w^2 = xs * shape(x)                     (electron; the ion's X_i = mu X, mu = Z m_e/m_i)
//      Y2 = (Wce/w)^2 = beta |B|^2                        (ion: Y_i^2 = mu^2 Y2)
//      u  = n_par^2   = (n.B)^2/|B|^2
//      v  = n^2
// and under w -> lambda w at fixed (x, k) all four scale as lambda^-2, hence W = -2 s, s = X D_X + Y2 D_Y2 + u D_u + v D_v.
//
// The hot path never forms D's gradient vectors and divides them by W component by component.  With r = 1/s, G = n.B:
//      dx/dtau = A n + C B ,                         A = D_v r,            C = (G/|B|^2) D_u r
//      dn/dtau = Ax (grad X)/2 + Ab (grad |B|^2)/2 - C grad_x(n.B)|_n ,
//                                                    Ax = -D_X r,          Ab = -(beta D_Y2 - u D_u/|B|^2) r
// so the reciprocal is folded into four scalars (disp_coefs) before anything multiplies a vector, and every structural
// zero of an equilibrium (slab: only d/dx; axisymmetric: no d/dphi of X and |B|^2) is skipped at compile time -- the
// FP64 pipe is the roofline of this path, so the instruction count per stage is what is optimised.
#pragma once

#include <math.h>

#ifdef __CUDACC__
#define RT_DEV __device__ __forceinline__
#else
#define RT_DEV inline
#endif

namespace rt {

// EQ_TOKAMAK is the circular tokamak with the configs' density exponent p_exp = 3/2 (evaluated as t sqrt(t));
// EQ_TOKAMAK_POW is the same equilibrium with a general exponent (pow).  Both come from RT_EQ_TOKAMAK_CIRCULAR.
enum { EQ_PARABOLIC = 0, EQ_LINEAR = 1, EQ_TOKAMAK = 2, EQ_GRID = 3, EQ_TOKAMAK_POW = 4 };
enum { DISP_O = 0, DISP_X = 1, DISP_FULL = 2 };

// Per-call constants, folded on the host in fp64 (step a0, rt_params.h) so that every device-side quantity is O(1) in
// fp32 too.
template <class T>
struct Params {
  T xs;         // X = xs * shape(x):  alpha n_ref (analytic kinds) or alpha ne_scale (grid), alpha = e^2/(eps0 m_e w^2)
  T xsh;        // xs / 2 (the hot loop carries HALF the gradient of X, see Local::hgX)
  T beta;       // Y_e^2 = beta |B|^2, beta = (e/(m_e w))^2
  T beta2;      // 2 beta
  T mu;         // Z m_e / m_i; 0 = electrons only
  T mu2, mu3, mu4, one_plus_mu;
  T y2cap;      // the ion terms' series (disp_coefs, SERIES) is exact to rounding for Y2 < y2cap (rt_params.h: series_cap)
  T k2n, n2k;   // c/w and w/c
  // slab_parabolic:  X = xs + par_g (x^2 + y^2)
  T par_g;      // xs / L^2
  // slab_linear_br:  X = (x - x_foot) lin_gx
  T x_foot, lin_gx, B0R0;   // lin_gx = -xs / L_ramp
  T lin_gxh;                // lin_gx / 2
  // analytic fields in units of the electron cyclotron ratio: sB0 = sqrt(beta) B0, sB0R0 = sqrt(beta) B0 R0, so that
  // |B'|^2 IS Y2 = (Wce/w)^2 and no beta multiplies anything in the hot loop (ray_rhs, SCALED)
  T sB0, sB0R0;
  // tokamak_circular
  T R0, B0, inv_a2, q0, q1_a2, two_q1_a2, p_exp, rmax2;   // q = q0 + q1_a2 r^2;  domain r^2 < rmax2 = (rho_max a)^2
  T two_xs_a2;  // 2 xs / a^2
  T tok_gxh;    // -p_exp xs / a^2:  (1/2) grad X = tok_gxh (1 - rho^2)^(p_exp - 1) (dR, 0, Z)
  // grid_rz
  T Rmin, Rmax, Zmin, Zmax, hR, hZ, inv_hR, inv_hZ, psi_min, psi_max, hP, inv_hP;
  int nRc, nZc, nPc;            // cell counts
  const T* psi_pp;              // [nRc][nZc][4][4]: psi = sum c[p][q] dR^p dZ^q
  const T* prof_pp;             // [nPc][8]: F = sum f[m] ds^m (m = 0..3), then n_e/ne_scale likewise
};

#ifdef __CUDACC__
struct f32x2;
template <> struct Params<f32x2> : Params<float> {      // the packed kernels take the scalar constants (broadcast at use)
  Params() = default;
  RT_DEV Params(const Params<float>& p) : Params<float>(p) {}
};
#endif

RT_DEV int rt_imin(int a, int b) { return a < b ? a : b; }
RT_DEV double rt_sqrt(double a) { return sqrt(a); }
RT_DEV float rt_sqrt(float a) { return sqrtf(a); }
RT_DEV double rt_pow(double a, double b) { return pow(a, b); }
RT_DEV float rt_pow(float a, float b) { return powf(a, b); }
RT_DEV double rt_floor(double a) { return floor(a); }
RT_DEV float rt_floor(float a) { return floorf(a); }
RT_DEV double rt_abs(double a) { return fabs(a); }
RT_DEV float rt_abs(float a) { return fabsf(a); }
RT_DEV double rt_fma(double a, double b, double c) { return fma(a, b, c); }
RT_DEV float rt_fma(float a, float b, float c) { return fmaf(a, b, c); }
RT_DEV bool rt_finite(double a) { return isfinite(a); }
RT_DEV bool rt_finite(float a) { return isfinite(a); }
template <class T> RT_DEV T rt_nan();
template <> RT_DEV double rt_nan<double>() { return nan(""); }
template <> RT_DEV float rt_nan<float>() { return nanf(""); }

// Reciprocal and reciprocal square root for the hot loop.  An IEEE fp64 division costs ~10 FP64-pipe instructions plus
// a slow-path branch; here the 20-bit MUFU seed is refined by ONE third-order Newton step (3 / 5 FMA-pipe instructions,
// branch-free), which leaves a relative error below 2^-52 for the normal, O(1) arguments of this path -- far inside
// the 1e-10 parity budget.  NaN propagates; zero / negative arguments give inf / NaN, which only
// occur at points outside the equilibrium's domain, whose results are discarded (reading A12).
#ifdef __CUDACC__
RT_DEV double rt_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);          // e = 1 - x r,  |e| <~ 2^-20
  return fma(r, fma(e, e, e), r);            // r (1 + e + e^2)
}
RT_DEV double rt_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x * y, y, 1.0);      // e = 1 - x y^2
  return y * fma(e, fma(0.375, e, 0.5), 1.0);  // y (1 + e/2 + 3 e^2/8)
}
RT_DEV float rt_rcp(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
RT_DEV float rt_rsqrt(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
// sqrt(x) from the same seed without forming 1/sqrt(x) first: g = x y, e = 1 - g y, sqrt = g (1 + e/2 + 3 e^2/8)
// (2 MUL + 3 FMA; one instruction fewer than x * rt_rsqrt(x)).
RT_DEV double rt_sqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double g = x * y;
  const double e = fma(-g, y, 1.0);
  return g * fma(e, fma(0.375, e, 0.5), 1.0);
}
RT_DEV float rt_sqrt_fast(float x) { return x * rt_rsqrt(x); }
// Domain tests of the fp64 hot loop as INTEGER comparisons of the bit patterns (a DSETP occupies the FP64 pipe, which is
// the roofline of this path; the ALU pipe is idle).  Exactly equivalent to the floating-point comparisons they replace:
//   rt_less_nonneg(a, b), a >= +0 or NaN, b > 0 finite:  a < b  <=>  bits(a) < bits(b) as unsigned (a NaN of either sign
//   has a larger pattern than any finite positive number);
//   rt_positive(a):  a > 0  <=>  0 < bits(a) <= bits(+inf)  <=>  (unsigned)(bits(a) - 1) < bits(+inf).
RT_DEV bool rt_less_nonneg(double a, double b) {
  return (unsigned long long)__double_as_longlong(a) < (unsigned long long)__double_as_longlong(b);
}
RT_DEV bool rt_less_nonneg(float a, float b) { return a < b; }
RT_DEV bool rt_positive(double a) {
  return (unsigned long long)(__double_as_longlong(a) - 1LL) < 0x7ff0000000000000ULL;
}
RT_DEV bool rt_positive(float a) { return a > 0.0f; }
#else
template <class T> RT_DEV T rt_rcp(T x) { return T(1) / x; }
template <class T> RT_DEV T rt_rsqrt(T x) { return T(1) / rt_sqrt(x); }
template <class T> RT_DEV T rt_sqrt_fast(T x) { return rt_sqrt(x); }
template <class T> RT_DEV bool rt_less_nonneg(T a, T b) { return a < b; }
template <class T> RT_DEV bool rt_positive(T a) { return a > T(0); }
#endif

// ---- two rays per thread in fp32: packed f32x2 arithmetic (sm_100a FFMA2 / FMUL2 / FADD2) ---------------------------
// The fp32 trace kernels are issue-bound, not FMA-pipe-bound (every FFMA takes a whole issue slot, and every MUFU seed,
// integer and LDS instruction displaces one), and an FFMA that reads three distinct registers occupies the pipe for 1.56
// slots.  A packed FFMA2 does the same arithmetic for TWO rays in ONE issue slot and two pipe cycles (127.9 FMA per clock
// per SM against 123.2 scalar; with three distinct register operands 84.9 against 78.8: profiles/r2_fma_peak_shapes.md),
// which moves the kernels from issue-bound to FMA-pipe-bound.
// f32x2 holds one value of ray A (low half) and of ray B (high half); every operation is the IEEE fp32 operation on
// each half, so a ray's result does not depend on which thread half it rides in.  A scalar (per-call constant)
// converts implicitly: ptxas turns the broadcast into a `.F32` operand of the packed instruction.  Negation and |x| are
// written per half so that ptxas folds them into operand modifiers.  Per-half predicates and integers are mask2 / int2v.
template <class T> struct Lane { typedef bool mask; typedef int index; typedef T scalar; static constexpr int N = 1; };
#ifdef __CUDACC__
struct f32x2 {
  unsigned long long v;
  f32x2() = default;
  RT_DEV f32x2(float s) { asm("mov.b64 %0, {%1, %1};" : "=l"(v) : "f"(s)); }
  RT_DEV explicit f32x2(double s) : f32x2((float)s) {}
  RT_DEV explicit f32x2(int s) : f32x2((float)s) {}
  RT_DEV f32x2(float lo, float hi) { asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(lo), "f"(hi)); }
  RT_DEV float lo() const { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return a; }
  RT_DEV float hi() const { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return b; }
};
struct mask2 { bool a, b; };
struct int2v { int a, b; };
template <> struct Lane<f32x2> { typedef mask2 mask; typedef int2v index; typedef float scalar; static constexpr int N = 2; };
RT_DEV f32x2 operator+(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
RT_DEV f32x2 operator-(f32x2 a, f32x2 b) { f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
RT_DEV f32x2 operator*(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
RT_DEV f32x2 operator-(f32x2 a) { return f32x2(-a.lo(), -a.hi()); }
RT_DEV f32x2& operator*=(f32x2& a, f32x2 b) { a = a * b; return a; }
RT_DEV f32x2 rt_fma(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return d;
}
RT_DEV f32x2 rt_abs(f32x2 a) { return f32x2(fabsf(a.lo()), fabsf(a.hi())); }
RT_DEV f32x2 rt_floor(f32x2 a) { return f32x2(floorf(a.lo()), floorf(a.hi())); }
RT_DEV f32x2 rt_pow(f32x2 a, f32x2 b) { return f32x2(powf(a.lo(), b.lo()), powf(a.hi(), b.hi())); }
RT_DEV f32x2 rt_sqrt(f32x2 a) { return f32x2(sqrtf(a.lo()), sqrtf(a.hi())); }
template <> RT_DEV f32x2 rt_nan<f32x2>() { return f32x2(nanf("")); }
RT_DEV f32x2 rt_rcp(f32x2 x) { return f32x2(rt_rcp(x.lo()), rt_rcp(x.hi())); }
RT_DEV f32x2 rt_rsqrt(f32x2 x) { return f32x2(rt_rsqrt(x.lo()), rt_rsqrt(x.hi())); }
RT_DEV f32x2 rt_sqrt_fast(f32x2 x) { return x * rt_rsqrt(x); }
RT_DEV mask2 rt_finite(f32x2 a) { return {isfinite(a.lo()), isfinite(a.hi())}; }
RT_DEV mask2 rt_less_nonneg(f32x2 a, f32x2 b) { return {a.lo() < b.lo(), a.hi() < b.hi()}; }
RT_DEV mask2 rt_positive(f32x2 a) { return {a.lo() > 0.0f, a.hi() > 0.0f}; }
RT_DEV mask2 operator>=(f32x2 a, f32x2 b) { return {a.lo() >= b.lo(), a.hi() >= b.hi()}; }
RT_DEV mask2 operator<=(f32x2 a, f32x2 b) { return {a.lo() <= b.lo(), a.hi() <= b.hi()}; }
RT_DEV mask2 rt_and(mask2 x, mask2 y) { return {x.a && y.a, x.b && y.b}; }
RT_DEV mask2 rt_not(mask2 x) { return {!x.a, !x.b}; }
RT_DEV bool rt_all(mask2 x) { return x.a && x.b; }
RT_DEV f32x2 rt_select(mask2 m, f32x2 x, f32x2 y) { return f32x2(m.a ? x.lo() : y.lo(), m.b ? x.hi() : y.hi()); }
RT_DEV int2v rt_select(mask2 m, int2v x, int y) { return {m.a ? x.a : y, m.b ? x.b : y}; }
RT_DEV int2v rt_floor_int(f32x2 a) { return {(int)floorf(a.lo()), (int)floorf(a.hi())}; }
RT_DEV int2v rt_imin(int2v a, int b) { return {rt_imin(a.a, b), rt_imin(a.b, b)}; }
RT_DEV int2v operator*(int2v a, int b) { return {a.a * b, a.b * b}; }
RT_DEV int2v operator+(int2v a, int2v b) { return {a.a + b.a, a.b + b.b}; }
template <class T> RT_DEV T rt_from_index(int2v i) { return f32x2((float)i.a, (float)i.b); }
#endif
template <class T> RT_DEV typename Lane<T>::mask rt_true() { return true; }
#ifdef __CUDACC__
template <> RT_DEV mask2 rt_true<f32x2>() { return {true, true}; }
#endif
RT_DEV bool rt_and(bool x, bool y) { return x && y; }
RT_DEV bool rt_all(bool x) { return x; }
RT_DEV bool rt_not(bool x) { return !x; }
template <class T> RT_DEV T rt_select(bool m, T x, T y) { return m ? x : y; }
RT_DEV int rt_floor_int(double a) { return (int)rt_floor(a); }
RT_DEV int rt_floor_int(float a) { return (int)rt_floor(a); }
template <class T> RT_DEV T rt_from_index(int i) { return T(i); }

#ifdef __CUDACC__
RT_DEV void ld16(const double* p, double& a, double& b) {
  const double2 t = __ldg(reinterpret_cast<const double2*>(p));
  a = t.x; b = t.y;
}
RT_DEV void ld4(const double* p, double* c) { ld16(p, c[0], c[1]); ld16(p + 2, c[2], c[3]); }
RT_DEV void ld4(const float* p, float* c) {
  const float4 t = __ldg(reinterpret_cast<const float4*>(p));
  c[0] = t.x; c[1] = t.y; c[2] = t.z; c[3] = t.w;
}
#else
template <class T> RT_DEV void ld4(const T* p, T* c) { for (int i = 0; i < 4; ++i) c[i] = p[i]; }
#endif

// How the grid equilibrium fetches a cell's spline pieces.  GatherDirect reads the global tables (diagnostic kernels,
// launch solver, host builds); the trace kernel passes a shared-memory cell cache instead (rt_kernels.cuh: GatherCached).
struct GatherDirect {
  template <class T, class I> RT_DEV bool psi_request(const Params<T>&, I) { return false; }
  template <class T, class I> RT_DEV bool prof_request(const Params<T>&, I) { return false; }
  RT_DEV void wait() {}
  template <class T> RT_DEV void psi_row(const Params<T>& P, int cell, int p, T* c) const { ld4(P.psi_pp + (size_t)cell * 16 + 4 * p, c); }
  template <class T> RT_DEV void prof_row(const Params<T>& P, int cell, int which, T* c) const { ld4(P.prof_pp + (size_t)cell * 8 + 4 * which, c); }
#ifdef __CUDACC__
  // per-half look-ups of the packed type (the grid branch of equilibrium<> has to compile for every T; the packed trace
  // kernel of the grid equilibrium does its look-ups per ray in scalar arithmetic instead: grid_values_per_ray)
  RT_DEV void psi_row(const Params<f32x2>& P, int2v cell, int p, f32x2* c) const {
    float a[4], b[4];
    ld4(P.psi_pp + (size_t)cell.a * 16 + 4 * p, a); ld4(P.psi_pp + (size_t)cell.b * 16 + 4 * p, b);
    for (int j = 0; j < 4; ++j) c[j] = f32x2(a[j], b[j]);
  }
  RT_DEV void prof_row(const Params<f32x2>& P, int2v cell, int which, f32x2* c) const {
    float a[4], b[4];
    ld4(P.prof_pp + (size_t)cell.a * 8 + 4 * which, a); ld4(P.prof_pp + (size_t)cell.b * 8 + 4 * which, b);
    for (int j = 0; j < 4; ++j) c[j] = f32x2(a[j], b[j]);
  }
#endif
};

// Cubic c0 + c1 s + c2 s^2 + c3 s^3 with its first derivative and HALF its second derivative in 6 fused multiply-adds
// (Horner's scheme, the derivative chains reusing the partial sums).
template <class T>
RT_DEV void cubic012(const T* c, T s, T& f, T& f1, T& f2h) {
  const T b1 = rt_fma(c[3], s, c[2]);
  const T b0 = rt_fma(b1, s, c[1]);
  f = rt_fma(b0, s, c[0]);
  const T d1 = rt_fma(c[3], s, b1);        // 2 c3 s + c2
  f1 = rt_fma(d1, s, b0);                  // 3 c3 s^2 + 2 c2 s + c1
  f2h = rt_fma(c[3], s, d1);               // 3 c3 s + c2
}
template <class T>
RT_DEV void cubic01(const T* c, T s, T& f, T& f1) {
  const T b1 = rt_fma(c[3], s, c[2]);
  const T b0 = rt_fma(b1, s, c[1]);
  f = rt_fma(b0, s, c[0]);
  f1 = rt_fma(rt_fma(c[3], s, b1), s, b0);
}

// Horner steps that share their multiplier, issued back to back.  An FP64 instruction that reads three distinct registers
// from the register file occupies the FP64 pipe for 3 cycles instead of 2; an operand found in the
// operand-reuse cache (the same register in the same slot of the preceding instruction) does not count.  The spline
// evaluation is made of Horner steps x * s + y with the SAME s (the offset inside the cell) for four rows at a time:
// written as volatile asm in row-interleaved order, ptxas keeps them adjacent with s in one slot and flags it `.reuse`,
// so every step after the first reads two registers.  (Plain C++ leaves the order to the scheduler, which spreads them.)
#ifdef __CUDACC__
RT_DEV double rt_fma_s(double x, double s, double y) {
  double d;
  asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(x), "d"(s), "d"(y));
  return d;
}
template <class T> RT_DEV T rt_fma_s(T x, T s, T y) { return rt_fma(x, s, y); }
#else
template <class T> RT_DEV T rt_fma_s(T x, T s, T y) { return rt_fma(x, s, y); }
#endif
// N cubics c[p][0..3] at the same argument s: value, first derivative and (D2) half the second derivative, level by level
// across the N polynomials (same arithmetic as cubic012 / cubic01 on each).
template <class T, int N, bool D2>
RT_DEV void cubics_at(const T (*c)[4], T s, T* f, T* f1, T* f2h) {
  T b1[N], b0[N], d1[N];
#pragma unroll
  for (int p = 0; p < N; ++p) b1[p] = rt_fma_s(c[p][3], s, c[p][2]);
#pragma unroll
  for (int p = 0; p < N; ++p) b0[p] = rt_fma_s(b1[p], s, c[p][1]);
#pragma unroll
  for (int p = 0; p < N; ++p) d1[p] = rt_fma_s(c[p][3], s, b1[p]);         // 2 c3 s + c2
#pragma unroll
  for (int p = 0; p < N; ++p) f[p] = rt_fma_s(b0[p], s, c[p][0]);
#pragma unroll
  for (int p = 0; p < N; ++p) f1[p] = rt_fma_s(d1[p], s, b0[p]);           // 3 c3 s^2 + 2 c2 s + c1
  if (D2) {
#pragma unroll
    for (int p = 0; p < N; ++p) f2h[p] = rt_fma_s(c[p][3], s, d1[p]);      // 3 c3 s + c2
  }
}

// ---- Stix elements (Eq. 8-10) as functions of X, Y2 ------------------------------------------
//   S = 1 - X sig,  sig = 1/(1-Y2) + mu/(1-mu^2 Y2)
//   Dx^2 = X^2 Y2 del^2,  del = mu^2/(1-mu^2 Y2) - 1/(1-Y2)      (eps12 = -i Dx; only Dx^2 enters D)
//   P = 1 - X (1 + mu)
template <class T>
struct StixT {
  T s, p, d2;            // S, P, Dx^2
  T sig, sigp, del, delp;  // sig, d sig/dY2, del, d del/dY2
};

template <class T>
RT_DEV StixT<T> stix(const Params<T>& P, T X, T Y2) {
  StixT<T> st;
  const T e1 = rt_rcp(T(1) - Y2);
  const T e2 = rt_rcp(T(1) - P.mu2 * Y2);
  const T e1s = e1 * e1, e2s = e2 * e2;
  st.sig = e1 + P.mu * e2;
  st.sigp = e1s + P.mu3 * e2s;
  st.del = P.mu2 * e2 - e1;
  st.delp = P.mu4 * e2s - e1s;
  st.s = T(1) - X * st.sig;
  st.p = T(1) - X * P.one_plus_mu;
  st.d2 = X * X * Y2 * st.del * st.del;
  return st;
}

// D(X, Y2, u, v) -- the value reported as the residual.  Not rescaled (reading A4).
//   O:    D = v - 1 + X                                     (BASELINE.json config 1)
//   X:    D = S v - (S^2 - Dx^2)                             (reading A5: S n^2 - R L)
//   full: D = (P - v + u)[(S - u)(S - v) - Dx^2] - (v - u) u (S - v)    (Eq. 5 expanded in the field frame)
//           = (P - v + u) RL + S [(v - u) v - P (v + u)] + P u v ,   RL = S^2 - Dx^2
template <class T, int DISP>
RT_DEV T disp_value(const Params<T>& P, T X, T Y2, T u, T v) {
  if (DISP == DISP_O) return v - T(1) + X;
  const StixT<T> st = stix(P, X, Y2);
  const T RL = st.s * st.s - st.d2;
  if (DISP == DISP_X) return st.s * v - RL;
  const T w = v - u;
  return (st.p - w) * RL + st.s * (w * v - st.p * (v + u)) + st.p * u * v;
}

// Partials of D with respect to (X, Y2, u, v) in their plain form (launch solver and diagnostics; the hot loop uses
// disp_coefs below).
template <class T, int DISP>
RT_DEV void disp_partials(const Params<T>& P, T X, T Y2, T u, T v, T& DX, T& DY2, T& Du, T& Dv) {
  if (DISP == DISP_O) { DX = T(1); DY2 = T(0); Du = T(0); Dv = T(1); return; }
  const StixT<T> st = stix(P, X, Y2);
  const T s = st.s, p = st.p;
  T Ds, Dp, Dd2;
  if (DISP == DISP_X) {
    Ds = v - T(2) * s; Dp = T(0); Dd2 = T(1);
    Du = T(0); Dv = s;
  } else {
    const T RL = s * s - st.d2;
    const T w = v - u;
    Du = RL - s * (v + p) + p * v;
    Dv = -RL + s * (v + w - p) + p * u;
    Ds = T(2) * s * (p - w) + w * v - p * (v + u);
    Dp = RL - s * (v + u) + u * v;
    Dd2 = w - p;
  }
  const T XYd = X * Y2 * st.del;
  DX = -st.sig * Ds - P.one_plus_mu * Dp + T(2) * XYd * st.del * Dd2;
  DY2 = -X * st.sigp * Ds + X * X * st.del * (st.del + T(2) * Y2 * st.delp) * Dd2;
}

// ---- the four scalars of the ray RHS (header comment) for the magnetised dispersion functions --------------------
// Reverse-mode differentiation of  D = pw ab - t b,  w = v - u, pw = P - w, a = S - u, b = S - v, ab = a b - Dx^2,
// t = w u  (the full determinant above), or of D = S v - S^2 + Dx^2 (X-mode):
//   D_S = pw b + (pw a - t),  D_P = ab,  D_{Dx^2} = -pw,  D_w = -(ab + b u),  D_v = D_w - (pw a - t),
//   D_u = -b w - pw b - D_w.
// With S_X = -sig, P_X = -(1+mu), (Dx^2)_X = q1 = 2 X Y2 del^2, S_Y2 = -X sig', (Dx^2)_Y2 = q2 = X^2 del (del + 2 Y2 del'):
//   -D_X = DXn = sig D_S + (1+mu) D_P + q1 pw ,     -D_Y2 = DYn = X sig' D_S + q2 pw.
// The coefficients are returned WITHOUT the common factor r = 1/s (Coef::r): rk4_step folds r into the step-size
// factors (two multiplications per stage instead of one per coefficient), ray_rhs_scaled applies it for the diagnostics.
template <class T>
struct Coef {
  T A, C, Ax, Ab, r;
  T YD;                              // Y2 DYn
  typename Lane<T>::mask fast;       // SERIES: Y2 < Params::y2cap, i.e. the series of the ion terms is exact to rounding here
};

// SC: the caller's field is already in units of sqrt(beta) (Params::sB0), i.e. b2 IS Y2 and Ab multiplies (1/2) grad Y2.
// Ax multiplies HALF the gradient of X (Local::hgX), which is where the 1/2 of the header comment has gone.
template <class T, int DISP, bool SC, bool SERIES>
RT_DEV Coef<T> disp_coefs(const Params<T>& P, T X, T b2, T G, T v) {
  const T Y2 = SC ? b2 : P.beta * b2, Y22 = SC ? b2 + b2 : P.beta2 * b2;
  const T e1 = rt_rcp(T(1) - Y2);
  const T e1s = e1 * e1;
  T sig, sigp, del, delp;
  Coef<T> c;
  if (SERIES) {
    // Ion terms by their series in z = mu^2 Y2 (mu = Z m_e/m_i <= 5.4e-4): e2 = 1/(1 - z) = 1 + z + z^2 + ..., so
    //   mu e2 = mu + mu^3 Y2 + O(mu z^2),  mu^3 e2^2 = mu^3 + O(mu^3 z),  mu^2 e2 = mu^2 + mu^4 Y2 + O(mu^2 z^2),
    //   mu^4 e2^2 = mu^4 + O(mu^4 z);
    // for Y2 < y2cap (folded on the host so that every dropped term is below a quarter ulp of the sum it enters) this is
    // the rounded exact value: one reciprocal and three FP instructions per stage fewer.  A stage with Y2 >= y2cap clears
    // c.fast and the caller repeats the step with SERIES = false.
    c.fast = rt_less_nonneg(Y2, T(P.y2cap));
    sig = e1 + rt_fma(P.mu3, Y2, P.mu);
    sigp = e1s + P.mu3;
    del = rt_fma(P.mu4, Y2, P.mu2) - e1;
    delp = P.mu4 - e1s;
  } else {
    c.fast = rt_true<T>();
    const T e2 = rt_rcp(rt_fma(-P.mu2, Y2, T(1)));
    const T e2s = e2 * e2;
    sig = rt_fma(P.mu, e2, e1);
    sigp = rt_fma(P.mu3, e2s, e1s);
    del = rt_fma(P.mu2, e2, -e1);
    delp = rt_fma(P.mu4, e2s, -e1s);
  }
  const T S = rt_fma(-X, sig, T(1));
  const T Xd = X * del;
  const T XdY22 = Xd * Y22;                          // 2 X Y2 del
  const T q1 = XdY22 * del;
  const T q2 = (Xd * X) * rt_fma(Y22, delp, del);
  const T Xsp = X * sigp;
  if (DISP == DISP_X) {
    const T DS = rt_fma(T(-2), S, v);
    const T DXn = rt_fma(sig, DS, -q1);
    const T DYn = rt_fma(Xsp, DS, -q2);
    c.YD = Y2 * DYn;
    const T s = rt_fma(v, S, -rt_fma(X, DXn, c.YD));
    c.r = rt_rcp(s);
    c.A = S;
    c.C = T(0);
    c.Ax = DXn;
    c.Ab = SC ? DYn : P.beta * DYn;
  } else {
    const T d2 = (T(0.5) * Xd) * XdY22;
    const T Pp = rt_fma(-X, P.one_plus_mu, T(1));
    const T Bc = G * rt_rcp(b2);
    const T u = G * Bc;
    const T w = v - u, pw = Pp - w, a = S - u, b = S - v;
    const T ab = rt_fma(a, b, -d2);
    const T pb = pw * b;
    const T pat = rt_fma(pw, a, -(w * u));
    const T DS = pb + pat;
    const T Dw = -rt_fma(b, u, ab);
    const T Du = rt_fma(-b, w, -pb) - Dw;
    const T Dv = Dw - pat;
    const T DXn = rt_fma(q1, pw, rt_fma(P.one_plus_mu, ab, sig * DS));
    const T DYn = rt_fma(q2, pw, Xsp * DS);
    c.YD = Y2 * DYn;
    const T s = rt_fma(v, Dv, rt_fma(u, Du, -rt_fma(X, DXn, c.YD)));
    c.r = rt_rcp(s);
    c.A = Dv;
    c.C = Bc * Du;
    c.Ax = DXn;
    c.Ab = SC ? rt_fma(Bc, c.C, DYn) : rt_fma(Bc, c.C, P.beta * DYn);
  }
  return c;
}

// ---- equilibrium at one stage point, in a local orthonormal frame ------------------------------------------------
// Frame: (e1, e2, e3) = (R^, phi^, Z^) for the axisymmetric kinds, Cartesian for the slabs.  Only the entries an
// equilibrium can make non-zero are written (and read): slabs vary along e1 = x only; axisymmetric X and |B|^2 have no
// e2 = phi derivative.  gG = grad_x (n.B) at fixed Cartesian n, hgb2 = (1/2) grad |B|^2, hgX = (1/2) grad X.
// SC (analytic kinds only): B is returned in units of 1/sqrt(beta), i.e. B' = sqrt(beta) B with |B'|^2 = Y2; the ray
// right-hand side is invariant under this scaling once beta is dropped from disp_coefs (C' B' = C B, C' grad(n.B') =
// C grad(n.B), Ab' grad Y2 = Ab grad |B|^2), and it removes three multiplications per stage.
template <class T>
struct Local {
  T X, hgX[3];   // X and HALF its gradient
  T B[3], b2, hgb2[3], G, gG[3];
  T ix;          // linear slab: 1/x
  T nl[3];       // n in the local frame
  T cph, sph;    // axisymmetric kinds: e1 = (cph, sph, 0), e2 = (-sph, cph, 0)
};

template <int EQ> struct is_axisym { static constexpr bool value = (EQ == EQ_TOKAMAK || EQ == EQ_TOKAMAK_POW || EQ == EQ_GRID); };

// Tail of the grid equilibrium: B = (-psi_Z, F, psi_R)/R and its derivatives from psi's and F's.  With
// Q = psi_R^2 + psi_Z^2 + F^2 = R^2 |B|^2 and g = -n_R psi_Z + n_phi F + n_Z psi_R = R (n.B):
//   (1/2) grad|B|^2 = (Q_R/2, Q_Z/2)/R^2 - (|B|^2/R) R^ ,   grad_x(n.B) = ((g_R - n.B)/R, (n_phi B_R - n_R B_phi)/R, g_Z/R).
// psiRRh / psiZZh are HALF the second derivatives.
template <class T, int DISP>
RT_DEV void axisym_field(T iR, T psiR, T psiZ, T psiRRh, T psiRZ, T psiZZh, T F, T Fp, Local<T>& L) {
  if (DISP == DISP_O) return;
  const T iR2 = iR * iR;
  const T Q = rt_fma(F, F, rt_fma(psiR, psiR, psiZ * psiZ));
  L.b2 = Q * iR2;
  const T psiRR = psiRRh + psiRRh, psiZZ = psiZZh + psiZZh;
  const T FFp = F * Fp;
  const T hQR = rt_fma(FFp, psiR, rt_fma(psiR, psiRR, psiZ * psiRZ));
  const T hQZ = rt_fma(FFp, psiZ, rt_fma(psiR, psiRZ, psiZ * psiZZ));
  L.hgb2[0] = rt_fma(hQR, iR2, -L.b2 * iR);
  L.hgb2[2] = hQZ * iR2;
  if (DISP == DISP_FULL) {
    const T nR = L.nl[0], nP = L.nl[1], nZ = L.nl[2];
    L.B[0] = -psiZ * iR; L.B[1] = F * iR; L.B[2] = psiR * iR;
    const T g = rt_fma(nZ, psiR, rt_fma(nP, F, -nR * psiZ));
    L.G = g * iR;
    const T nPFp = nP * Fp;
    const T gR = rt_fma(nZ, psiRR, rt_fma(nPFp, psiR, -nR * psiRZ));
    const T gZ = rt_fma(nZ, psiRZ, rt_fma(nPFp, psiZ, -nR * psiZZ));
    L.gG[0] = (gR - L.G) * iR;
    L.gG[1] = -rt_fma(nP, psiZ, nR * F) * iR2;
    L.gG[2] = gZ * iR;
  }
}

// ---- grid equilibrium: the spline look-ups at one point (config 5) -------------------------------------
// psi(R, Z) bicubic with its first and second derivatives, then F(psi), n_e(psi) cubic with their first derivatives
// (n_e in units of Params::xs / alpha, i.e. X = xs Ne).  psiRRh / psiZZh are HALF the second derivatives.
template <class T>
struct GridVals { T psiR, psiZ, psiRRh, psiRZ, psiZZh, F, Fp, Ne, Nep; };

// The look-up in four parts, so that a caller with several rays in flight (the packed kernel, below) can issue every ray's
// cell-cache refill before it waits for any of them:
//   grid_psi_cell   cell index and offsets of (R, Z), rectangle test          -> gather.psi_request(cell) [+ gather.wait()]
//   grid_psi_eval   psi and its derivatives from the cell's 16 pieces, psi-range test
//   grid_prof_cell  profile cell index and offset of psi                      -> gather.prof_request(cell) [+ gather.wait()]
//   grid_prof_eval  F, F', n_e, n_e' from the profile cell's 8 pieces
template <class T>
RT_DEV typename Lane<T>::index grid_psi_cell(const Params<T>& P, T R, T Z, typename Lane<T>::mask& inside, T& dR, T& dZ) {
  // R > 0 is implied by R >= Rmin: rt_create_equilibrium requires Rmin > 0.  Inside the rectangle R - Rmin >= +0 exactly,
  // so the cell index is >= 0 and only needs the upper clamp (R = Rmax belongs to the last cell); outside -- including NaN
  // positions, which convert to unspecified ints -- the index is forced to 0 to keep the gather in bounds.
  typedef typename Lane<T>::index I;
  inside = rt_and(rt_and(R >= T(P.Rmin), R <= T(P.Rmax)), rt_and(Z >= T(P.Zmin), Z <= T(P.Zmax)));
  const T Ro = R - P.Rmin, Zo = Z - P.Zmin;                       // offsets from the grid's corner
  I iRc = rt_imin(rt_floor_int(Ro * P.inv_hR), P.nRc - 1);
  I iZc = rt_imin(rt_floor_int(Zo * P.inv_hZ), P.nZc - 1);
  iRc = rt_select(inside, iRc, 0); iZc = rt_select(inside, iZc, 0);
  // offset inside the cell: (R - Rmin) - i hR in one fused step (i hR is exact in the fma; the oracle's R - (Rmin + i hR)
  // differs by a rounding of R)
  dR = rt_fma(-rt_from_index<T>(iRc), T(P.hR), Ro); dZ = rt_fma(-rt_from_index<T>(iZc), T(P.hZ), Zo);
  return iRc * P.nZc + iZc;
}

template <class T, int DISP, class Gather>
RT_DEV T grid_psi_eval(const Params<T>& P, typename Lane<T>::index cell, T dR, T dZ, Gather& gather, GridVals<T>& V) {
  T a[4], a1[4], a2h[4];   // a_p(dZ) = sum_q c[p][q] dZ^q, its first dZ-derivative and half its second
  T psi, psiR, psiRRh = T(0), psiZ, psiRZ = T(0), psiZZh = T(0);
  if (sizeof(T) == 8 && DISP != DISP_O) {
    // fp64: the 24 + 13 Horner steps grouped by their multiplier (dZ, then dR), see rt_fma_s
    T c[4][4];
#pragma unroll
    for (int p = 0; p < 4; ++p) gather.psi_row(P, cell, p, c[p]);
    cubics_at<T, 4, true>(c, dZ, a, a1, a2h);
    const T b1 = rt_fma_s(a[3], dR, a[2]), e1 = rt_fma_s(a1[3], dR, a1[2]), g1 = rt_fma_s(a2h[3], dR, a2h[2]);
    const T b0 = rt_fma_s(b1, dR, a[1]), e0 = rt_fma_s(e1, dR, a1[1]), g0 = rt_fma_s(g1, dR, a2h[1]);
    const T d1 = rt_fma_s(a[3], dR, b1), h1 = rt_fma_s(a1[3], dR, e1);
    psi = rt_fma_s(b0, dR, a[0]); psiZ = rt_fma_s(e0, dR, a1[0]); psiZZh = rt_fma_s(g0, dR, a2h[0]);
    psiR = rt_fma_s(d1, dR, b0); psiRZ = rt_fma_s(h1, dR, e0);
    psiRRh = rt_fma_s(a[3], dR, d1);
  } else {
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      T c[4];
      gather.psi_row(P, cell, p, c);
      if (DISP == DISP_O) cubic01(c, dZ, a[p], a1[p]);
      else cubic012(c, dZ, a[p], a1[p], a2h[p]);
    }
    if (DISP == DISP_O) {
      cubic01(a, dR, psi, psiR);
      psiZ = rt_fma(rt_fma(rt_fma(a1[3], dR, a1[2]), dR, a1[1]), dR, a1[0]);
    } else {
      cubic012(a, dR, psi, psiR, psiRRh);
      cubic01(a1, dR, psiZ, psiRZ);
      psiZZh = rt_fma(rt_fma(rt_fma(a2h[3], dR, a2h[2]), dR, a2h[1]), dR, a2h[0]);
    }
  }
  V.psiR = psiR; V.psiZ = psiZ; V.psiRRh = psiRRh; V.psiRZ = psiRZ; V.psiZZh = psiZZh;
  return psi;
}

template <class T>
RT_DEV typename Lane<T>::index grid_prof_cell(const Params<T>& P, T psi, typename Lane<T>::mask& inside, T& ds) {
  typedef typename Lane<T>::index I;
  inside = rt_and(inside, rt_and(psi >= T(P.psi_min), psi <= T(P.psi_max)));
  const T po = psi - P.psi_min;
  I iP = rt_imin(rt_floor_int(po * P.inv_hP), P.nPc - 1);                        // same argument: psi >= psi_min when inside
  iP = rt_select(inside, iP, 0);
  ds = rt_fma(-rt_from_index<T>(iP), T(P.hP), po);
  return iP;
}

template <class T, int DISP, class Gather>
RT_DEV void grid_prof_eval(const Params<T>& P, typename Lane<T>::index iP, T ds, Gather& gather, GridVals<T>& V) {
  T Ne, Nep, F = T(0), Fp = T(0);
  if (sizeof(T) == 8 && DISP != DISP_O) {
    T pq[2][4], v[2], v1[2];
    gather.prof_row(P, iP, 1, pq[0]);
    gather.prof_row(P, iP, 0, pq[1]);
    cubics_at<T, 2, false>(pq, ds, v, v1, v);
    Ne = v[0]; Nep = v1[0]; F = v[1]; Fp = v1[1];
  } else {
    T g[4];
    gather.prof_row(P, iP, 1, g);
    cubic01(g, ds, Ne, Nep);
    if (DISP != DISP_O) {
      T f[4];
      gather.prof_row(P, iP, 0, f);
      cubic01(f, ds, F, Fp);
    }
  }
  V.F = F; V.Fp = Fp; V.Ne = Ne; V.Nep = Nep;
}

template <class T, int DISP, class Gather>
RT_DEV typename Lane<T>::mask grid_splines(const Params<T>& P, T R, T Z, Gather& gather, GridVals<T>& V) {
  typename Lane<T>::mask inside;
  T dR, dZ, ds;
  const typename Lane<T>::index cell = grid_psi_cell(P, R, Z, inside, dR, dZ);
  if (gather.psi_request(P, cell)) gather.wait();
  const T psi = grid_psi_eval<T, DISP>(P, cell, dR, dZ, gather, V);
  const typename Lane<T>::index iP = grid_prof_cell(P, psi, inside, ds);
  if (gather.prof_request(P, iP)) gather.wait();
  grid_prof_eval<T, DISP>(P, iP, ds, gather, V);
  return inside;
}

// How grid_full_rhs reaches the spline look-ups.  Normally the look-ups run in the caller's lane type.  The packed fp32 trace
// kernel of the grid equilibrium (rt_kernels.cuh: trace_kernel_x2<EQ_GRID>) instead does them PER RAY in scalar arithmetic,
// each ray with its own shared-memory cell cache, and packs the nine results: the pieces of a cell come out of shared
// memory as four consecutive registers per row, which suits scalar Horner steps as they are, whereas packed Horner steps
// would need every piece paired with the other ray's first (measured: ~100 register moves per stage, profiles/r2_tuning.md).
template <class G> struct gather_is_pair { static constexpr bool value = false; };
template <class T, int DISP, class Gather>
RT_DEV typename Lane<T>::mask grid_values(const Params<T>& P, T R, T Z, Gather& gather, GridVals<T>& V) {
  return grid_splines<T, DISP>(P, R, Z, gather, V);
}
#ifdef __CUDACC__
template <int DISP, class Pair>
RT_DEV mask2 grid_values_per_ray(const Params<f32x2>& P, f32x2 R, f32x2 Z, Pair& gather, GridVals<f32x2>& V) {
  const Params<float>& Pf = P;
  GridVals<float> a, b;
  bool ina, inb;
  float dRa, dZa, dRb, dZb, dsa, dsb;
  // both rays' refills are in flight before the thread waits for either (a refill is a round trip to L2)
  const int ca = grid_psi_cell(Pf, R.lo(), Z.lo(), ina, dRa, dZa), cb = grid_psi_cell(Pf, R.hi(), Z.hi(), inb, dRb, dZb);
  gather.a.psi_request(Pf, ca); gather.b.psi_request(Pf, cb);
  gather.a.wait();                 // unconditionally: a branch around it costs more than the empty wait (264 against 276 ms)
  const float psia = grid_psi_eval<float, DISP>(Pf, ca, dRa, dZa, gather.a, a);
  const int pa = grid_prof_cell(Pf, psia, ina, dsa);
  gather.a.prof_request(Pf, pa);
  const float psib = grid_psi_eval<float, DISP>(Pf, cb, dRb, dZb, gather.b, b);
  const int pb = grid_prof_cell(Pf, psib, inb, dsb);
  gather.b.prof_request(Pf, pb);
  gather.b.wait();
  grid_prof_eval<float, DISP>(Pf, pa, dsa, gather.a, a);
  grid_prof_eval<float, DISP>(Pf, pb, dsb, gather.b, b);
  V.psiR = f32x2(a.psiR, b.psiR); V.psiZ = f32x2(a.psiZ, b.psiZ); V.psiRRh = f32x2(a.psiRRh, b.psiRRh);
  V.psiRZ = f32x2(a.psiRZ, b.psiRZ); V.psiZZh = f32x2(a.psiZZh, b.psiZZh);
  V.F = f32x2(a.F, b.F); V.Fp = f32x2(a.Fp, b.Fp); V.Ne = f32x2(a.Ne, b.Ne); V.Nep = f32x2(a.Nep, b.Nep);
  return mask2{ina, inb};
}
#endif

template <class T, int EQ, int DISP, bool SC = false, class Gather>
RT_DEV typename Lane<T>::mask equilibrium(const Params<T>& P, const T* x, const T* n, Local<T>& L, Gather& gather) {
  typedef typename Lane<T>::mask M;
  if (EQ == EQ_PARABOLIC) {
    // X = xs (1 + (x^2+y^2)/L^2)                                          (BASELINE.json config 1)
    L.X = rt_fma(P.par_g, rt_fma(x[0], x[0], x[1] * x[1]), P.xs);
    return rt_true<T>();                                                   // everywhere; grad X = 2 par_g (x, y, 0): see ray_rhs
  }
  if (EQ == EQ_LINEAR) {
    // n_e = n_ref (x_foot - x)/L_ramp ;  B = (B0 R0 / x) z^                (config 3; Eq. 4 profile)
    const M inside = rt_positive(x[0]);
    L.X = (x[0] - P.x_foot) * P.lin_gx;                                    // grad X = (lin_gx, 0, 0)
    if (DISP != DISP_O) {
      const T ix = rt_rcp(x[0]);
      L.ix = ix;
      const T Bz = (SC ? P.sB0R0 : P.B0R0) * ix;
      L.B[2] = Bz;
      L.b2 = Bz * Bz;
      L.hgb2[0] = -L.b2 * ix;
      if (DISP == DISP_FULL) {
        L.G = n[2] * Bz;
        L.gG[0] = -L.G * ix;
      }
    }
    return inside;
  }
  // axisymmetric kinds: cylindrical frame at the point
  const T R2 = rt_fma(x[0], x[0], x[1] * x[1]);
  const T iR = rt_rsqrt(R2);
  const T R = R2 * iR;
  const T Z = x[2];
  L.cph = x[0] * iR; L.sph = x[1] * iR;
  if (DISP == DISP_FULL) {
    L.nl[0] = rt_fma(n[0], L.cph, n[1] * L.sph);
    L.nl[1] = rt_fma(n[1], L.cph, -n[0] * L.sph);
    L.nl[2] = n[2];
  }
  if (EQ == EQ_TOKAMAK || EQ == EQ_TOKAMAK_POW) {
    // psi'(r) = B0 r / q, q = q0 + q1 rho^2, F = B0 R0, n_e = n_ref (1 - rho^2)^p       (config 4; reading A9)
    const T dR = R - P.R0;
    const T r2 = rt_fma(dR, dR, Z * Z);
    // r^2 < (rho_max a)^2 implies R > 0 because rt_create_equilibrium requires a < R0 and rho_max < 1
    const M inside = rt_less_nonneg(r2, T(P.rmax2));
    const T t = rt_fma(-P.inv_a2, r2, T(1));                               // 1 - rho^2
    T gx;                                                                  // (1/2) grad X = gx (dR, 0, Z)
    if (EQ == EQ_TOKAMAK) {
      const T sq = rt_sqrt_fast(t);
      L.X = (P.xs * sq) * t;
      gx = P.tok_gxh * sq;
    } else {
      const T pw = rt_pow(t, P.p_exp - T(1));
      L.X = (P.xs * pw) * t;
      gx = P.tok_gxh * pw;
    }
    L.hgX[0] = gx * dR; L.hgX[2] = gx * Z;
    if (DISP != DISP_O) {
      // B = (-h Z, g, h dR), h = B0/(q R), g = B0 R0/R; with e = 1/R + c dR, c = q'/q = 2 q1/(a^2 q):
      //   h_R = -h e, h_Z = -h c Z, g_R = -g/R.
      const T iq = rt_rcp(rt_fma(P.q1_a2, r2, P.q0));
      const T h = ((SC ? P.sB0 : P.B0) * iq) * iR;
      const T g = (SC ? P.sB0R0 : P.B0R0) * iR;
      const T c = P.two_q1_a2 * iq;
      const T e = rt_fma(c, dR, iR);
      const T h2 = h * h, g2 = g * g;
      const T giR = g * iR;
      L.b2 = rt_fma(h2, r2, g2);                                           // |B|^2 = h^2 r^2 + g^2
      L.hgb2[0] = rt_fma(h2, rt_fma(-r2, e, dR), -g * giR);                // h^2 (dR - r^2 e) - g^2/R
      L.hgb2[2] = (h2 * Z) * rt_fma(-c, r2, T(1));                         // h^2 Z (1 - c r^2)
      if (DISP == DISP_FULL) {
        const T nR = L.nl[0], nP = L.nl[1], nZ = L.nl[2];
        L.B[0] = -h * Z; L.B[1] = g; L.B[2] = h * dR;
        const T m = rt_fma(nZ, dR, -nR * Z);
        L.G = rt_fma(h, m, g * nP);
        L.gG[0] = rt_fma(-nP, giR, h * rt_fma(-e, m, nZ));                 // h (n_Z - e m) - n_phi g/R
        L.gG[1] = rt_fma(nP, L.B[0], -nR * g) * iR;                        // (n_phi B_R - n_R B_phi)/R
        L.gG[2] = -h * rt_fma(c * Z, m, nR);                               // -h (n_R + c Z m)
      }
    }
    return inside;
  }
  // EQ_GRID: bicubic psi(R,Z), cubic F(psi), n_e(psi)                                    (config 5)
  GridVals<T> V;
  const M inside = grid_splines<T, DISP>(P, R, Z, gather, V);
  L.X = P.xs * V.Ne;
  const T gx = P.xsh * V.Nep;
  L.hgX[0] = gx * V.psiR; L.hgX[2] = gx * V.psiZ;
  if (DISP != DISP_O) axisym_field<T, DISP>(iR, V.psiR, V.psiZ, V.psiRRh, V.psiRZ, V.psiZZh, V.F, V.Fp, L);
  return inside;
}

// ---- the full determinant over the analytic tokamak (config 4, the headline kernel), written out ------------------
// Same mathematics as equilibrium<EQ_TOKAMAK, DISP_FULL, SC> + disp_coefs + the generic assembly of ray_rhs, with the
// products shared between the field, its gradients and the assembly formed once (6 FP64 instructions fewer per stage).
// With h = sqrt(beta) B0/(q R), g = sqrt(beta) B0 R0/R, c = q'/q, e = 1/R + c dR, m = n_Z dR - n_R Z (header of
// equilibrium<>):  B' = (-h Z, g, h dR),  (1/2) grad Y2 = (h^2 (dR - r^2 e) - g^2/R, 0, h^2 Z (1 - c r^2)),
// grad_x(n.B') = (h (n_Z - e m) - n_phi g/R, (n_phi B'_R - n_R g)/R, -h (n_R + c Z m)),  (1/2) grad X = gx (dR, 0, Z).  Then
//   f_R = Ax gx dR + Ab h^2 (dR - r^2 e) + (g/R)(C n_phi - Ab g) - C h (n_Z - e m)
//   f_Z = Z (Ax gx + Ab h^2 (1 - c r^2)) + C h (n_R + c Z m)
//   f_phi = (n_phi (C h Z) + n_R (C g)) / R
//   f_x = A n + C B':  C B'_R = -(C h) Z,  C B'_phi = C g,  C B'_Z = (C h) dR.
template <class T, int EQ, bool SERIES>
RT_DEV typename Lane<T>::mask tokamak_full_rhs(const Params<T>& P, const T* y, T* f, T& r, typename Lane<T>::mask& fast) {
  const T* n = y + 3;
  const T R2 = rt_fma(y[0], y[0], y[1] * y[1]);
  const T iR = rt_rsqrt(R2);
  const T R = R2 * iR;
  const T Z = y[2];
  const T cph = y[0] * iR, sph = y[1] * iR;
  const T nR = rt_fma(n[0], cph, n[1] * sph);
  const T nP = rt_fma(n[1], cph, -n[0] * sph);
  const T nZ = n[2];
  const T dR = R - P.R0;
  const T r2 = rt_fma(dR, dR, Z * Z);
  const typename Lane<T>::mask inside = rt_less_nonneg(r2, T(P.rmax2));   // implies R > 0 (a < R0, rho_max < 1)
  const T t = rt_fma(-P.inv_a2, r2, T(1));                       // 1 - rho^2
  T X, gx;
  if (EQ == EQ_TOKAMAK) {
    const T sq = rt_sqrt_fast(t);
    X = (P.xs * sq) * t;
    gx = P.tok_gxh * sq;
  } else {
    const T pw = rt_pow(t, P.p_exp - T(1));
    X = (P.xs * pw) * t;
    gx = P.tok_gxh * pw;
  }
  const T iq = rt_rcp(rt_fma(P.q1_a2, r2, P.q0));
  const T h = (P.sB0 * iq) * iR;
  const T g = P.sB0R0 * iR;
  const T c = P.two_q1_a2 * iq;
  const T h2 = h * h;
  const T Y2 = rt_fma(h2, r2, g * g);
  const T m = rt_fma(nZ, dR, -nR * Z);
  const T G = rt_fma(h, m, g * nP);
  const T v = rt_fma(n[0], n[0], rt_fma(n[1], n[1], n[2] * n[2]));
  const Coef<T> k = disp_coefs<T, DISP_FULL, true, SERIES>(P, X, Y2, G, v);
  r = k.r;
  fast = rt_and(fast, k.fast);
  const T Axg = k.Ax * gx, Abh2 = k.Ab * h2, Ch = k.C * h, Cg = k.C * g, ChZ = Ch * Z;
  const T ze = rt_fma(-c, r2, T(1));                             // 1 - c r^2
  const T K = rt_fma(Ch, c * m, rt_fma(Abh2, ze, Axg));          // Ax gx + Ab h^2 (1 - c r^2) + C h c m
  const T fR = rt_fma(dR, K, rt_fma(-iR, k.YD, -Ch * nZ));
  f[5] = rt_fma(Z, K, Ch * nR);
  const T fP = rt_fma(nP, ChZ, nR * Cg) * iR;
  f[3] = rt_fma(fR, cph, -fP * sph);
  f[4] = rt_fma(fR, sph, fP * cph);
  f[0] = rt_fma(-ChZ, cph, rt_fma(-Cg, sph, k.A * n[0]));
  f[1] = rt_fma(-ChZ, sph, rt_fma(Cg, cph, k.A * n[1]));
  f[2] = rt_fma(Ch, dR, k.A * n[2]);
  return inside;
}

// ---- the full determinant over the grid equilibrium (config 5), assembly written out ------------------------------------
// Same mathematics as equilibrium<EQ_GRID, DISP_FULL> + axisym_field + disp_coefs + the generic assembly of ray_rhs; the
// products C/R, Ab/R^2 and Ax gx that the field, its gradients and the assembly share are formed once (5 FP instructions
// per stage fewer).  With Q = psi_R^2 + psi_Z^2 + F^2 = R^2 |B|^2, g = n_Z psi_R + n_phi F - n_R psi_Z = R (n.B),
// hQ_R = F F' psi_R + psi_R psi_RR + psi_Z psi_RZ = (1/2) dQ/dR (hQ_Z likewise), g_R, g_Z the derivatives of g at fixed n:
//   f_R = Ax gx psi_R + (Ab/R^2) hQ_R - (Ab |B|^2 + C (g_R - n.B))/R ,   f_Z = Ax gx psi_Z + (Ab/R^2) hQ_Z - (C/R) g_Z ,
//   f_phi = (C/R) (n_phi psi_Z + n_R F)/R ,   C B = (C/R)(-psi_Z, F, psi_R).
template <class T, bool SERIES, class Gather>
RT_DEV typename Lane<T>::mask grid_full_rhs(const Params<T>& P, const T* y, T* f, T& r, Gather& gather, typename Lane<T>::mask& fast) {
  const T* n = y + 3;
  const T R2 = rt_fma(y[0], y[0], y[1] * y[1]);
  const T iR = rt_rsqrt(R2);
  const T R = R2 * iR;
  const T cph = y[0] * iR, sph = y[1] * iR;
  const T nR = rt_fma(n[0], cph, n[1] * sph);
  const T nP = rt_fma(n[1], cph, -n[0] * sph);
  const T nZ = n[2];
  GridVals<T> V;
  typename Lane<T>::mask inside;
#ifdef __CUDACC__
  if constexpr (gather_is_pair<Gather>::value) inside = grid_values_per_ray<DISP_FULL>(P, R, y[2], gather, V);
  else
#endif
    inside = grid_values<T, DISP_FULL>(P, R, y[2], gather, V);
  const T X = P.xs * V.Ne, gx = P.xsh * V.Nep;
  const T iR2 = iR * iR;
  const T Q = rt_fma(V.F, V.F, rt_fma(V.psiR, V.psiR, V.psiZ * V.psiZ));
  const T b2 = Q * iR2;
  const T psiRR = V.psiRRh + V.psiRRh, psiZZ = V.psiZZh + V.psiZZh;
  const T FFp = V.F * V.Fp;
  const T hQR = rt_fma(FFp, V.psiR, rt_fma(V.psiR, psiRR, V.psiZ * V.psiRZ));
  const T hQZ = rt_fma(FFp, V.psiZ, rt_fma(V.psiR, V.psiRZ, V.psiZ * psiZZ));
  const T g = rt_fma(nZ, V.psiR, rt_fma(nP, V.F, -nR * V.psiZ));
  const T G = g * iR;
  const T nPFp = nP * V.Fp;
  const T gR = rt_fma(nZ, psiRR, rt_fma(nPFp, V.psiR, -nR * V.psiRZ));
  const T gZ = rt_fma(nZ, V.psiRZ, rt_fma(nPFp, V.psiZ, -nR * psiZZ));
  const T v = rt_fma(n[0], n[0], rt_fma(n[1], n[1], n[2] * n[2]));
  const Coef<T> k = disp_coefs<T, DISP_FULL, false, SERIES>(P, X, b2, G, v);
  r = k.r;
  fast = rt_and(fast, k.fast);
  const T Ci = k.C * iR, Ai2 = k.Ab * iR2, Axg = k.Ax * gx;
  const T t2 = rt_fma(k.C, gR, k.YD);                            // C (g_R - n.B) + Ab |B|^2 = C g_R + Y2 DYn (Ab = beta DYn + C (n.B)/|B|^2)
  const T fR = rt_fma(Axg, V.psiR, rt_fma(Ai2, hQR, -iR * t2));
  f[5] = rt_fma(Axg, V.psiZ, rt_fma(Ai2, hQZ, -Ci * gZ));
  const T fP = (Ci * iR) * rt_fma(nP, V.psiZ, nR * V.F);
  f[3] = rt_fma(fR, cph, -fP * sph);
  f[4] = rt_fma(fR, sph, fP * cph);
  const T xR = -Ci * V.psiZ, xP = Ci * V.F;
  f[0] = rt_fma(xR, cph, rt_fma(-xP, sph, k.A * n[0]));
  f[1] = rt_fma(xR, sph, rt_fma(xP, cph, k.A * n[1]));
  f[2] = rt_fma(Ci, V.psiR, k.A * n[2]);
  return inside;
}

// ---- one evaluation of the ray right-hand side, y = (x, n) --------------------------------------------------------
// Returns the right-hand side as (f, r): dy/dtau = r f, r = 1/s the reciprocal of the header comment.  Returns false
// (and f, r unspecified) if x is outside the equilibrium's domain.
// SERIES: the ion terms of the Stix elements by their series (disp_coefs); `fast` is cleared (never set) if a point lies
// outside the series' range, in which case the caller has to repeat the evaluation with SERIES = false.
template <class T, int EQ, int DISP, bool SERIES, class Gather>
RT_DEV typename Lane<T>::mask ray_rhs(const Params<T>& P, const T* y, T* f, T& r, Gather& gather, typename Lane<T>::mask& fast) {
  Local<T> L;
  const T* n = y + 3;
  if (EQ == EQ_PARABOLIC) {
    // O-mode in X = xs + par_g (x^2 + y^2) (config 1-2), written out so that the two products par_g x, par_g y serve
    // both grad X / 2 and X itself:  s = v + X = n_x^2 + n_y^2 + (par_g x) x + (par_g y) y + (n_z^2 + xs), whose last
    // term is constant along the ray (dn_z/dtau = 0).
    const T gx = P.par_g * y[0], gy = P.par_g * y[1];
    const T base = rt_fma(n[2], n[2], P.xs);
    r = rt_rcp(rt_fma(n[0], n[0], rt_fma(n[1], n[1], rt_fma(gx, y[0], rt_fma(gy, y[1], base)))));
    f[0] = n[0]; f[1] = n[1]; f[2] = n[2];
    f[3] = -gx; f[4] = -gy; f[5] = T(0);
    return rt_true<T>();
  }
  if constexpr ((EQ == EQ_TOKAMAK || EQ == EQ_TOKAMAK_POW) && DISP == DISP_FULL) {
    return tokamak_full_rhs<T, EQ, SERIES>(P, y, f, r, fast);
  } else if constexpr (EQ == EQ_GRID && DISP == DISP_FULL) {
    return grid_full_rhs<T, SERIES>(P, y, f, r, gather, fast);
  } else {
    constexpr bool SC = (EQ != EQ_GRID);      // analytic fields come in units of 1/sqrt(beta); the grid's table is in tesla
    const typename Lane<T>::mask inside = equilibrium<T, EQ, DISP, SC>(P, y, n, L, gather);
    const T v = rt_fma(n[0], n[0], rt_fma(n[1], n[1], n[2] * n[2]));
    if (DISP == DISP_O) {
      // D = v - 1 + X:  dD/dn = 2 n, dD/dx = grad X, W = -2 (v + X)   =>   dx/dtau = n r, dn/dtau = -grad X r/2, r = 1/(v+X)
      r = rt_rcp(v + L.X);
      f[0] = n[0]; f[1] = n[1]; f[2] = n[2];
      if (EQ == EQ_LINEAR) {
        f[3] = -P.lin_gxh; f[4] = T(0); f[5] = T(0);
      } else {
        const T fR = -L.hgX[0];
        f[3] = fR * L.cph; f[4] = fR * L.sph; f[5] = -L.hgX[2];
      }
      return inside;
    }
    const Coef<T> c = disp_coefs<T, DISP, SC, SERIES>(P, L.X, L.b2, (DISP == DISP_FULL) ? L.G : T(0), v);
    r = c.r;
    fast = rt_and(fast, c.fast);
    f[0] = c.A * n[0]; f[1] = c.A * n[1]; f[2] = c.A * n[2];               // A n is frame-independent
    if (EQ == EQ_LINEAR) {
      // B = (c/x) z^:  (1/2) d|B'|^2/dx = -Y2/x and d(n.B')/dx = -(n.B')/x, so the curvature terms collapse as in
      // tokamak_full_rhs:  Ab (1/2) dY2/dx - C d(n.B')/dx = -(Ab Y2 - C (n.B'))/x = -Y2 DYn / x
      if (DISP == DISP_FULL) f[2] = rt_fma(c.C, L.B[2], f[2]);
      f[3] = rt_fma(-c.YD, L.ix, c.Ax * P.lin_gxh); f[4] = T(0); f[5] = T(0);
      return inside;
    }
    // axisymmetric kinds: assemble in (R^, phi^, Z^), rotate to Cartesian
    T fR = rt_fma(c.Ab, L.hgb2[0], c.Ax * L.hgX[0]);
    T fZ = rt_fma(c.Ab, L.hgb2[2], c.Ax * L.hgX[2]);
    if (DISP == DISP_FULL) {
      const T xR = c.C * L.B[0], xP = c.C * L.B[1];
      f[0] = rt_fma(xR, L.cph, rt_fma(-xP, L.sph, f[0]));
      f[1] = rt_fma(xR, L.sph, rt_fma(xP, L.cph, f[1]));
      f[2] = rt_fma(c.C, L.B[2], f[2]);
      fR = rt_fma(-c.C, L.gG[0], fR);
      fZ = rt_fma(-c.C, L.gG[2], fZ);
      const T fP = -c.C * L.gG[1];
      f[3] = rt_fma(fR, L.cph, -fP * L.sph);
      f[4] = rt_fma(fR, L.sph, fP * L.cph);
    } else {
      f[3] = fR * L.cph; f[4] = fR * L.sph;
    }
    f[5] = fZ;
    return inside;
  }
}

// dy/dtau itself (diagnostics: rt_rhs), evaluated the way the trace kernels do it: with the ion series first, exactly if the
// point is outside the series' range
template <class T, int EQ, int DISP, class Gather>
RT_DEV typename Lane<T>::mask ray_rhs_scaled(const Params<T>& P, const T* y, T* f, Gather& gather) {
  T r;
  typename Lane<T>::mask fast = rt_true<T>();
  typename Lane<T>::mask inside = ray_rhs<T, EQ, DISP, true>(P, y, f, r, gather, fast);
  if (!rt_all(fast)) inside = ray_rhs<T, EQ, DISP, false>(P, y, f, r, gather, fast);
#pragma unroll
  for (int j = 0; j < 6; ++j) f[j] *= r;
  return inside;
}

// signed D at y = (x, n); *inside reports the domain test
template <class T, int EQ, int DISP, class Gather>
RT_DEV T ray_D(const Params<T>& P, const T* y, typename Lane<T>::mask* inside, Gather& gather) {
  Local<T> L;
  *inside = equilibrium<T, EQ, DISP>(P, y, y + 3, L, gather);
  const T v = y[3] * y[3] + y[4] * y[4] + y[5] * y[5];
  if (DISP == DISP_O) return disp_value<T, DISP>(P, L.X, T(0), T(0), v);
  const T u = (DISP == DISP_FULL) ? L.G * L.G * rt_rcp(L.b2) : T(0);
  return disp_value<T, DISP>(P, L.X, P.beta * L.b2, u, v);
}

}  // namespace rt
