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
// and under w -> lambda w at fixed (x, k) all four scale as lambda^-2, hence W = -2 (X D_X + Y2 D_Y2 + u D_u + v D_v).
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

// Per-call constants, folded on the host in fp64 (step a0) so that every device-side quantity is O(1) in fp32 too.
template <class T>
struct Params {
  T xs;         // X = xs * shape(x):  alpha n_ref (analytic kinds) or alpha ne_scale (grid), alpha = e^2/(eps0 m_e w^2)
  T beta;       // Y_e^2 = beta |B|^2, beta = (e/(m_e w))^2
  T mu;         // Z m_e / m_i; 0 = electrons only
  T mu2, mu3, mu4, one_plus_mu;
  T k2n, n2k;   // c/w and w/c
  // slab_parabolic
  T inv_L2;
  // slab_linear_br
  T x_foot, inv_Lramp, B0R0;
  // tokamak_circular
  T R0, B0, inv_a2, q0, q1, two_q1_a2, p_exp, rho_max2;
  T two_xs_a2;  // 2 xs / a^2
  // grid_rz
  T Rmin, Rmax, Zmin, Zmax, hR, hZ, inv_hR, inv_hZ, psi_min, psi_max, hP, inv_hP;
  int nRc, nZc, nPc;            // cell counts
  const T* psi_pp;              // [nRc][nZc][4][4]: psi = sum c[p][q] dR^p dZ^q
  const T* prof_pp;             // [nPc][8]: F = sum f[m] ds^m (m = 0..3), then n_e/ne_scale likewise
};

RT_DEV double rt_sqrt(double a) { return sqrt(a); }
RT_DEV float rt_sqrt(float a) { return sqrtf(a); }
RT_DEV double rt_pow(double a, double b) { return pow(a, b); }
RT_DEV float rt_pow(float a, float b) { return powf(a, b); }
RT_DEV double rt_floor(double a) { return floor(a); }
RT_DEV float rt_floor(float a) { return floorf(a); }
RT_DEV double rt_abs(double a) { return fabs(a); }
RT_DEV float rt_abs(float a) { return fabsf(a); }
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
  return fma(y * e, fma(0.375, e, 0.5), y);  // y (1 + e/2 + 3 e^2/8)
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
#else
template <class T> RT_DEV T rt_rcp(T x) { return T(1) / x; }
template <class T> RT_DEV T rt_rsqrt(T x) { return T(1) / rt_sqrt(x); }
#endif

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

// Partials of D with respect to (X, Y2, u, v); also returns D's scale-free pieces for W.
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

// ---- equilibrium at one stage point, in a local orthonormal frame ------------------------------------------------
// Frame: (e1, e2, e3) = (R^, phi^, Z^) for the axisymmetric kinds, Cartesian for the slabs (cph = 1, sph = 0).
// Gradients are the frame components of the Cartesian gradient; gG = grad_x (n.B) at fixed Cartesian n.
template <class T>
struct Local {
  T X, gX[3];
  T B[3], b2, gb2[3], gG[3], G;
  T nl[3];       // n in the local frame
  T cph, sph;    // e1 = (cph, sph, 0), e2 = (-sph, cph, 0)
};

// shared tail of the two axisymmetric kinds: psi derivatives, F, its (R,Z) derivatives -> B and its gradients
template <class T, int DISP>
RT_DEV void axisym_field(T iR, T psiR, T psiZ, T psiRR, T psiRZ, T psiZZ, T F, T FR, T FZ, Local<T>& L) {
  if (DISP == DISP_O) return;
  const T BR = -psiZ * iR, BZ = psiR * iR, Bp = F * iR;
  const T BR_R = -iR * (psiRZ + BR), BR_Z = -psiZZ * iR;
  const T BZ_R = iR * (psiRR - BZ), BZ_Z = psiRZ * iR;
  const T Bp_R = iR * (FR - Bp), Bp_Z = FZ * iR;
  L.B[0] = BR; L.B[1] = Bp; L.B[2] = BZ;
  L.b2 = BR * BR + BZ * BZ + Bp * Bp;
  L.gb2[0] = T(2) * (BR * BR_R + BZ * BZ_R + Bp * Bp_R);
  L.gb2[1] = T(0);
  L.gb2[2] = T(2) * (BR * BR_Z + BZ * BZ_Z + Bp * Bp_Z);
  const T nR = L.nl[0], nP = L.nl[1], nZ = L.nl[2];
  L.G = nR * BR + nP * Bp + nZ * BZ;
  L.gG[0] = nR * BR_R + nP * Bp_R + nZ * BZ_R;
  L.gG[1] = (nP * BR - nR * Bp) * iR;      // (1/R) d/dphi of n.B at fixed Cartesian n
  L.gG[2] = nR * BR_Z + nP * Bp_Z + nZ * BZ_Z;
}

template <class T, int EQ, int DISP>
RT_DEV bool equilibrium(const Params<T>& P, const T* x, const T* n, Local<T>& L) {
  if (EQ == EQ_PARABOLIC) {
    // X = xs (1 + (x^2+y^2)/L^2)                                          (BASELINE.json config 1)
    const T g = P.xs * P.inv_L2;
    L.X = P.xs + g * (x[0] * x[0] + x[1] * x[1]);
    L.gX[0] = T(2) * g * x[0]; L.gX[1] = T(2) * g * x[1]; L.gX[2] = T(0);
    L.nl[0] = n[0]; L.nl[1] = n[1]; L.nl[2] = n[2];
    L.cph = T(1); L.sph = T(0);
    return true;
  }
  if (EQ == EQ_LINEAR) {
    // n_e = n_ref (x_foot - x)/L_ramp ;  B = (B0 R0 / x) z^                (config 3; Eq. 4 profile)
    const bool inside = x[0] > T(0);
    const T gx = -P.xs * P.inv_Lramp;
    L.X = (x[0] - P.x_foot) * gx;
    L.gX[0] = gx; L.gX[1] = T(0); L.gX[2] = T(0);
    L.nl[0] = n[0]; L.nl[1] = n[1]; L.nl[2] = n[2];
    L.cph = T(1); L.sph = T(0);
    if (DISP != DISP_O) {
      const T ix = rt_rcp(x[0]);
      const T Bz = P.B0R0 * ix;
      L.B[0] = T(0); L.B[1] = T(0); L.B[2] = Bz;
      L.b2 = Bz * Bz;
      L.gb2[0] = T(-2) * L.b2 * ix; L.gb2[1] = T(0); L.gb2[2] = T(0);
      L.G = n[2] * Bz;
      L.gG[0] = -L.G * ix; L.gG[1] = T(0); L.gG[2] = T(0);
    }
    return inside;
  }
  // axisymmetric kinds: cylindrical frame at the point
  const T R2 = x[0] * x[0] + x[1] * x[1];
  const T iR = rt_rsqrt(R2);
  const T R = R2 * iR;
  const T Z = x[2];
  L.cph = x[0] * iR; L.sph = x[1] * iR;
  L.nl[0] = n[0] * L.cph + n[1] * L.sph;
  L.nl[1] = n[1] * L.cph - n[0] * L.sph;
  L.nl[2] = n[2];
  L.gX[1] = T(0);
  if (EQ == EQ_TOKAMAK || EQ == EQ_TOKAMAK_POW) {
    // psi'(r) = B0 r / q, q = q0 + q1 rho^2, F = B0 R0, n_e = n_ref (1 - rho^2)^p       (config 4; reading A9)
    const T dR = R - P.R0;
    const T rho2 = (dR * dR + Z * Z) * P.inv_a2;
    const bool inside = (R > T(0)) && (rho2 < P.rho_max2);
    const T t = T(1) - rho2;
    T shape, dshape;     // t^p and d(t^p)/d(rho^2)
    if (EQ == EQ_TOKAMAK) {
      const T sq = t * rt_rsqrt(t);
      shape = t * sq; dshape = T(-1.5) * sq;
    } else {
      const T pw = rt_pow(t, P.p_exp - T(1));
      shape = pw * t; dshape = -P.p_exp * pw;
    }
    L.X = P.xs * shape;
    const T gx = P.two_xs_a2 * dshape;
    L.gX[0] = gx * dR; L.gX[2] = gx * Z;
    if (DISP != DISP_O) {
      const T iq = rt_rcp(P.q0 + P.q1 * rho2);
      const T Bq = P.B0 * iq;
      const T c = P.two_q1_a2 * iq;
      axisym_field<T, DISP>(iR, Bq * dR, Bq * Z, Bq * (T(1) - c * dR * dR), -Bq * c * dR * Z, Bq * (T(1) - c * Z * Z),
                            P.B0R0, T(0), T(0), L);
    }
    return inside;
  }
  // EQ_GRID: bicubic psi(R,Z), cubic F(psi), n_e(psi)                                    (config 5)
  bool inside = (R >= P.Rmin) && (R <= P.Rmax) && (Z >= P.Zmin) && (Z <= P.Zmax) && (R > T(0));
  int iRc = (int)rt_floor((R - P.Rmin) * P.inv_hR), iZc = (int)rt_floor((Z - P.Zmin) * P.inv_hZ);
  iRc = iRc < 0 ? 0 : (iRc > P.nRc - 1 ? P.nRc - 1 : iRc);
  iZc = iZc < 0 ? 0 : (iZc > P.nZc - 1 ? P.nZc - 1 : iZc);
  if (!inside) { iRc = 0; iZc = 0; }      // NaN positions convert to unspecified ints: keep the gather in bounds
  const T dR = R - (P.Rmin + T(iRc) * P.hR), dZ = Z - (P.Zmin + T(iZc) * P.hZ);
  const T* cc = P.psi_pp + ((size_t)iRc * P.nZc + iZc) * 16;
  T a[4], a1[4], a2[4];   // a_p(dZ) = sum_q c[p][q] dZ^q and its first / second dZ-derivatives
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    T c[4];
    ld4(cc + 4 * p, c);
    a[p] = ((c[3] * dZ + c[2]) * dZ + c[1]) * dZ + c[0];
    a1[p] = (T(3) * c[3] * dZ + T(2) * c[2]) * dZ + c[1];
    a2[p] = T(6) * c[3] * dZ + T(2) * c[2];
  }
  const T psi = ((a[3] * dR + a[2]) * dR + a[1]) * dR + a[0];
  const T psiR = (T(3) * a[3] * dR + T(2) * a[2]) * dR + a[1];
  const T psiZ = ((a1[3] * dR + a1[2]) * dR + a1[1]) * dR + a1[0];
  inside = inside && (psi >= P.psi_min) && (psi <= P.psi_max);
  int iP = (int)rt_floor((psi - P.psi_min) * P.inv_hP);
  iP = iP < 0 ? 0 : (iP > P.nPc - 1 ? P.nPc - 1 : iP);
  if (!inside) iP = 0;
  const T ds = psi - (P.psi_min + T(iP) * P.hP);
  T f[4], g[4];
  ld4(P.prof_pp + (size_t)iP * 8, f);
  ld4(P.prof_pp + (size_t)iP * 8 + 4, g);
  const T Ne = ((g[3] * ds + g[2]) * ds + g[1]) * ds + g[0];
  const T Nep = (T(3) * g[3] * ds + T(2) * g[2]) * ds + g[1];
  L.X = P.xs * Ne;
  const T gx = P.xs * Nep;
  L.gX[0] = gx * psiR; L.gX[2] = gx * psiZ;
  if (DISP != DISP_O) {
    const T F = ((f[3] * ds + f[2]) * ds + f[1]) * ds + f[0];
    const T Fp = (T(3) * f[3] * ds + T(2) * f[2]) * ds + f[1];
    const T psiRR = T(6) * a[3] * dR + T(2) * a[2];
    const T psiRZ = (T(3) * a1[3] * dR + T(2) * a1[2]) * dR + a1[1];
    const T psiZZ = ((a2[3] * dR + a2[2]) * dR + a2[1]) * dR + a2[0];
    axisym_field<T, DISP>(iR, psiR, psiZ, psiRR, psiRZ, psiZZ, F, Fp * psiR, Fp * psiZ, L);
  }
  return inside;
}

// ---- one evaluation of the ray right-hand side f(y), y = (x, n) --------------------------------------------------
// Returns false (and f unspecified) if x is outside the equilibrium's domain.
template <class T, int EQ, int DISP>
RT_DEV bool ray_rhs(const Params<T>& P, const T* y, T* f) {
  Local<T> L;
  const bool inside = equilibrium<T, EQ, DISP>(P, y, y + 3, L);
  const T* nl = L.nl;
  const T v = nl[0] * nl[0] + nl[1] * nl[1] + nl[2] * nl[2];
  T fx[3], fn[3];        // local-frame components
  if (DISP == DISP_O) {
    // D = v - 1 + X:  dD/dn = 2 n, dD/dx = grad X, W = -2 (v + X)
    const T iW = rt_rcp(v + L.X);
#pragma unroll
    for (int j = 0; j < 3; ++j) { fx[j] = nl[j] * iW; fn[j] = T(-0.5) * L.gX[j] * iW; }
  } else {
    const T ib2 = rt_rcp(L.b2);
    const T Y2 = P.beta * L.b2;
    const T u = (DISP == DISP_FULL) ? L.G * L.G * ib2 : T(0);
    T DX, DY2, Du, Dv;
    disp_partials<T, DISP>(P, L.X, Y2, u, v, DX, DY2, Du, Dv);
    const T W = T(-2) * (L.X * DX + Y2 * DY2 + u * Du + v * Dv);
    const T iW = rt_rcp(W);
    const T DG = T(2) * L.G * ib2 * Du;            // dD/dG at fixed |B|^2
    const T Db2 = P.beta * DY2 - u * ib2 * Du;     // dD/d|B|^2 at fixed G: through Y2 and through u = G^2/|B|^2
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      T dn = T(2) * Dv * nl[j], dx = DX * L.gX[j] + Db2 * L.gb2[j];
      if (DISP == DISP_FULL) { dn += DG * L.B[j]; dx += DG * L.gG[j]; }
      fx[j] = -dn * iW; fn[j] = dx * iW;
    }
  }
  f[0] = fx[0] * L.cph - fx[1] * L.sph; f[1] = fx[0] * L.sph + fx[1] * L.cph; f[2] = fx[2];
  f[3] = fn[0] * L.cph - fn[1] * L.sph; f[4] = fn[0] * L.sph + fn[1] * L.cph; f[5] = fn[2];
  return inside;
}

// signed D at y = (x, n); *inside reports the domain test
template <class T, int EQ, int DISP>
RT_DEV T ray_D(const Params<T>& P, const T* y, bool* inside) {
  Local<T> L;
  *inside = equilibrium<T, EQ, DISP>(P, y, y + 3, L);
  const T v = y[3] * y[3] + y[4] * y[4] + y[5] * y[5];
  if (DISP == DISP_O) return disp_value<T, DISP>(P, L.X, T(0), T(0), v);
  const T u = (DISP == DISP_FULL) ? L.G * L.G * rt_rcp(L.b2) : T(0);
  return disp_value<T, DISP>(P, L.X, P.beta * L.b2, u, v);
}

}  // namespace rt
