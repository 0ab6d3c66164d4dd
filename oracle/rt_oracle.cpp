// rt_oracle.cpp -- CPU ORACLE for batched RF ray tracing.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
// load or call this file.  It shares no code, header, table or constant generator with the CUDA path
// (paper_2508_15967_b200/csrc).  It is plain, slow and meant to be checked against the paper by eye.
//
// What it computes (citations are /root/reference/PAPER.md line numbers, "L<n>"):
//   * the ray equations  dx/dt = -(dD/dk)/(dD/dw),  dk/dt = +(dD/dx)/(dD/dw)      (Eq. 2-3;
//     Eq. 3's printed denominator is garbled, reading A1; sign per reading A2)
//   * integrated by the classical 4th-order Runge-Kutta tableau at fixed step     (L147; reading A7)
//   * for D one of
//       OMODE      D = c^2|k|^2/w^2 - 1 + wpe^2/w^2                (BASELINE.json config 1; L157/L191)
//       XMODE      D = S n^2 - R L                                  (reading A5; L157/L191)
//       COLD_FULL  D = Det(eps + n n - n^2 I)                       (Eq. 5) with eps from
//                  Eq. 7-10 (L177-189) rotated to Cartesian axes: eps = S (I - b b^T) + P b b^T + i Dx [b]x,
//                  b = B/|B|, n = c k / w (Eq. 6); regular at n parallel to B
//   * over four plasma equilibria B(x), n_e(x) (L151).
//
// State and units here are the paper's own: x [m], k [rad/m], t [s], w [rad/s]  (L147: "inputs for
// x, k, t and w").  The C-ABI's step `dt` is given in tau = c*t metres (reading A3), so h = dt/c seconds.
//
// Gradients of D: forward-mode automatic differentiation with dual numbers carrying the 7 partials
// (x, y, z, kx, ky, kz, w) through the *plain expression* of D -- the paper's own route is chain-rule
// auto-differentiation (L66, L147).  Nothing here is hand-differentiated, so it is independent of the
// CUDA path's hand-derived chain rule.
//
// Step acceptance rule (reading A12): a step is rejected, and the ray frozen from then on,
// if any of its 4 stage points lies outside the equilibrium's domain (status 1) or if the new state
// is not finite (status 2).  |D| at a saved state outside the domain is NaN.
//
// Also here: per-ray frequencies and critical-surface diagnostics, the second ensemble workload,
// full-orbit charged particles in the same equilibria (oracle_orbit), and the paper's own launch
// iteration (L159: Newton on k_x at fixed k_y, k_z; oracle_launch_kx).
//
// Parity pins: tests/test_oracle_*.py (P1..P20 in DESIGN.md).  No function here is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- physical constants: CODATA-2022 numerals (reading A6) -------------------------------
constexpr double C_LIGHT = 299792458.0;        // m/s
constexpr double CHARGE_E = 1.602176634e-19;    // C
constexpr double MASS_E  = 9.1093837139e-31;   // kg
constexpr double EPS0    = 8.8541878188e-12;   // F/m

// ---- dual numbers: value + 7 partial derivatives ----------------------------------------------------
constexpr int ND = 7;  // 0..2: x,y,z   3..5: kx,ky,kz   6: omega
struct Dual {
  double v;
  double d[ND];
};
inline Dual mk(double v) { Dual r; r.v = v; for (int i = 0; i < ND; ++i) r.d[i] = 0.0; return r; }
inline Dual seed(double v, int i) { Dual r = mk(v); r.d[i] = 1.0; return r; }

inline Dual operator+(const Dual& a, const Dual& b) { Dual r; r.v = a.v + b.v; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
inline Dual operator-(const Dual& a, const Dual& b) { Dual r; r.v = a.v - b.v; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
inline Dual operator-(const Dual& a) { Dual r; r.v = -a.v; for (int i = 0; i < ND; ++i) r.d[i] = -a.d[i]; return r; }
inline Dual operator*(const Dual& a, const Dual& b) { Dual r; r.v = a.v * b.v; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
inline Dual operator/(const Dual& a, const Dual& b) {
  Dual r; r.v = a.v / b.v;
  for (int i = 0; i < ND; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v;
  return r;
}
inline Dual operator+(const Dual& a, double b) { Dual r = a; r.v += b; return r; }
inline Dual operator+(double a, const Dual& b) { return b + a; }
inline Dual operator-(const Dual& a, double b) { Dual r = a; r.v -= b; return r; }
inline Dual operator-(double a, const Dual& b) { return (-b) + a; }
inline Dual operator*(const Dual& a, double b) { Dual r; r.v = a.v * b; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] * b; return r; }
inline Dual operator*(double a, const Dual& b) { return b * a; }
inline Dual operator/(const Dual& a, double b) { Dual r; r.v = a.v / b; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] / b; return r; }
inline Dual operator/(double a, const Dual& b) { return mk(a) / b; }

inline double sqrt_(double a) { return std::sqrt(a); }
inline Dual sqrt_(const Dual& a) {
  Dual r; r.v = std::sqrt(a.v);
  for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] / (2.0 * r.v);
  return r;
}
inline double pow_(double a, double p) { return std::pow(a, p); }
inline Dual pow_(const Dual& a, double p) {
  Dual r; r.v = std::pow(a.v, p);
  const double dp = p * std::pow(a.v, p - 1.0);
  for (int i = 0; i < ND; ++i) r.d[i] = dp * a.d[i];
  return r;
}
inline double val(double a) { return a; }
inline double val(const Dual& a) { return a.v; }

// ---- complex numbers over T (for the Hermitian 3x3 determinant of Eq. 5) ----------------------------
template <class T> struct Cx { T re, im; };
template <class T> inline Cx<T> operator+(const Cx<T>& a, const Cx<T>& b) { return {a.re + b.re, a.im + b.im}; }
template <class T> inline Cx<T> operator-(const Cx<T>& a, const Cx<T>& b) { return {a.re - b.re, a.im - b.im}; }
template <class T> inline Cx<T> operator*(const Cx<T>& a, const Cx<T>& b) {
  return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}

}  // namespace

// ---- the C structs shared with oracle/__init__.py (ctypes) ------------------------------------------
extern "C" {

enum { ORC_EQ_SLAB_PARABOLIC = 0, ORC_EQ_SLAB_LINEAR_BR = 1, ORC_EQ_TOKAMAK_CIRCULAR = 2, ORC_EQ_GRID_RZ = 3 };
enum { ORC_DISP_OMODE = 0, ORC_DISP_XMODE = 1, ORC_DISP_COLD_FULL = 2 };

struct orc_equilibrium {
  int32_t kind;
  int32_t nR, nZ, nPsi;
  double n_ref, L;                    // parabolic:  n_e = n_ref (1 + (x^2+y^2)/L^2)
  double x_foot, L_ramp, B0, R0;      // linear slab: n_e = n_ref (x_foot - x)/L_ramp ; B = (B0 R0 / x) z^
  double a, q0, q1, p_exp, rho_max;   // tokamak: q = q0 + q1 rho^2, n_e = n_ref (1 - rho^2)^p_exp, domain rho < rho_max
  double Rmin, Rmax, Zmin, Zmax, psi_min, psi_max;
  // piecewise-polynomial spline pieces, ascending powers of the offset from the cell's lower node:
  const double* psi_pp;               // [nR-1][nZ-1][4][4]   psi = sum_pq c[p][q] dR^p dZ^q
  const double* F_pp;                 // [nPsi-1][4]          F   = sum_m f[m] ds^m ,  ds = psi - psi_i
  const double* ne_pp;                // [nPsi-1][4]
  double ion_mass, ion_charge;        // kg, units of e; ion_mass = 0 => electrons only; n_i = n_e / ion_charge
};

}  // extern "C"

namespace {

// ---- equilibrium: n_e(x) and B(x) at one point (L151) ------------------------------------------------
template <class T> struct Plasma {
  T ne;
  T B[3];
  bool inside;
};

template <class T>
Plasma<T> equilibrium(const orc_equilibrium& eq, const T x[3]) {
  Plasma<T> pl;
  const T zero = x[0] * 0.0;
  pl.B[0] = zero; pl.B[1] = zero; pl.B[2] = zero; pl.ne = zero;
  pl.inside = true;
  switch (eq.kind) {
    case ORC_EQ_SLAB_PARABOLIC: {
      // BASELINE.json config 1: wpe^2/w^2 = 0.5 (1 + (x^2+y^2)/L^2)  <=>  n_e = n_ref (1 + (x^2+y^2)/L^2).
      pl.ne = eq.n_ref * (1.0 + (x[0] * x[0] + x[1] * x[1]) / (eq.L * eq.L));
      break;
    }
    case ORC_EQ_SLAB_LINEAR_BR: {
      // BASELINE.json config 3; linear unclamped profile as in Eq. 4 (L153).  x plays the role of R.
      pl.inside = val(x[0]) > 0.0;
      pl.ne = eq.n_ref * (eq.x_foot - x[0]) / eq.L_ramp;
      if (pl.inside) pl.B[2] = (eq.B0 * eq.R0) / x[0];
      break;
    }
    case ORC_EQ_TOKAMAK_CIRCULAR: {
      // BASELINE.json config 4; reading A9:  B = grad(phi) x grad(psi) + F grad(phi),
      // F = B0 R0,  dpsi/dr = B0 r / q(rho),  q = q0 + q1 rho^2.
      const T R = sqrt_(x[0] * x[0] + x[1] * x[1]);
      const T Z = x[2];
      const T r2 = (R - eq.R0) * (R - eq.R0) + Z * Z;
      const T rho2 = r2 / (eq.a * eq.a);
      pl.inside = (val(R) > 0.0) && (val(rho2) < eq.rho_max * eq.rho_max);
      if (!pl.inside) break;
      const T q = eq.q0 + eq.q1 * rho2;
      const T psi_R = eq.B0 * (R - eq.R0) / q;   // dpsi/dr * (R-R0)/r
      const T psi_Z = eq.B0 * Z / q;             // dpsi/dr * Z/r
      const T BR = -psi_Z / R;
      const T BZ = psi_R / R;
      const T Bphi = (eq.B0 * eq.R0) / R;
      const T cosphi = x[0] / R, sinphi = x[1] / R;
      pl.B[0] = BR * cosphi - Bphi * sinphi;
      pl.B[1] = BR * sinphi + Bphi * cosphi;
      pl.B[2] = BZ;
      pl.ne = eq.n_ref * pow_(1.0 - rho2, eq.p_exp);
      break;
    }
    case ORC_EQ_GRID_RZ: {
      // BASELINE.json config 5: psi(R,Z), F(psi), n_e(psi) from cubic spline pieces (L60).
      const T R = sqrt_(x[0] * x[0] + x[1] * x[1]);
      const T Z = x[2];
      const double Rv = val(R), Zv = val(Z);
      pl.inside = (Rv >= eq.Rmin) && (Rv <= eq.Rmax) && (Zv >= eq.Zmin) && (Zv <= eq.Zmax) && (Rv > 0.0);
      if (!pl.inside) break;
      const double hR = (eq.Rmax - eq.Rmin) / (eq.nR - 1), hZ = (eq.Zmax - eq.Zmin) / (eq.nZ - 1);
      int iR = (int)std::floor((Rv - eq.Rmin) / hR), iZ = (int)std::floor((Zv - eq.Zmin) / hZ);
      if (iR < 0) iR = 0; if (iR > eq.nR - 2) iR = eq.nR - 2;
      if (iZ < 0) iZ = 0; if (iZ > eq.nZ - 2) iZ = eq.nZ - 2;
      const T dR = R - (eq.Rmin + iR * hR), dZ = Z - (eq.Zmin + iZ * hZ);
      const double* c = eq.psi_pp + ((size_t)iR * (eq.nZ - 1) + iZ) * 16;
      T pR[4], pZ[4];
      pR[0] = zero + 1.0; pZ[0] = zero + 1.0;
      for (int m = 1; m < 4; ++m) { pR[m] = pR[m - 1] * dR; pZ[m] = pZ[m - 1] * dZ; }
      T psi = zero, psi_R = zero, psi_Z = zero;
      for (int p = 0; p < 4; ++p)
        for (int q = 0; q < 4; ++q) {
          const double cpq = c[p * 4 + q];
          psi = psi + cpq * pR[p] * pZ[q];
          if (p > 0) psi_R = psi_R + (cpq * p) * pR[p - 1] * pZ[q];
          if (q > 0) psi_Z = psi_Z + (cpq * q) * pR[p] * pZ[q - 1];
        }
      const double psiv = val(psi);
      if (!(psiv >= eq.psi_min && psiv <= eq.psi_max)) { pl.inside = false; break; }
      const double hP = (eq.psi_max - eq.psi_min) / (eq.nPsi - 1);
      int iP = (int)std::floor((psiv - eq.psi_min) / hP);
      if (iP < 0) iP = 0; if (iP > eq.nPsi - 2) iP = eq.nPsi - 2;
      const T ds = psi - (eq.psi_min + iP * hP);
      const double* f = eq.F_pp + (size_t)iP * 4;
      const double* g = eq.ne_pp + (size_t)iP * 4;
      const T F = f[0] + f[1] * ds + f[2] * ds * ds + f[3] * ds * ds * ds;
      pl.ne = g[0] + g[1] * ds + g[2] * ds * ds + g[3] * ds * ds * ds;
      const T BR = -psi_Z / R;
      const T BZ = psi_R / R;
      const T Bphi = F / R;
      const T cosphi = x[0] / R, sinphi = x[1] / R;
      pl.B[0] = BR * cosphi - Bphi * sinphi;
      pl.B[1] = BR * sinphi + Bphi * cosphi;
      pl.B[2] = BZ;
      break;
    }
    default:
      pl.inside = false;
  }
  return pl;
}

// ---- Stix elements: eps11 = S, eps12 = -i Dx, eps33 = P  (Eq. 8-10) -----------------------
template <class T> struct Stix { T S, Dx, P; };

template <class T>
Stix<T> stix(const orc_equilibrium& eq, const Plasma<T>& pl, const T& w) {
  const T Bmag = sqrt_(pl.B[0] * pl.B[0] + pl.B[1] * pl.B[1] + pl.B[2] * pl.B[2]);
  const int n_species = (eq.ion_mass > 0.0) ? 2 : 1;
  T S = w * 0.0 + 1.0, Dx = w * 0.0, P = w * 0.0 + 1.0;
  for (int s = 0; s < n_species; ++s) {
    const double q_s = (s == 0) ? -CHARGE_E : eq.ion_charge * CHARGE_E;
    const double m_s = (s == 0) ? MASS_E : eq.ion_mass;
    const T n_s = (s == 0) ? pl.ne : pl.ne / eq.ion_charge;        // quasi-neutral, reading A6
    const T wp2 = n_s * (q_s * q_s / (EPS0 * m_s));                // plasma frequency squared
    const T Om = Bmag * (q_s / m_s);                               // signed cyclotron frequency
    const T X = wp2 / (w * w);
    const T Y = Om / w;
    S = S - X / (1.0 - Y * Y);                                     // Eq. 8
    Dx = Dx + Y * X / (1.0 - Y * Y);                               // Eq. 9: eps12 = -i Dx
    P = P - X;                                                     // Eq. 10
  }
  return {S, Dx, P};
}

// ---- the dispersion function D(x, k, w) --------------------------------------------------------------
template <class T>
T dispersion(const orc_equilibrium& eq, int disp, const T x[3], const T k[3], const T& w, bool* inside) {
  const Plasma<T> pl = equilibrium(eq, x);
  *inside = pl.inside;
  const T zero = w * 0.0;
  if (!pl.inside) return zero + std::numeric_limits<double>::quiet_NaN();
  T n[3];
  for (int i = 0; i < 3; ++i) n[i] = C_LIGHT * k[i] / w;           // Eq. 6
  const T n2 = n[0] * n[0] + n[1] * n[1] + n[2] * n[2];
  if (disp == ORC_DISP_OMODE) {
    const T X = pl.ne * (CHARGE_E * CHARGE_E / (EPS0 * MASS_E)) / (w * w);      // wpe^2 / w^2
    return n2 - 1.0 + X;                                           // BASELINE.json config 1
  }
  const Stix<T> st = stix(eq, pl, w);
  if (disp == ORC_DISP_XMODE) {
    const T Rr = st.S + st.Dx, Ll = st.S - st.Dx;
    return st.S * n2 - Rr * Ll;                                    // reading A5
  }
  // COLD_FULL: Det(eps + n n - n^2 I) (Eq. 5) written out in the CARTESIAN axes the state lives in.  Eq. 7 (L177)
  // gives eps in the frame whose 3rd axis is b = B/|B|: diag(S, S, P) with eps12 = -i Dx = -eps21.  Rotated to
  // Cartesian axes that tensor is
  //      eps = S (I - b b^T) + P b b^T + i Dx [b]x ,      ([b]x v = b x v, i.e. ([b]x)_ij = -e_ijk b_k;
  //                                                        for b = z^ this is eps12 = -i Dx, eps21 = +i Dx: Eq. 7)
  // ("the explicit 3x3 matrix with Cartesian dB_i/dx_j").  No frame is built from the
  // perpendicular part of n, so nothing non-smooth is differentiated and the dual-number partials are finite at exactly
  // parallel propagation (theta = 0, the R and L waves of Fig. 3) -- D is a polynomial in n there.
  const T Bmag = sqrt_(pl.B[0] * pl.B[0] + pl.B[1] * pl.B[1] + pl.B[2] * pl.B[2]);
  T b[3];
  for (int i = 0; i < 3; ++i) b[i] = pl.B[i] / Bmag;
  const T bx[3][3] = {{zero, -b[2], b[1]}, {b[2], zero, -b[0]}, {-b[1], b[0], zero}};   // [b]x
  Cx<T> M[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      const T bb = b[i] * b[j];
      T re = st.P * bb - st.S * bb + n[i] * n[j];                  // (P - S) b_i b_j + n_i n_j
      if (i == j) re = re + st.S - n2;                             // + (S - n^2) delta_ij
      M[i][j] = {re, st.Dx * bx[i][j]};
    }
  const Cx<T> det = M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1])
                  - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
                  + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
  return det.re;                                                   // imaginary part vanishes (Hermitian M)
}

// D and its 7 partials at a double-precision point.
bool eval_D(const orc_equilibrium& eq, int disp, const double x[3], const double k[3], double w, double* D, double grad[ND]) {
  Dual xd[3], kd[3];
  for (int i = 0; i < 3; ++i) { xd[i] = seed(x[i], i); kd[i] = seed(k[i], 3 + i); }
  const Dual wd = seed(w, 6);
  bool inside;
  const Dual Dd = dispersion<Dual>(eq, disp, xd, kd, wd, &inside);
  *D = Dd.v;
  for (int i = 0; i < ND; ++i) grad[i] = Dd.d[i];
  return inside;
}

// Right-hand side of the ray equations at y = (x, k): Eq. 2-3.
bool rhs(const orc_equilibrium& eq, int disp, double w, const double y[6], double f[6]) {
  double D, g[ND];
  const bool inside = eval_D(eq, disp, y, y + 3, w, &D, g);
  if (!inside) { for (int i = 0; i < 6; ++i) f[i] = 0.0; return false; }
  for (int i = 0; i < 3; ++i) {
    f[i] = -g[3 + i] / g[6];      // dx/dt = -(dD/dk)/(dD/dw)
    f[3 + i] = g[i] / g[6];       // dk/dt = +(dD/dx)/(dD/dw)
  }
  return true;
}

double residual(const orc_equilibrium& eq, int disp, double w, const double y[6]) {
  bool inside;
  const double D = dispersion<double>(eq, disp, y, y + 3, w, &inside);
  return inside ? std::fabs(D) : std::numeric_limits<double>::quiet_NaN();
}

// One classical RK4 step (reading A7).  Returns 0 accepted, 1 left domain, 2 non-finite.
int rk4_step(const orc_equilibrium& eq, int disp, double w, double h, double y[6]) {
  double k1[6], k2[6], k3[6], k4[6], ys[6];
  if (!rhs(eq, disp, w, y, k1)) return 1;
  for (int i = 0; i < 6; ++i) ys[i] = y[i] + 0.5 * h * k1[i];
  if (!rhs(eq, disp, w, ys, k2)) return 1;
  for (int i = 0; i < 6; ++i) ys[i] = y[i] + 0.5 * h * k2[i];
  if (!rhs(eq, disp, w, ys, k3)) return 1;
  for (int i = 0; i < 6; ++i) ys[i] = y[i] + h * k3[i];
  if (!rhs(eq, disp, w, ys, k4)) return 1;
  for (int i = 0; i < 6; ++i) ys[i] = y[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
  for (int i = 0; i < 6; ++i) if (!std::isfinite(ys[i])) return 2;
  for (int i = 0; i < 6; ++i) y[i] = ys[i];
  return 0;
}

bool combo_supported(const orc_equilibrium& eq, int disp) {
  if (eq.kind < 0 || eq.kind > 3 || disp < 0 || disp > 2) return false;
  if (eq.kind == ORC_EQ_SLAB_PARABOLIC && disp != ORC_DISP_OMODE) return false;   // no B field
  return true;
}

}  // namespace

extern "C" {

// Trace n_rays rays.  All pointers are HOST pointers.  Layouts equal the C-ABI's (include/rt.h):
// x0,k0 [3][n_rays]; out_traj [n_steps/save_stride+1][6][n_rays]; out_final [6][n_rays];
// out_residual [n_saved][n_rays] if out_traj else [n_rays]; out_status [n_rays].  Any output may be NULL.
// omega_rays: one frequency per ray [n_rays] (L147: w is a per-ray kernel input), or NULL to use `omega_all` for every ray.
static int trace_impl(const orc_equilibrium* eq, int disp, const double* x0, const double* k0, double omega_all,
                      const double* omega_rays, int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride,
                      double* out_traj, double* out_final, double* out_residual, int32_t* out_status, int n_threads) {
  if (!eq || !combo_supported(*eq, disp) || n_rays < 0 || n_steps < 0 || save_stride < 1) return -1;
  if (out_traj && (n_steps % save_stride) != 0) return -1;
  const double h = dt / C_LIGHT;   // seconds (reading A3: dt is in tau = c t)
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < n_rays; ++i) {
    const double omega = omega_rays ? omega_rays[i] : omega_all;
    double y[6];
    for (int c = 0; c < 3; ++c) { y[c] = x0[c * n_rays + i]; y[3 + c] = k0[c * n_rays + i]; }
    // DESIGN.md reading A20: a wave frequency that is not positive and finite defines no ray (n = c k / w, Eq. 6): the
    // ray is never advanced (status 2), every sample is the launch state, and |D| is NaN.
    const bool bad_omega = !(omega > 0.0 && std::isfinite(omega));
    int status = bad_omega ? 2 : 0;
    auto res = [&]() { return bad_omega ? std::numeric_limits<double>::quiet_NaN() : residual(*eq, disp, omega, y); };
    if (out_traj) {
      for (int c = 0; c < 6; ++c) out_traj[(0 * 6 + c) * n_rays + i] = y[c];
      if (out_residual) out_residual[0 * n_rays + i] = res();
    }
    for (int64_t s = 1; s <= n_steps; ++s) {
      if (status == 0) status = rk4_step(*eq, disp, omega, h, y);
      if (out_traj && (s % save_stride) == 0) {
        const int64_t m = s / save_stride;
        for (int c = 0; c < 6; ++c) out_traj[(m * 6 + c) * n_rays + i] = y[c];
        if (out_residual) out_residual[m * n_rays + i] = res();
      }
    }
    if (out_final) for (int c = 0; c < 6; ++c) out_final[c * n_rays + i] = y[c];
    if (!out_traj && out_residual) out_residual[i] = res();
    if (out_status) out_status[i] = status;
  }
  return 0;
}

int oracle_trace(const orc_equilibrium* eq, int disp, const double* x0, const double* k0, double omega,
                 int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, double* out_traj,
                 double* out_final, double* out_residual, int32_t* out_status, int n_threads) {
  return trace_impl(eq, disp, x0, k0, omega, nullptr, n_rays, n_steps, dt, save_stride, out_traj, out_final, out_residual,
                    out_status, n_threads);
}

// The same with one frequency per ray: omega [n_rays].
int oracle_trace_w(const orc_equilibrium* eq, int disp, const double* x0, const double* k0, const double* omega,
                   int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, double* out_traj,
                   double* out_final, double* out_residual, int32_t* out_status, int n_threads) {
  if (!omega) return -1;
  return trace_impl(eq, disp, x0, k0, 0.0, omega, n_rays, n_steps, dt, save_stride, out_traj, out_final, out_residual,
                    out_status, n_threads);
}

// The convergence workflow (L80, section 2.3: "workflows ... can be implemented by chaining calls to evaluation and
// reduction kernels until a tolerance is met"; L76: reduction kernels; SURVEY 8(f)-2 "stop-when-all-frozen"), stated for
// the ray tracer: advance the ensemble in chunks of `chunk_steps` RK4 steps; after each chunk reduce over the rays
//      n_active = number of rays with status 0,        max_D = max |D| over the rays whose |D| is finite,
// and stop after the first chunk at which n_active == 0 (every ray is frozen), or max_D > tol (the ensemble has drifted
// off the dispersion surface by more than the tolerance), or `max_chunks` chunks have run.  A frozen ray stays frozen
// across chunks (reading A12).  Outputs: out_final [6][n], out_residual [n] (|D| at the final state), out_status [n],
// out_info [4] = {chunks run, n_active at the stop, reason (0 max_chunks reached, 1 all rays frozen, 2 tolerance
// exceeded; 1 wins if both hold), 0} and *out_maxD = max_D at the stop (0 if no ray has a finite |D|).
int oracle_trace_until(const orc_equilibrium* eq, int disp, const double* x0, const double* k0, double omega, int64_t n_rays,
                       int64_t chunk_steps, int64_t max_chunks, double dt, double tol, double* out_final,
                       double* out_residual, int32_t* out_status, int64_t* out_info, double* out_maxD, int n_threads) {
  if (!eq || !combo_supported(*eq, disp) || n_rays < 0 || chunk_steps < 1 || max_chunks < 0 || !(tol > 0.0)) return -1;
  if (!out_final || !out_residual || !out_status || !out_info || !out_maxD) return -1;
  for (int64_t i = 0; i < n_rays; ++i) {
    for (int c = 0; c < 3; ++c) { out_final[c * n_rays + i] = x0[c * n_rays + i]; out_final[(3 + c) * n_rays + i] = k0[c * n_rays + i]; }
    out_status[i] = (omega > 0.0 && std::isfinite(omega)) ? 0 : 2;           // reading A20
  }
  const double h = dt / C_LIGHT;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
  int64_t chunks = 0, n_active = 0, reason = 0;
  double max_D = 0.0;
  while (chunks < max_chunks) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n_rays; ++i) {                                   // the "evaluation kernel": one chunk
      double y[6];
      for (int c = 0; c < 6; ++c) y[c] = out_final[c * n_rays + i];
      int status = out_status[i];
      for (int64_t s = 0; s < chunk_steps && status == 0; ++s) status = rk4_step(*eq, disp, omega, h, y);
      for (int c = 0; c < 6; ++c) out_final[c * n_rays + i] = y[c];
      out_status[i] = status;
      out_residual[i] = (status == 2 && !(omega > 0.0 && std::isfinite(omega))) ? std::numeric_limits<double>::quiet_NaN()
                                                                               : residual(*eq, disp, omega, y);
    }
    ++chunks;
    n_active = 0; max_D = 0.0;                                               // the "reduction kernel"
    for (int64_t i = 0; i < n_rays; ++i) {
      if (out_status[i] == 0) ++n_active;
      if (std::isfinite(out_residual[i]) && out_residual[i] > max_D) max_D = out_residual[i];
    }
    if (n_active == 0) { reason = 1; break; }
    if (max_D > tol) { reason = 2; break; }
  }
  if (chunks == 0)                                                           // max_chunks == 0: report the launch state
    for (int64_t i = 0; i < n_rays; ++i) {
      double y[6];
      for (int c = 0; c < 6; ++c) y[c] = out_final[c * n_rays + i];
      out_residual[i] = (out_status[i] == 2) ? std::numeric_limits<double>::quiet_NaN() : residual(*eq, disp, omega, y);
      if (out_status[i] == 0) ++n_active;
      if (std::isfinite(out_residual[i]) && out_residual[i] > max_D) max_D = out_residual[i];
    }
  out_info[0] = chunks; out_info[1] = n_active; out_info[2] = reason; out_info[3] = 0;
  *out_maxD = max_D;
  return 0;
}

// Critical-surface diagnostics (L149: cut-offs and resonances; Fig. 3-4 L157/L175) at n points with one frequency per
// point: out [10][n] = n_e, |B|, X = wpe^2/w^2, Y = |Wce|/w (electrons), S, Dx, P (Eq. 8-10), R = S + Dx, L = S - Dx,
// n_par^2 = (n.B/|B|)^2 with n = c k / w (Eq. 6); n_par^2 = 0 where B = 0.  NaN outside the domain.
int oracle_diagnostics(const orc_equilibrium* eq, const double* x, const double* k, const double* omega, int64_t n,
                       double* out) {
  if (!eq || !omega) return -1;
  for (int64_t i = 0; i < n; ++i) {
    const double xi[3] = {x[i], x[n + i], x[2 * n + i]};
    const double w = omega[i];
    const Plasma<double> pl = equilibrium<double>(*eq, xi);
    if (!pl.inside) {
      for (int r = 0; r < 10; ++r) out[r * n + i] = std::numeric_limits<double>::quiet_NaN();
      continue;
    }
    const Stix<double> st = stix<double>(*eq, pl, w);
    const double Bm = std::sqrt(pl.B[0] * pl.B[0] + pl.B[1] * pl.B[1] + pl.B[2] * pl.B[2]);
    double npar = 0.0;
    if (Bm > 0.0)
      for (int c = 0; c < 3; ++c) npar += (C_LIGHT * k[c * n + i] / w) * (pl.B[c] / Bm);
    out[0 * n + i] = pl.ne;
    out[1 * n + i] = Bm;
    out[2 * n + i] = pl.ne * (CHARGE_E * CHARGE_E / (EPS0 * MASS_E)) / (w * w);
    out[3 * n + i] = (CHARGE_E / MASS_E) * Bm / w;
    out[4 * n + i] = st.S;
    out[5 * n + i] = st.Dx;
    out[6 * n + i] = st.P;
    out[7 * n + i] = st.S + st.Dx;
    out[8 * n + i] = st.S - st.Dx;
    out[9 * n + i] = npar * npar;
  }
  return 0;
}

// D and its partials (x,y,z,kx,ky,kz,w) at n points; x,k are [3][n]; grad is [7][n]; inside is [n].
int oracle_dispersion(const orc_equilibrium* eq, int disp, const double* x, const double* k, double omega,
                      int64_t n, double* D, double* grad, int32_t* inside) {
  if (!eq || !combo_supported(*eq, disp)) return -1;
  for (int64_t i = 0; i < n; ++i) {
    const double xi[3] = {x[i], x[n + i], x[2 * n + i]}, ki[3] = {k[i], k[n + i], k[2 * n + i]};
    double Di, g[ND];
    const bool in = eval_D(*eq, disp, xi, ki, omega, &Di, g);
    if (D) D[i] = Di;
    if (grad) for (int j = 0; j < ND; ++j) grad[j * n + i] = g[j];
    if (inside) inside[i] = in ? 1 : 0;
  }
  return 0;
}

// D alone, evaluated in plain double arithmetic (no dual numbers): the function finite differences act on.
int oracle_dispersion_value(const orc_equilibrium* eq, int disp, const double* x, const double* k,
                            const double* omega /* [n] */, int64_t n, double* D) {
  if (!eq || !combo_supported(*eq, disp)) return -1;
  for (int64_t i = 0; i < n; ++i) {
    const double xi[3] = {x[i], x[n + i], x[2 * n + i]}, ki[3] = {k[i], k[n + i], k[2 * n + i]};
    bool in;
    D[i] = dispersion<double>(*eq, disp, xi, ki, omega[i], &in);
  }
  return 0;
}

// Equilibrium and Stix elements at n points: ne [n], B [3][n], SDP [3][n] (S, Dx, P), inside [n].
int oracle_plasma(const orc_equilibrium* eq, const double* x, double omega, int64_t n, double* ne, double* B,
                  double* SDP, int32_t* inside) {
  if (!eq) return -1;
  for (int64_t i = 0; i < n; ++i) {
    const double xi[3] = {x[i], x[n + i], x[2 * n + i]};
    const Plasma<double> pl = equilibrium<double>(*eq, xi);
    if (inside) inside[i] = pl.inside ? 1 : 0;
    if (ne) ne[i] = pl.ne;
    if (B) for (int c = 0; c < 3; ++c) B[c * n + i] = pl.B[c];
    if (SDP) {
      const Stix<double> st = stix<double>(*eq, pl, omega);
      SDP[i] = st.S; SDP[n + i] = st.Dx; SDP[2 * n + i] = st.P;
    }
  }
  return 0;
}

// Launch states (L159): given position x0 and unit direction dir, find |n| with D = 0 on the chosen branch,
// Newton-polished to |D| < 1e-15 (at most 8 iterations), and return k0 = |n| dir w / c.
//   OMODE: n^2 = 1 - X.   XMODE: n^2 = R L / S.
//   COLD_FULL: the biquadratic A n^4 - B n^2 + C = 0 (Stix), A = S sin^2 + P cos^2, B = R L sin^2 + P S (1 + cos^2),
//   C = P R L, theta the angle between dir and B; branch 0 = the root nearer to P ("O"), 1 = the other ("X")
//   (reading A11).
static int launch_impl(const orc_equilibrium* eq, int disp, int branch, const double* x0, const double* dir,
                       double omega_all, const double* omega_rays, int64_t n, double* k0, double* D_out) {
  if (!eq || !combo_supported(*eq, disp)) return -1;
  for (int64_t i = 0; i < n; ++i) {
    const double omega = omega_rays ? omega_rays[i] : omega_all;
    const double xi[3] = {x0[i], x0[n + i], x0[2 * n + i]}, di[3] = {dir[i], dir[n + i], dir[2 * n + i]};
    const Plasma<double> pl = equilibrium<double>(*eq, xi);
    double n2 = std::numeric_limits<double>::quiet_NaN();
    if (pl.inside) {
      if (disp == ORC_DISP_OMODE) {
        n2 = 1.0 - pl.ne * (CHARGE_E * CHARGE_E / (EPS0 * MASS_E)) / (omega * omega);
      } else {
        const Stix<double> st = stix<double>(*eq, pl, omega);
        const double Rr = st.S + st.Dx, Ll = st.S - st.Dx;
        if (disp == ORC_DISP_XMODE) {
          n2 = Rr * Ll / st.S;
        } else {
          const double Bm = std::sqrt(pl.B[0] * pl.B[0] + pl.B[1] * pl.B[1] + pl.B[2] * pl.B[2]);
          const double ct = (di[0] * pl.B[0] + di[1] * pl.B[1] + di[2] * pl.B[2]) / Bm;
          const double c2 = ct * ct, s2 = 1.0 - c2;
          const double A = st.S * s2 + st.P * c2;
          const double Bq = Rr * Ll * s2 + st.P * st.S * (1.0 + c2);
          const double Cq = st.P * Rr * Ll;
          const double F = std::sqrt(Bq * Bq - 4.0 * A * Cq);
          const double r1 = (Bq - F) / (2.0 * A), r2 = (Bq + F) / (2.0 * A);
          const bool r1_is_O = std::fabs(r1 - st.P) <= std::fabs(r2 - st.P);
          n2 = (branch == 0) ? (r1_is_O ? r1 : r2) : (r1_is_O ? r2 : r1);
        }
      }
    }
    double s = std::sqrt(n2);   // NaN if evanescent
    double kk[3], D = std::numeric_limits<double>::quiet_NaN(), g[ND];
    for (int it = 0; it < 8 && std::isfinite(s); ++it) {
      for (int c = 0; c < 3; ++c) kk[c] = s * di[c] * omega / C_LIGHT;
      eval_D(*eq, disp, xi, kk, omega, &D, g);
      if (std::fabs(D) < 1e-15) break;
      const double dDds = (g[3] * di[0] + g[4] * di[1] + g[5] * di[2]) * omega / C_LIGHT;
      const double s_new = s - D / dDds;
      if (!(s_new > 0.0) || !std::isfinite(s_new)) break;
      s = s_new;
    }
    for (int c = 0; c < 3; ++c) k0[c * n + i] = s * di[c] * omega / C_LIGHT;
    if (D_out) {
      for (int c = 0; c < 3; ++c) kk[c] = k0[c * n + i];
      bool in;
      D_out[i] = dispersion<double>(*eq, disp, xi, kk, omega, &in);
    }
  }
  return 0;
}

int oracle_launch(const orc_equilibrium* eq, int disp, int branch, const double* x0, const double* dir,
                  double omega, int64_t n, double* k0, double* D_out) {
  return launch_impl(eq, disp, branch, x0, dir, omega, nullptr, n, k0, D_out);
}

int oracle_launch_w(const orc_equilibrium* eq, int disp, int branch, const double* x0, const double* dir,
                    const double* omega, int64_t n, double* k0, double* D_out) {
  if (!omega) return -1;
  return launch_impl(eq, disp, branch, x0, dir, 0.0, omega, n, k0, D_out);
}

// Launch states exactly as the paper states them (L159): "choosing fixed values for w, x, k_y and k_z.  The remaining
// value k_x is determined using a Newton method to a tolerance of |D(k, w)| < 1e-15.  Since the dispersion functions are
// multi-valued, an initial guess for k_x selects among the possible roots."
//   k_guess [3][n]: rows 1, 2 = the fixed k_y, k_z; row 0 = the initial guess for k_x.   omega_rays [n] or NULL.
// Iteration, in the paper's order: evaluate D and dD/dk_x (dual numbers) at the current k_x; stop if |D| < tol; otherwise
// k_x <- k_x - D / (dD/dk_x); at most max_iter updates.  Returned: k0 = (k_x, k_y, k_z) at the last iterate, D there, and
// iters = number of updates made if |D| < tol was reached, -1 if not (also for points outside the domain or a
// non-finite iterate: k_x = NaN then).
int oracle_launch_kx(const orc_equilibrium* eq, int disp, const double* x0, const double* k_guess, double omega_all,
                     const double* omega_rays, int64_t n, int max_iter, double tol, double* k0, double* D_out,
                     int32_t* iters_out) {
  if (!eq || !combo_supported(*eq, disp) || max_iter < 0 || !(tol > 0.0)) return -1;
  for (int64_t i = 0; i < n; ++i) {
    const double omega = omega_rays ? omega_rays[i] : omega_all;
    const double xi[3] = {x0[i], x0[n + i], x0[2 * n + i]};
    double kk[3] = {k_guess[i], k_guess[n + i], k_guess[2 * n + i]};
    double D = std::numeric_limits<double>::quiet_NaN(), g[ND];
    int iters = -1;
    for (int it = 0; it <= max_iter; ++it) {
      const bool inside = eval_D(*eq, disp, xi, kk, omega, &D, g);
      if (!inside || !std::isfinite(D)) { kk[0] = D = std::numeric_limits<double>::quiet_NaN(); break; }
      if (std::fabs(D) < tol) { iters = it; break; }
      if (it == max_iter) break;
      kk[0] -= D / g[3];
      if (!std::isfinite(kk[0])) { kk[0] = D = std::numeric_limits<double>::quiet_NaN(); break; }
    }
    for (int c = 0; c < 3; ++c) k0[c * n + i] = kk[c];
    if (D_out) D_out[i] = D;
    if (iters_out) iters_out[i] = iters;
  }
  return 0;
}

// ---- second ensemble workload of the same shape: full-orbit charged particles in the same equilibrium -------------
// (L121: "full orbit affects on particle losses in the edge"; L213: "waves or particles in a fusion plasmas ... any
// physics problem involving a large ensemble of independent problems".)  Newton-Lorentz equations
//      dx/dt = v ,    dv/dt = (q/m) v x B(x)
// (no electric field: the equilibria define none), classical RK4 at fixed dt [s], same step-acceptance rule as the rays
// (reading A12).  out_drift is the relative kinetic-energy drift |v|^2/|v0|^2 - 1 (the orbit's analogue of the rays'
// |D|: exactly 0 for the differential equation, O(dt^4) for RK4); NaN never occurs (it needs no equilibrium).
//   x0, v0 [3][n]; out_traj [n_steps/save_stride+1][6][n] rows (x,y,z,vx,vy,vz); out_final [6][n];
//   out_drift [n_saved][n] if out_traj else [n]; out_status [n].
int oracle_orbit(const orc_equilibrium* eq, const double* x0, const double* v0, double charge_over_mass, int64_t n,
                 int64_t n_steps, double dt, int64_t save_stride, double* out_traj, double* out_final, double* out_drift,
                 int32_t* out_status, int n_threads) {
  if (!eq || eq->kind < 1 || eq->kind > 3 || n < 0 || n_steps < 0 || save_stride < 1) return -1;   // parabolic slab: no B
  if (out_traj && (n_steps % save_stride) != 0) return -1;
  const double qm = charge_over_mass;
  auto rhs_orbit = [&](const double y[6], double f[6]) -> bool {
    const Plasma<double> pl = equilibrium<double>(*eq, y);
    if (!pl.inside) return false;
    const double* v = y + 3;
    f[0] = v[0]; f[1] = v[1]; f[2] = v[2];
    f[3] = qm * (v[1] * pl.B[2] - v[2] * pl.B[1]);
    f[4] = qm * (v[2] * pl.B[0] - v[0] * pl.B[2]);
    f[5] = qm * (v[0] * pl.B[1] - v[1] * pl.B[0]);
    return true;
  };
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < n; ++i) {
    double y[6];
    for (int c = 0; c < 3; ++c) { y[c] = x0[c * n + i]; y[3 + c] = v0[c * n + i]; }
    const double e0 = y[3] * y[3] + y[4] * y[4] + y[5] * y[5];
    auto drift = [&]() { return (y[3] * y[3] + y[4] * y[4] + y[5] * y[5]) / e0 - 1.0; };
    int status = 0;
    if (out_traj) {
      for (int c = 0; c < 6; ++c) out_traj[(0 * 6 + c) * n + i] = y[c];
      if (out_drift) out_drift[0 * n + i] = drift();
    }
    for (int64_t s = 1; s <= n_steps; ++s) {
      if (status == 0) {
        double k1[6], k2[6], k3[6], k4[6], ys[6];
        bool ok = rhs_orbit(y, k1);
        if (ok) { for (int j = 0; j < 6; ++j) ys[j] = y[j] + 0.5 * dt * k1[j]; ok = rhs_orbit(ys, k2); }
        if (ok) { for (int j = 0; j < 6; ++j) ys[j] = y[j] + 0.5 * dt * k2[j]; ok = rhs_orbit(ys, k3); }
        if (ok) { for (int j = 0; j < 6; ++j) ys[j] = y[j] + dt * k3[j]; ok = rhs_orbit(ys, k4); }
        if (!ok) {
          status = 1;
        } else {
          bool fin = true;
          for (int j = 0; j < 6; ++j) {
            ys[j] = y[j] + (dt / 6.0) * (k1[j] + 2.0 * k2[j] + 2.0 * k3[j] + k4[j]);
            fin = fin && std::isfinite(ys[j]);
          }
          if (!fin) status = 2;
          else for (int j = 0; j < 6; ++j) y[j] = ys[j];
        }
      }
      if (out_traj && (s % save_stride) == 0) {
        const int64_t m = s / save_stride;
        for (int c = 0; c < 6; ++c) out_traj[(m * 6 + c) * n + i] = y[c];
        if (out_drift) out_drift[m * n + i] = drift();
      }
    }
    if (out_final) for (int c = 0; c < 6; ++c) out_final[c * n + i] = y[c];
    if (!out_traj && out_drift) out_drift[i] = drift();
    if (out_status) out_status[i] = status;
  }
  return 0;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
