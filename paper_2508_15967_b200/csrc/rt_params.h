// rt_params.h -- step a0 of the hot path: fold the wave frequency w into O(1) constants, once per call, in fp64 on the
// host (Eq. 6: n = c k / w; L189: w_p, W_c per species), so that every device-side quantity stays O(1)
// in fp32 as well.  Host code only; no CUDA dependency.
#pragma once

#include <cstring>

#include "../../include/rt.h"
#include "rt_math.cuh"

namespace rt {

// CODATA-2022 numerals (reading A6)
constexpr double kC = 299792458.0;          // m/s
constexpr double kQe = 1.602176634e-19;     // C
constexpr double kMe = 9.1093837139e-31;    // kg
constexpr double kEps0 = 8.8541878188e-12;  // F/m

// Range of the series the hot loop uses for the ion terms of the Stix elements (rt_math.cuh: disp_coefs, SERIES): the
// largest Y2 = (W_ce/w)^2 up to which every term dropped from
//   sig  = e1   + mu   e2   -> e1   + (mu + mu^3 Y2)        dropped: mu z^2/(1-z)              z = mu^2 Y2, e2 = 1/(1-z)
//   sig' = e1^2 + mu^3 e2^2 -> e1^2 + mu^3                  dropped: mu^3 (2z - z^2)/(1-z)^2
//   del  = mu^2 e2   - e1   -> (mu^2 + mu^4 Y2) - e1        dropped: mu^2 z^2/(1-z)
//   del' = mu^4 e2^2 - e1^2 -> mu^4 - e1^2                  dropped: mu^4 (2z - z^2)/(1-z)^2
// stays below `tol` (a quarter ulp of the working precision) relative to the smallest magnitude the electron term
// e1 = 1/(1 - Y2) (resp. e1^2) takes on [0, Y2]: 1/max(1, Y2 - 1).  The bounds grow with Y2, so bisection finds the cap.
// Deuterium, fp64: Y2 < 3.3 (w > 0.55 W_ce); electrons only (mu = 0): no limit.
inline double series_cap(double mu, double tol) {
  if (!(mu > 0.0)) return 1.7e308;
  auto ok = [&](double Y2) {
    const double z = mu * mu * Y2;
    if (!(z < 0.5)) return false;
    const double m = Y2 > 2.0 ? Y2 - 1.0 : 1.0;                          // 1 / min |e1| on [0, Y2] (ignoring the pole)
    const double d1 = z * z / (1.0 - z), d2 = (2.0 * z - z * z) / ((1.0 - z) * (1.0 - z));
    return mu * d1 * m <= tol && mu * mu * mu * d2 * m * m <= tol;        // the del / del' bounds are these times mu
  };
  double lo = 0.0, hi = 1.0;
  while (ok(hi) && hi < 1e300) { lo = hi; hi *= 2.0; }
  for (int it = 0; it < 100; ++it) { const double mid = 0.5 * (lo + hi); (ok(mid) ? lo : hi) = mid; }
  return lo;
}

// d: the equilibrium's scalars; rho_max: resolved domain radius (tokamak); ne_scale: what the grid's n_e table was
// divided by; psi_pp / prof_pp: device tables of element type T (grid kind), else NULL.
template <class T>
Params<T> fold_params(const rt_equilibrium_desc& d, double rho_max, double ne_scale, double omega, const T* psi_pp,
                      const T* prof_pp) {
  Params<T> P;
  std::memset(&P, 0, sizeof(P));
  const double alpha = kQe * kQe / (kEps0 * kMe * omega * omega);       // X_e = alpha n_e
  const double nscale = (d.kind == RT_EQ_GRID_RZ) ? ne_scale : d.n_ref;
  const double xs = alpha * nscale;
  P.xs = (T)xs;
  P.xsh = (T)(0.5 * xs);
  const double wce_per_T = kQe / (kMe * omega);
  P.beta = (T)(wce_per_T * wce_per_T);
  P.beta2 = (T)(2.0 * wce_per_T * wce_per_T);
  const double mu = (d.ion_mass > 0.0) ? d.ion_charge * kMe / d.ion_mass : 0.0;
  P.mu = (T)mu; P.mu2 = (T)(mu * mu); P.mu3 = (T)(mu * mu * mu); P.mu4 = (T)(mu * mu * mu * mu);
  P.one_plus_mu = (T)(1.0 + mu);
  P.y2cap = (T)series_cap(mu, sizeof(T) == 8 ? 0x1p-54 : 0x1p-25);
  P.k2n = (T)(kC / omega);
  P.n2k = (T)(omega / kC);
  P.par_g = (T)(d.L != 0.0 ? xs / (d.L * d.L) : 0.0);
  P.x_foot = (T)d.x_foot;
  P.lin_gx = (T)(d.L_ramp != 0.0 ? -xs / d.L_ramp : 0.0);
  P.lin_gxh = (T)(d.L_ramp != 0.0 ? -0.5 * xs / d.L_ramp : 0.0);
  P.B0R0 = (T)(d.B0 * d.R0);
  P.sB0 = (T)(wce_per_T * d.B0);                 // sqrt(beta) B0: the field in units of the electron cyclotron ratio
  P.sB0R0 = (T)(wce_per_T * d.B0 * d.R0);
  P.R0 = (T)d.R0;
  P.B0 = (T)d.B0;
  const double inv_a2 = d.a != 0.0 ? 1.0 / (d.a * d.a) : 0.0;
  P.inv_a2 = (T)inv_a2;
  P.q0 = (T)d.q0;
  P.q1_a2 = (T)(d.q1 * inv_a2);
  P.two_q1_a2 = (T)(2.0 * d.q1 * inv_a2);
  P.p_exp = (T)d.p_exp;
  P.two_xs_a2 = (T)(2.0 * xs * inv_a2);
  P.tok_gxh = (T)(-d.p_exp * xs * inv_a2);
  P.rmax2 = (T)(rho_max * rho_max * d.a * d.a);
  if (d.kind == RT_EQ_GRID_RZ) {
    const double hR = (d.Rmax - d.Rmin) / (d.nR - 1), hZ = (d.Zmax - d.Zmin) / (d.nZ - 1);
    const double hP = (d.psi_max - d.psi_min) / (d.nPsi - 1);
    P.Rmin = (T)d.Rmin; P.Rmax = (T)d.Rmax; P.Zmin = (T)d.Zmin; P.Zmax = (T)d.Zmax;
    P.hR = (T)hR; P.hZ = (T)hZ; P.inv_hR = (T)(1.0 / hR); P.inv_hZ = (T)(1.0 / hZ);
    P.psi_min = (T)d.psi_min; P.psi_max = (T)d.psi_max; P.hP = (T)hP; P.inv_hP = (T)(1.0 / hP);
    P.nRc = d.nR - 1; P.nZc = d.nZ - 1; P.nPc = d.nPsi - 1;
    P.psi_pp = psi_pp;
    P.prof_pp = prof_pp;
  }
  return P;
}

}  // namespace rt
