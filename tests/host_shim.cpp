// Test shim (not product code): C entry points around the library's HOST-side logic -- the spline fit (csrc/spline_fit.h)
// and the per-call constant folding (csrc/rt_params.h, step a0) -- so that the CPU test suite can drive them through
// ctypes without a GPU (tests/test_host_logic.py compiles this with g++; rt_math.cuh compiles as plain C++ here).
#include <cstring>
#include <vector>

#include "../paper_2508_15967_b200/csrc/rt_params.h"
#include "../paper_2508_15967_b200/csrc/spline_fit.h"

// out[0..15] = xs, xsh, beta, beta2, mu, mu2, one_plus_mu, k2n, n2k, par_g, lin_gx, lin_gxh, sB0, sB0R0, tok_gxh, rmax2
template <class T>
static void fold_to(const rt_equilibrium_desc* d, double rho_max, double omega, double* out) {
  const rt::Params<T> P = rt::fold_params<T>(*d, rho_max, 1.0, omega, nullptr, nullptr);
  const T v[16] = {P.xs, P.xsh, P.beta, P.beta2, P.mu, P.mu2, P.one_plus_mu, P.k2n, P.n2k, P.par_g, P.lin_gx, P.lin_gxh,
                   P.sB0, P.sB0R0, P.tok_gxh, P.rmax2};
  for (int i = 0; i < 16; ++i) out[i] = (double)v[i];
}

extern "C" {

int shim_fit_cubic(const double* x, const double* y, long stride, int n, double* pp) {
  return rt::fit_cubic_not_a_knot(x, y, (std::size_t)stride, n, pp) ? 0 : -1;
}

// pp must hold (nR-1)*(nZ-1)*16 doubles
int shim_fit_bicubic(const double* R, const double* Z, const double* f, int nR, int nZ, double* pp) {
  std::vector<double> out;
  if (!rt::fit_bicubic_not_a_knot(R, Z, f, nR, nZ, out)) return -1;
  std::memcpy(pp, out.data(), out.size() * sizeof(double));
  return (int)out.size();
}

// the largest Y2 up to which the hot loop evaluates the ion terms of the Stix elements by their series (rt_params.h)
double shim_series_cap(double mu, double tol) { return rt::series_cap(mu, tol); }

void shim_fold_params(const rt_equilibrium_desc* d, double rho_max, double omega, int fp32, double* out) {
  if (fp32) fold_to<float>(d, rho_max, omega, out); else fold_to<double>(d, rho_max, omega, out);
}

}  // extern "C"
