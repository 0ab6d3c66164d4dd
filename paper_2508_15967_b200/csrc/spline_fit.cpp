// spline_fit.cpp -- see spline_fit.h.  Classical moment formulation: unknowns are the second derivatives M_i at the
// nodes; interior rows express continuity of the first derivative, the two not-a-knot conditions (continuity of the
// third derivative at x_1 and x_{n-2}) are eliminated by hand so the system stays tridiagonal, and the Thomas
// recursion solves it.  Intermediate arithmetic is long double; inputs and outputs are double.
#include "spline_fit.h"

namespace rt {

bool fit_cubic_not_a_knot(const double* x, const double* y, std::size_t stride, int n, double* pp) {
  if (n < 4) return false;
  typedef long double real;
  const int m = n - 1;                       // intervals
  std::vector<real> h(m), d(m), M(n), sub(n), dia(n), sup(n), rhs(n);
  for (int i = 0; i < m; ++i) {
    h[i] = (real)x[i + 1] - (real)x[i];
    d[i] = ((real)y[(std::size_t)(i + 1) * stride] - (real)y[(std::size_t)i * stride]) / h[i];
  }
  for (int i = 1; i <= n - 2; ++i) {
    sub[i] = h[i - 1];
    dia[i] = 2 * (h[i - 1] + h[i]);
    sup[i] = h[i];
    rhs[i] = 6 * (d[i] - d[i - 1]);
  }
  // M_0 = (1 + h0/h1) M_1 - (h0/h1) M_2   folded into row 1
  {
    const real r = h[0] / h[1];
    dia[1] += h[0] * (1 + r);
    sup[1] -= h[0] * r;
    sub[1] = 0;
  }
  // M_{n-1} = (1 + hb/ha) M_{n-2} - (hb/ha) M_{n-3}   folded into row n-2
  {
    const real r = h[m - 1] / h[m - 2];
    dia[n - 2] += h[m - 1] * (1 + r);
    sub[n - 2] -= h[m - 1] * r;
    sup[n - 2] = 0;
  }
  // Thomas recursion on rows 1..n-2
  for (int i = 2; i <= n - 2; ++i) {
    const real w = sub[i] / dia[i - 1];
    dia[i] -= w * sup[i - 1];
    rhs[i] -= w * rhs[i - 1];
  }
  M[n - 2] = rhs[n - 2] / dia[n - 2];
  for (int i = n - 3; i >= 1; --i) M[i] = (rhs[i] - sup[i] * M[i + 1]) / dia[i];
  M[0] = M[1] - (h[0] / h[1]) * (M[2] - M[1]);
  M[n - 1] = M[n - 2] + (h[m - 1] / h[m - 2]) * (M[n - 2] - M[n - 3]);
  for (int i = 0; i < m; ++i) {
    pp[i * 4 + 0] = y[(std::size_t)i * stride];
    pp[i * 4 + 1] = (double)(d[i] - h[i] * (2 * M[i] + M[i + 1]) / 6);
    pp[i * 4 + 2] = (double)(M[i] / 2);
    pp[i * 4 + 3] = (double)((M[i + 1] - M[i]) / (6 * h[i]));
  }
  return true;
}

bool fit_bicubic_not_a_knot(const double* R, const double* Z, const double* f, int nR, int nZ, std::vector<double>& pp) {
  if (nR < 4 || nZ < 4) return false;
  const int cR = nR - 1, cZ = nZ - 1;
  // pass 1: along Z at every R node -> cz[(iR*cZ + jZ)*4 + q]
  std::vector<double> cz((std::size_t)nR * cZ * 4);
  for (int i = 0; i < nR; ++i) fit_cubic_not_a_knot(Z, f + (std::size_t)i * nZ, 1, nZ, &cz[(std::size_t)i * cZ * 4]);
  // pass 2: along R, each Z-coefficient treated as nodal data (the 1-D fit is linear in its data)
  pp.assign((std::size_t)cR * cZ * 16, 0.0);
  std::vector<double> piece((std::size_t)cR * 4);
  for (int j = 0; j < cZ; ++j)
    for (int q = 0; q < 4; ++q) {
      fit_cubic_not_a_knot(R, &cz[(std::size_t)j * 4 + q], (std::size_t)cZ * 4, nR, piece.data());
      for (int i = 0; i < cR; ++i)
        for (int p = 0; p < 4; ++p) pp[(((std::size_t)i * cZ + j) * 4 + p) * 4 + q] = piece[(std::size_t)i * 4 + p];
    }
  return true;
}

}  // namespace rt
