// spline_fit.h -- host-side (fp64) not-a-knot cubic spline fitting for the grid equilibrium (PAPER.md L60:
// "piecewise constant nodes ... used to implement spline interpolation"; reading A10).  Runs once per
// rt_create_equilibrium; the kernels only ever see the per-cell polynomial pieces produced here.
#pragma once

#include <cstddef>
#include <vector>

namespace rt {

// 1-D: nodal y[i] at strictly increasing x[i], i < n (n >= 4) -> pieces pp[i*4 + m], i < n-1, multiplying (x - x_i)^m.
// `stride` is the distance between consecutive y samples in memory.  Returns false if n < 4.
bool fit_cubic_not_a_knot(const double* x, const double* y, std::size_t stride, int n, double* pp);

// 2-D tensor product on nodes R[i], Z[j]; f is row-major [nR][nZ].  Output pp[((iR*(nZ-1) + iZ)*4 + p)*4 + q]
// multiplying (R - R_iR)^p (Z - Z_iZ)^q.  Returns false if nR < 4 or nZ < 4.
bool fit_bicubic_not_a_knot(const double* R, const double* Z, const double* f, int nR, int nZ, std::vector<double>& pp);

}  // namespace rt
