// Test shim (not product code): C entry points around csrc/spline_fit.h so that the CPU test suite can drive the
// library's host-side spline fit through ctypes without a GPU (tests/test_spline_fit.py compiles this with g++).
#include <cstring>
#include <vector>

#include "../paper_2508_15967_b200/csrc/spline_fit.h"

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

}  // extern "C"
