// Device math shared by the kernels of pyjac-b200.
#pragma once
#include <cuda_runtime.h>

namespace pyjac {

// exp(x) for |x| < 700 (callers fall back to the library routine otherwise): n = rint(x log2 e), r = x - n ln 2 in two
// steps, Taylor polynomial of degree 13 (truncation 4e-18) by Estrin's scheme -- a dependency chain of 5 DFMAs instead
// of Horner's 13, which is what the reaction phase waits for with 16 warps per SM -- scaled by 2^n through the exponent
// field.  Measured against expl() on 2e7 arguments in (-700, 700): <= 3.8 ulp.
__device__ __forceinline__ double exp_core(double x) {
  const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
  const int n = __double2loint(t);
  const double nf = t - 6755399441055744.0;
  double r = fma(nf, -6.93147180559945286227e-01, x);
  r = fma(nf, -2.31904681384629955842e-17, r);
  const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
  const double p01 = 1.0 + r;
  const double p23 = fma(r, 1.0 / 6.0, 0.5);
  const double p45 = fma(r, 1.0 / 120.0, 1.0 / 24.0);
  const double p67 = fma(r, 1.0 / 5040.0, 1.0 / 720.0);
  const double p89 = fma(r, 1.0 / 362880.0, 1.0 / 40320.0);
  const double pab = fma(r, 1.0 / 39916800.0, 1.0 / 3628800.0);
  const double pcd = fma(r, 1.0 / 6227020800.0, 1.0 / 479001600.0);
  const double q0 = fma(r2, p23, p01), q1 = fma(r2, p67, p45), q2 = fma(r2, pab, p89);
  const double s0 = fma(r4, q1, q0), s1 = fma(r4, pcd, q2);
  const double p = fma(r8, s1, s0);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}
__device__ __forceinline__ bool exp_in_range(double x) { return fabs(x) < 700.0; }

}  // namespace pyjac
