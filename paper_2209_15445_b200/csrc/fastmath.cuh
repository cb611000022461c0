// Lean fp64 math for the step kernels.  The transport path is bound by instruction issue, not by HBM
// (DESIGN.md §5), and libdevice's log / division sequences spend a third of their instructions on
// special cases that cannot occur here (zero, negative, subnormal, infinite or NaN arguments).  These
// versions assume positive, finite, normal arguments and are accurate to a few 1e-16 relative, far
// inside the 1e-12 parity tolerance against the oracle's libm (tests/parity.py).
#pragma once
#include <cuda_runtime.h>

namespace adept {

// 1/x for positive normal x: MUFU.RCP64H seed (2^-23) + two Newton steps.
__device__ __forceinline__ double rcp_pos(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// a / b for normal b > 0 and finite a, within 1 ulp
__device__ __forceinline__ double div_pos(double a, double b) {
  const double r = rcp_pos(b);
  const double q = a * r;
  return fma(fma(-b, q, a), r, q);
}

// ln x for positive, finite, normal x.  x = m 2^e with m in [sqrt(1/2), sqrt(2)); with f = (m-1)/(m+1),
// ln m = 2 atanh f = 2f (1 + f^2/3 + f^4/5 + ...), |f| <= 0.1716, truncated after f^20 (next term 6e-19).
__device__ __forceinline__ double log_pos(double x) {
  int hi = __double2hiint(x);
  const int lo = __double2loint(x);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;
  if (hi >= 0x3ff6a09f) { hi -= 0x00100000; e += 1; }
  const double m = __hiloint2double(hi, lo);
  const double a = m - 1.0, b = m + 1.0;
  const double r = rcp_pos(b);
  double f = a * r;
  f = fma(fma(-b, f, a), r, f);
  const double s = f * f;
  double p = 1.0 / 21.0;
  p = fma(p, s, 1.0 / 19.0);
  p = fma(p, s, 1.0 / 17.0);
  p = fma(p, s, 1.0 / 15.0);
  p = fma(p, s, 1.0 / 13.0);
  p = fma(p, s, 1.0 / 11.0);
  p = fma(p, s, 1.0 / 9.0);
  p = fma(p, s, 1.0 / 7.0);
  p = fma(p, s, 1.0 / 5.0);
  p = fma(p, s, 1.0 / 3.0);
  const double f2 = f + f;
  const double lm = fma(f2, p * s, f2);
  return fma(static_cast<double>(e), 0.6931471805599453094, lm);
}

}  // namespace adept
