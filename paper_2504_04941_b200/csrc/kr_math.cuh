// kr_math.cuh -- lean FP64 primitives of the specialised kernels (B200 has no FP64 SFU path: every exp / divide
// is a string of DFMAs, so they are kept as short as the 1e-9 parity bar allows -- both are ~1 ulp).
#pragma once

// 1/x: MUFU.RCP64H seed (rcp.approx.ftz.f64, ~2^-20) + two Newton steps.  x must be a normal number.
__device__ __forceinline__ double krs_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// exp(x) for x <= 690 (callers clamp, reading R18); flushes to 0 below -708 (results there are < 1e-307 and only ever
// multiply number densities).  Cody-Waite reduction by ln 2, degree-13 Taylor polynomial on |r| <= 0.347
// (remainder < 5e-18), exponent patched into the high word.
__device__ __forceinline__ double krs_exp_core(double x) {
  const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
  const int n = __double2loint(t);
  const double fn = t - 6755399441055744.0;
  double r = fma(fn, -6.93147180369123816490e-01, x);
  r = fma(fn, -1.90821492927058770002e-10, r);
  double p = 1.0 / 6227020800.0;
  p = fma(p, r, 1.0 / 479001600.0);
  p = fma(p, r, 1.0 / 39916800.0);
  p = fma(p, r, 1.0 / 3628800.0);
  p = fma(p, r, 1.0 / 362880.0);
  p = fma(p, r, 1.0 / 40320.0);
  p = fma(p, r, 1.0 / 5040.0);
  p = fma(p, r, 1.0 / 720.0);
  p = fma(p, r, 1.0 / 120.0);
  p = fma(p, r, 1.0 / 24.0);
  p = fma(p, r, 1.0 / 6.0);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  const double s = __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
  return (x < -708.0) ? 0.0 : s;
}

__device__ __forceinline__ double krs_exp(double lnk) { return krs_exp_core(lnk > 690.0 ? 690.0 : lnk); }
