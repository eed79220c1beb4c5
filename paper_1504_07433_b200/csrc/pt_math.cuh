// pt_math.cuh — lean fp64 primitives for the hot loops.
//
// The FP64 pipe of an SM issues one warp instruction every two cycles, and every instruction of any kind costs an issue
// slot, so the hot loops avoid the CUDA math library's general-purpose entry points (argument checks, slow-path calls,
// Payne–Hanek tables) where the arguments are known to be tame:
//   rcp_fast / rsqrt_fast / sqrt_fast / div_fast : MUFU seed (rcp/rsqrt.approx.ftz.f64, ~2^-19) + one third-order
//       Newton step (error ~ seed^3 ~ 2^-57) [+ one residual correction]; <= 1-2 ulp; operands must be normal, finite, > 0
//       for the roots.
//   sincos_bounded : |x| <= ~1e3; two-constant Cody–Waite reduction by π/2 and Taylor polynomials on |r| <= π/4
//       (sin through r^15, cos through r^16: truncation < 5e-17).
// None of this is shared with the oracle (libm / libquadmath).
#pragma once
#include <cuda_runtime.h>

namespace pt {

__device__ __forceinline__ double rcp_seed(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
__device__ __forceinline__ double rsqrt_seed(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}

// 1/x, |x| normal.  y0(1 + e + e²), e = 1 - x y0.
__device__ __forceinline__ double rcp_fast(double x) {
  const double y0 = rcp_seed(x);
  const double e = fma(-x, y0, 1.0);
  const double e2 = fma(e, e, e);
  return fma(y0, e2, y0);
}

// a/b with one residual correction (<= 1 ulp).
__device__ __forceinline__ double div_fast(double a, double b) {
  const double y = rcp_fast(b);
  const double q = a * y;
  const double r = fma(-q, b, a);
  return fma(r, y, q);
}

// 1/sqrt(x), x normal > 0.  y0(1 + h/2 + 3h²/8), h = 1 - x y0².
__device__ __forceinline__ double rsqrt_fast(double x) {
  const double y0 = rsqrt_seed(x);
  const double h = fma(-x, y0 * y0, 1.0);
  const double c = fma(0.375, h, 0.5);
  return fma(c, y0 * h, y0);
}

// sqrt(x), x normal > 0 (x == 0 must be handled by the caller).
__device__ __forceinline__ double sqrt_fast(double x) {
  const double y = rsqrt_fast(x);
  const double s = x * y;
  const double r = fma(-s, s, x);
  return fma(r, 0.5 * y, s);
}

// sin and cos of x for |x| up to ~1e3 (k = round(2x/π) stays small, so the two-term reduction is exact to ~1e-19 |k|).
__device__ __forceinline__ void sincos_bounded(double x, double* sn, double* cs) {
  const double two_over_pi = 0.63661977236758134308;
  const double pio2_hi = 1.57079632679489655800e+00;   // π/2 rounded to double
  const double pio2_lo = 6.12323399573676603587e-17;   // π/2 - pio2_hi
  const double magic = 6755399441055744.0;             // 1.5 * 2^52: adds round-to-nearest-integer in the low word
  const double kd_m = fma(x, two_over_pi, magic);
  const int k = __double2loint(kd_m);
  const double kd = kd_m - magic;
  double r = fma(-kd, pio2_hi, x);
  r = fma(-kd, pio2_lo, r);
  const double r2 = r * r;
  // sin r = r + r³ (s3 + r²(s5 + ... )) ; cos r = 1 - r²/2 + r⁴ (c4 + r²(c6 + ...))   (Taylor coefficients ±1/n!)
  double ps = 7.6471637318198164759e-13;              //  1/15!
  ps = fma(ps, r2, -1.6059043836821614599e-10);       // -1/13!
  ps = fma(ps, r2, 2.5052108385441718775e-08);        //  1/11!
  ps = fma(ps, r2, -2.7557319223985890653e-06);       // -1/9!
  ps = fma(ps, r2, 1.9841269841269841270e-04);        //  1/7!
  ps = fma(ps, r2, -8.3333333333333333333e-03);       // -1/5!
  ps = fma(ps, r2, 1.6666666666666666667e-01);        //  1/3!  (sign applied below)
  double pc = 4.7794773323873852974e-14;              //  1/16!
  pc = fma(pc, r2, -1.1470745597729724714e-11);       // -1/14!
  pc = fma(pc, r2, 2.0876756987868098979e-09);        //  1/12!
  pc = fma(pc, r2, -2.7557319223985890653e-07);       // -1/10!
  pc = fma(pc, r2, 2.4801587301587301587e-05);        //  1/8!
  pc = fma(pc, r2, -1.3888888888888888889e-03);       // -1/6!
  pc = fma(pc, r2, 4.1666666666666666667e-02);        //  1/4!
  const double s = fma(-ps * r2, r, r);                // r - r³ (1/6 - ...)
  const double c = fma(pc * r2, r2, fma(-0.5, r2, 1.0));
  // quadrant: k mod 4 = 0: (s, c); 1: (c, -s); 2: (-s, -c); 3: (-c, s)
  const double ss = (k & 1) ? c : s;
  const double cc = (k & 1) ? s : c;
  *sn = (k & 2) ? -ss : ss;
  *cs = ((k + 1) & 2) ? -cc : cc;
}

}  // namespace pt
