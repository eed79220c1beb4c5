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
//   atan2_pos : atan2(y, x) for y >= 0 (result in [0, π]); one reciprocal, reduction to |t| <= tan(π/8), odd polynomial.
// Constants that are not exactly representable in the 32 high bits of a double cannot be instruction immediates on
// sm_100a: written as literals they are rebuilt with two UMOV/IMAD.MOV per use (a quarter of all issued instructions in
// the first ncu capture, profiles/r1a_ncu_dense.md).  They live in __constant__ arrays instead, laid out in use order so
// that one LDCU.128 fetches two of them into uniform registers.
// None of this is shared with the oracle (libm / libquadmath); coefficients: csrc/gen_poly.py.
#pragma once
#include <cuda_runtime.h>

namespace pt {

// [0..6] sin: S(r²), sin r = r + r³ S;  [7..13] cos: C(r²), cos r = 1 - r²/2 + r⁴ C;  [14] 2/π, [15] π/2 hi, [16] π/2 lo
__constant__ double kTrig[18] = {
    -7.6471637318198164759e-13, 1.6059043836821614599e-10, -2.5052108385441718775e-08, 2.7557319223985890653e-06,
    -1.9841269841269841270e-04, 8.3333333333333333333e-03, -1.6666666666666666667e-01,
    4.7794773323873852974e-14, -1.1470745597729724714e-11, 2.0876756987868098979e-09, -2.7557319223985890653e-07,
    2.4801587301587301587e-05, -1.3888888888888888889e-03, 4.1666666666666666667e-02,
    0.63661977236758134308, 1.57079632679489655800e+00, 6.12323399573676603587e-17, 0.0};

// atan(t) = t + t u P(u), u = t², |t| <= tan(π/8): P coefficients u^10 ... u^0; then [11] tan(π/8), [12] π/4, [13] π/2, [14] π
__constant__ double kAtan[16] = {
    -0.017805397205419445228, 0.037965257453865936236, -0.050351024566015518428, 0.058468782973308725201,
    -0.066629518136291900881, 0.076920453309022249521, -0.090908968090640270761, 0.11111110744919658237,
    -0.14285714279250244942, 0.19999999999940891462, -0.33333333333333121163,
    0.41421356237309504880, 0.78539816339744830962, 1.57079632679489661923, 3.14159265358979323846, 0.0};

// π, 2π, π/2, 1/π, 1/(2π), 2/3, 1/3, 1/(9π), 2/(9π)
enum { C_PI = 0, C_TWOPI, C_HALFPI, C_INVPI, C_HALF_INVPI, C_TWOTHIRDS, C_THIRD, C_INV9PI, C_2INV9PI };
__constant__ double kC[10] = {3.14159265358979323846, 6.28318530717958647692, 1.57079632679489661923,
                              0.31830988618379067154, 0.15915494309189533577, 0.66666666666666666667,
                              0.33333333333333333333, 0.035367765131532296838, 0.070735530263064593676, 0.0};

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

// sin and cos of r for |r| <= π/4 (no range reduction).
__device__ __forceinline__ void sincos_kernel(double r, double* sn, double* cs) {
  const double r2 = r * r;
  double ps = kTrig[0], pc = kTrig[7];
#pragma unroll
  for (int j = 1; j < 7; ++j) {
    ps = fma(ps, r2, kTrig[j]);
    pc = fma(pc, r2, kTrig[7 + j]);
  }
  *sn = fma(ps * r2, r, r);
  *cs = fma(pc * r2, r2, fma(-0.5, r2, 1.0));
}

// sin and cos of x for |x| up to ~1e3 (k = round(2x/π) stays small, so the two-term reduction is exact to ~1e-19 |k|).
__device__ __forceinline__ void sincos_bounded(double x, double* sn, double* cs) {
  const double magic = 6755399441055744.0;             // 1.5 * 2^52: adds round-to-nearest-integer in the low word
  const double kd_m = fma(x, kTrig[14], magic);
  const int k = __double2loint(kd_m);
  const double kd = kd_m - magic;
  double r = fma(-kd, kTrig[15], x);
  r = fma(-kd, kTrig[16], r);
  double s, c;
  sincos_kernel(r, &s, &c);
  // quadrant: k mod 4 = 0: (s, c); 1: (c, -s); 2: (-s, -c); 3: (-c, s)
  const double ss = (k & 1) ? c : s;
  const double cc = (k & 1) ? s : c;
  *sn = (k & 2) ? -ss : ss;
  *cs = ((k + 1) & 2) ? -cc : cc;
}

// atan2(y, x) for y >= 0, (x, y) != (0, 0), both finite: the angle in [0, π].
// r = min/max in [0,1]; for r > tan(π/8) the argument is moved to (r-1)/(r+1) = (min-max)/(min+max) and π/4 added, which
// needs no second reciprocal because numerator and denominator are chosen before the single division.
__device__ __forceinline__ double atan2_pos(double y, double x) {
  const double ax = fabs(x);
  const bool swap = y > ax;
  const double mn = swap ? ax : y, mx = swap ? y : ax;
  const bool big = mn > kAtan[11] * mx;
  const double num = big ? mn - mx : mn;
  const double den = big ? mn + mx : mx;
  const double t = num * rcp_fast(den);
  const double u = t * t;
  double p = kAtan[0];
#pragma unroll
  for (int j = 1; j < 11; ++j) p = fma(p, u, kAtan[j]);
  double a = fma(t * u, p, t);           // atan(t), |t| <= tan(π/8)
  a = big ? a + kAtan[12] : a;           // angle of (mx, mn) in [0, π/4]
  a = swap ? kAtan[13] - a : a;          // angle of (|x|, y) in [0, π/2]
  return x < 0.0 ? kAtan[14] - a : a;
}

}  // namespace pt
