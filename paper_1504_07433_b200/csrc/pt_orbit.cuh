// pt_orbit.cuh — per-parameter-vector constants and the fused orbit stage (time -> folded phase -> projected separation).
//
// The paper gives no orbit equations (P:L31 only names the solvers); R5 fixes the geometry: standard two-body
// projection, observer on +Z, t0 = time of inferior conjunction (true anomaly π/2 - w), circular routine for e == 0 and
// Newton's method on Kepler's equation for e > 0.  Two steps are pinned to IEEE double operations (H1, H2):
// the subsample time and the phase fold.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#include "pt_math.cuh"

namespace pt {

constexpr double kTwoPi = 6.28318530717958647692;   // host-side / setup use; hot paths read kC[]
constexpr double kPi = 3.14159265358979323846;

enum PvFlags : int { PV_BAD = 1, PV_CIRCULAR = 2, PV_NEVER = 4, PV_ALWAYS = 8, PV_OFF_TABLE = 16, PV_SLOWDIV = 32 };

// Constants of one parameter vector (shared memory, one per block).
struct PvConst {
  double t0, P, invP;
  double a, cosi, e, sinw, cosw, rt1me2, Mtr, sin_e, cos_e;
  double khat;
  double ph_lo, ph_hi;   // conservative phase window of the transit (cycles, relative to conjunction), sample-level
  double ex_lo, ex_hi;   // the same widened by half an exposure: exposure-level test on the exposure centre
  double win_mid, win_half;   // centre / half-width of [ex_lo, ex_hi]; half = -inf: never in transit, +inf: always
  int flags;
};

// H1: phase fold — one subtraction, one IEEE division, round-to-nearest-even, one (exact) subtraction.
// The correctly rounded quotient is obtained without the generic division sequence: with y = RN(1/P) (computed once per
// parameter vector), q0 = RN(x y), r = x - q0 P (exact in an FMA), q = RN(q0 + r y) equals RN(x/P) for every x
// (Markstein's theorem) unless the significand of P is all ones; that one case takes the division instruction sequence.
__device__ __forceinline__ double fold_phase(double t, double t0, double P, double invP, bool slow_div) {
  const double xs = __dsub_rn(t, t0);
  double x;
  if (slow_div) {
    x = __ddiv_rn(xs, P);
  } else {
    const double q0 = __dmul_rn(xs, invP);
    const double r = __fma_rn(-q0, P, xs);
    x = __fma_rn(r, invP, q0);
  }
  return __dsub_rn(x, rint(x));
}

// H2: offset of subsample s inside an exposure (midpoints of n_ss equal parts); ts = t + off, no contraction.
__device__ __forceinline__ double subsample_offset(int s, int n_ss, double t_exp) {
  return __dmul_rn(t_exp, __dsub_rn(__ddiv_rn((double)s + 0.5, (double)n_ss), 0.5));
}

// Cheap window test on an exposure time: can any subsample of it be in transit?  It is only ever used to SKIP exposures
// whose flux is exactly 1, so it must never say "no" wrongly: it folds with (t-t0)*(1/P) instead of the pinned division
// and rounds with the 1.5*2^52 trick, both of which differ from the pinned fold by less than 1e-15 |x| cycles — the
// window is widened by exactly that (plus the fixed 1e-7 margin built into mid/half).  For |x| >= 2^51 the widened
// half-width exceeds 2, so the test passes whatever the rounding did; NaN/inf times fail it (flux 1, as in the oracle,
// where every comparison with NaN is false).  6 FP64-pipe instructions per exposure.
__device__ __forceinline__ bool in_window(double t, double t0, double invP, double mid, double half) {
  const double x = (t - t0) * invP;
  const double magic = 6755399441055744.0;   // 1.5 * 2^52
  const double r = __dsub_rn(__dadd_rn(x, magic), magic);
  const double ph = x - r;
  return fabs(ph - mid) < fma(fabs(x), 0x1p-50, half);
}

// Eccentric anomaly from mean anomaly M in (-π, π] by Newton's method.  Starter: for e <= 0.8 the third-order
// guess M + e sin M / (1 - sin(M+e) + sin M) (<= 6 steps); above that E0 = M ± e, which lies on the convex side of the
// root so Newton descends monotonically (<= 12 steps at e = 0.999).
__device__ __forceinline__ void kepler_newton(double M, double e, double sin_e, double cos_e, double* sinE, double* cosE) {
  double E;
  double sE, cE, dE;
  if (e <= 0.8) {
    double sM, cM;
    sincos_bounded(M, &sM, &cM);
    const double sMe = fma(sM, cos_e, cM * sin_e);   // sin(M + e), (sin e, cos e) are per-orbit constants
    E = fma(e * sM, rcp_fast(1.0 - sMe + sM), M);
  } else {
    E = M + copysign(e, M);
  }
  const double tol = 0x1p-30 * (1.0 - e);
  bool conv = false;
  sincos_bounded(E, &sE, &cE);
#pragma unroll 1
  for (int it = 0; it < 32; ++it) {
    const double f = E - fma(e, sE, M);
    const double fp = fma(-e, cE, 1.0);
    dE = f * rcp_fast(fp);
    E -= dE;
    const double ad = fabs(dE);
    if (ad < tol) { conv = true; break; }   // the step just applied squares the error: converged to rounding
    if (ad < 0x1p-7) {
      // small step: rotate (sin E, cos E) by -dE with short series (sin through dE^5, cos through dE^6: the neglected
      // terms are below 4e-19) instead of a full sincos
      const double d2 = dE * dE;
      const double sd = dE * fma(d2, fma(d2, 1.0 / 120.0, -1.0 / 6.0), 1.0);
      const double cd = fma(d2, fma(d2, fma(d2, -1.0 / 720.0, 1.0 / 24.0), -0.5), 1.0);
      const double ns = fma(sE, cd, -cE * sd);
      cE = fma(cE, cd, sE * sd);
      sE = ns;
    } else {
      sincos_bounded(E, &sE, &cE);
    }
  }
  if (conv) {   // sin/cos of E - dE to first order in dE (|dE| < 1e-9: the neglected term is < 5e-19)
    *sinE = fma(-cE, dE, sE);
    *cosE = fma(sE, dE, cE);
  } else {
    sincos_bounded(E, sinE, cosE);
  }
}

// Signed projected separation at pinned folded phase ph (cycles): +z in front of the star, -z behind.
__device__ __forceinline__ double orbit_z_signed(const PvConst& c, double ph) {
  if (c.flags & PV_CIRCULAR) {
    if (fabs(ph) <= 0.125) {
      // within an eighth of a cycle of conjunction (every transit of a/R* > 1.5): no range reduction, no cosine;
      // z² = a² (cos²i + sin²i sin²φ), planet in front (cos φ > 0)
      const double r = kC[C_TWOPI] * ph, r2 = r * r;
      double ps = kTrig[0];
#pragma unroll
      for (int j = 1; j < 7; ++j) ps = fma(ps, r2, kTrig[j]);
      const double sn = fma(ps * r2, r, r);
      const double ci2 = c.cosi * c.cosi;
      return c.a * sqrt_fast(fmax(fma(1.0 - ci2, sn * sn, ci2), 0x1p-1000));
    }
    double sn, cs;
    sincos_bounded(kC[C_TWOPI] * ph, &sn, &cs);
    const double cc = c.cosi * cs;
    const double z = c.a * sqrt_fast(fmax(fma(sn, sn, cc * cc), 0x1p-1000));
    return cs > 0.0 ? z : -z;
  }
  double M = fma(kC[C_TWOPI], ph, c.Mtr);
  if (M > kC[C_PI]) M -= kC[C_TWOPI];
  if (M <= -kC[C_PI]) M += kC[C_TWOPI];
  double sE, cE;
  kepler_newton(M, c.e, c.sin_e, c.cos_e, &sE, &cE);
  const double x = cE - c.e, y = c.rt1me2 * sE;
  const double A = c.cosw * x - c.sinw * y;   // (r/a) cos(w+f)
  const double B = c.sinw * x + c.cosw * y;   // (r/a) sin(w+f)
  const double Bc = B * c.cosi;
  const double z = c.a * sqrt_fast(fmax(fma(A, A, Bc * Bc), 0x1p-1000));
  return B > 0.0 ? z : -z;
}

// ---- the other orbit routines of P:L31 (R19): fixed-point iteration and the two series
// approximations of the equation of the centre, selectable per call (pt_orbit_z_solver) or by the eccentricity.
enum OrbitSolver : int { SOLVER_EXACT = 0, SOLVER_NEWTON = 1, SOLVER_ITER = 2, SOLVER_PS3 = 3, SOLVER_PS5 = 4, SOLVER_FAST = 5 };

// The routine the eccentricity selects: exact = circular for e == 0 else Newton; fast = the cheapest routine whose
// truncation error in the true anomaly is below 2e-9 rad (order 3: 1.5 e^4, e <= 0.006; order 5: 2.2 e^6, e <= 0.03).
__host__ __device__ __forceinline__ int dispatch_solver(int solver, double e) {
  if (solver == SOLVER_FAST) return e == 0.0 ? SOLVER_EXACT : (e <= 0.006 ? SOLVER_PS3 : (e <= 0.03 ? SOLVER_PS5 : SOLVER_NEWTON));
  return solver;
}

// Coefficients of sin kM, k = 1..5, of f - M truncated after e^3 (order 3) or e^5 (classical expansion, e.g. Murray &
// Dermott 1999 eq. 2.88): once per parameter vector.
__device__ __forceinline__ void series_coefficients(double e, int order, double* c) {
  const double e2 = e * e, e3 = e2 * e;
  if (order == 3) {
    c[0] = 2.0 * e - 0.25 * e3; c[1] = 1.25 * e2; c[2] = (13.0 / 12.0) * e3; c[3] = 0.0; c[4] = 0.0;
  } else {
    const double e4 = e2 * e2, e5 = e4 * e;
    c[0] = 2.0 * e - 0.25 * e3 + (5.0 / 96.0) * e5;
    c[1] = 1.25 * e2 - (11.0 / 24.0) * e4;
    c[2] = (13.0 / 12.0) * e3 - (43.0 / 64.0) * e5;
    c[3] = (103.0 / 96.0) * e4;
    c[4] = (1097.0 / 960.0) * e5;
  }
}

// Signed projected separation by one of the non-default routines: SOLVER_ITER (E <- M + e sin E from E = M until it moves
// by less than an ulp; linear convergence with rate e) or SOLVER_PS3 / SOLVER_PS5 (series for the true anomaly, `ser` from
// series_coefficients; sin kM by the Chebyshev recurrence from one sincos).
__device__ __forceinline__ double orbit_z_signed_alt(const PvConst& c, const double* ser, double ph, int solver) {
  double M = fma(kC[C_TWOPI], ph, c.Mtr);
  if (M > kC[C_PI]) M -= kC[C_TWOPI];
  if (M <= -kC[C_PI]) M += kC[C_TWOPI];
  double A, B;
  if (solver == SOLVER_ITER) {
    double E = M, sE, cE, dprev = CUDART_INF;
#pragma unroll 1
    for (int it = 0; it < 100000; ++it) {
      sincos_bounded(E, &sE, &cE);
      const double En = fma(c.e, sE, M);
      const double d = fabs(En - E);
      E = En;
      // a fixed point to rounding: the step is below an ulp, or it no longer shrinks (the last bit may flip for ever)
      if (d <= 0x1p-53 * (fabs(E) + 1.0) || (d >= dprev && d <= 0x1p-48 * (fabs(E) + 1.0))) break;
      dprev = d;
    }
    sincos_bounded(E, &sE, &cE);
    const double x = cE - c.e, y = c.rt1me2 * sE;
    A = c.cosw * x - c.sinw * y;
    B = c.sinw * x + c.cosw * y;
  } else {
    double s1, c1;
    sincos_bounded(M, &s1, &c1);
    const double tc = 2.0 * c1;
    const double s2 = tc * s1, s3 = fma(tc, s2, -s1), s4 = fma(tc, s3, -s2), s5 = fma(tc, s4, -s3);
    const double f = M + fma(ser[4], s5, fma(ser[3], s4, fma(ser[2], s3, fma(ser[1], s2, ser[0] * s1))));
    double sf, cf;
    sincos_bounded(f, &sf, &cf);
    const double rr = (1.0 - c.e) * (1.0 + c.e) * rcp_fast(fma(c.e, cf, 1.0));   // r / a
    A = rr * (c.cosw * cf - c.sinw * sf);
    B = rr * (c.sinw * cf + c.cosw * sf);
  }
  const double Bc = B * c.cosi;
  const double z = c.a * sqrt_fast(fmax(fma(A, A, Bc * Bc), 0x1p-1000));
  return B > 0.0 ? z : -z;
}

// Mean anomaly of true anomaly f (|f| up to a few turns), reduced to (-π, π]: tan(E/2) = sqrt((1-e)/(1+e)) tan(f/2),
// M = E - e sin E.  rm = sqrt(1-e), rp = sqrt(1+e).  Lean primitives (pt_math.cuh): this runs once per tile.
__device__ __forceinline__ double mean_anomaly_of_true(double f, double e, double rm, double rp) {
  double sh, ch;
  sincos_bounded(0.5 * f, &sh, &ch);
  const double y = rm * sh, x = rp * ch;
  const double E = 2.0 * copysign(atan2_pos(fabs(y), x), y);
  double sE, cE;
  sincos_bounded(E, &sE, &cE);
  return fma(-e, sE, E);
}

// asin(x) for 0 <= x < 1.
__device__ __forceinline__ double asin_unit(double x) {
  return atan2_pos(x, sqrt_fast(fmax((1.0 - x) * (1.0 + x), 0x1p-1000)));
}

// Validate a parameter row and fill the orbit part of PvConst (khat is set by the caller beforehand).
// `row` = [t0, P, a/R*, i, e, w, ...]; half_exp_phase = half the exposure in cycles (0 when n_ss == 1).
__device__ __forceinline__ void pv_setup_orbit(PvConst& c, const double* row, bool row_ok, int n_ss, double t_exp) {
  const double t0 = __ldg(row), P = __ldg(row + 1), a = __ldg(row + 2), inc = __ldg(row + 3), e = __ldg(row + 4);
  double w = __ldg(row + 5);
  int flags = 0;
  if (!row_ok || !(isfinite(t0) && isfinite(P) && isfinite(a) && isfinite(inc) && isfinite(e) && isfinite(w)) ||
      !(P > 0.0) || !(a > 0.0) || !(e >= 0.0 && e < 1.0)) {
    c.flags = PV_BAD;
    return;
  }
  c.t0 = t0; c.P = P; c.invP = __drcp_rn(P); c.a = a; c.e = e;
  if ((__double_as_longlong(P) & 0x000fffffffffffffLL) == 0x000fffffffffffffLL) flags |= PV_SLOWDIV;
  // cos i, sin i: the lean kernel for ordinary inclinations, the library for anything else
  double sini;
  if (fabs(inc) <= 1.0e3) sincos_bounded(inc, &sini, &c.cosi);
  else sincos(inc, &sini, &c.cosi);
  const double k = c.khat;
  const double margin = 1.0e-7;   // cycles; the cheap fold differs from the pinned one by < 2.3e-16 |x| <= 2.3e-8
  double lo, hi;
  if (e == 0.0) {
    flags |= PV_CIRCULAR;
    c.sinw = 0.0; c.cosw = 1.0; c.rt1me2 = 1.0; c.Mtr = 0.0; c.sin_e = 0.0; c.cos_e = 1.0;
    // overlap needs a²(cos²i + sin²i sin²φ) < (1+k)² and cos φ > 0
    const double ci2 = c.cosi * c.cosi;
    const double si2 = 1.0 - ci2;
    const double r = (1.0 + k) / a;
    const double S = (r * r - ci2) / si2 + 1.0e-12;   // sin²φ below this value; si2 == 0 gives ±inf/NaN (handled)
    if (S <= 0.0) { flags |= PV_NEVER; hi = 0.0; }
    else if (!(S < 1.0)) hi = 0.25;
    else hi = fmin(0.25, atan2_pos(sqrt_fast(S), sqrt_fast(1.0 - S)) * kC[C_HALF_INVPI]);   // asin(sqrt S) / 2π
    hi = hi * (1.0 + 1.0e-9) + margin;
    lo = -hi;
  } else {
    if (fabs(w) <= 1.0e3) {
      sincos_bounded(w, &c.sinw, &c.cosw);
    } else {
      sincos(w, &c.sinw, &c.cosw);
      w = atan2(c.sinw, c.cosw);              // same angle, small enough for the lean kernels below
    }
    sincos_bounded(e, &c.sin_e, &c.cos_e);
    const double rm = sqrt_fast(1.0 - e), rp = sqrt_fast(1.0 + e);
    c.rt1me2 = rm * rp;
    const double ftr = 0.5 * kPi - w;
    c.Mtr = mean_anomaly_of_true(ftr, e, rm, rp);
    // overlap needs r |cos(w+f)| < 1+k and sin(w+f) > 0.  First bound with r >= a(1-e), then tighten with the smallest
    // r on the resulting true-anomaly range (any in-transit f lies in the first range, so the second is still safe).
    const double one_k = 1.0 + k;
    double C = one_k / (a * (1.0 - e));
    if (!(C < 1.0)) {
      flags |= PV_ALWAYS; lo = -1.0; hi = 1.0;
    } else {
      double D = asin_unit(C);
      // max of cos f over [ftr-D, ftr+D]
      const double fc = ftr - kTwoPi * rint(ftr * (1.0 / kTwoPi));   // reduce to [-π, π]
      double s1, c1, s2, c2;
      sincos_bounded(fc - D, &s1, &c1);
      sincos_bounded(fc + D, &s2, &c2);
      const double cmax = (fabs(fc) <= D) ? 1.0 : fmax(c1, c2);
      const double rmin = a * (1.0 - e) * (1.0 + e) / fma(e, cmax, 1.0);
      C = fmin(C, one_k / rmin);
      D = asin_unit(C) * (1.0 + 1.0e-9) + 1.0e-9;
      double dhi = mean_anomaly_of_true(ftr + D, e, rm, rp) - c.Mtr;
      double dlo = c.Mtr - mean_anomaly_of_true(ftr - D, e, rm, rp);
      dhi -= kTwoPi * floor(dhi * (1.0 / kTwoPi));   // both differences are in [0, 2π)
      dlo -= kTwoPi * floor(dlo * (1.0 / kTwoPi));
      hi = dhi * (1.0 / kTwoPi) * (1.0 + 1.0e-9) + margin;
      lo = -(dlo * (1.0 / kTwoPi) * (1.0 + 1.0e-9) + margin);
      if (!(hi < 0.45 && lo > -0.45)) { flags |= PV_ALWAYS; lo = -1.0; hi = 1.0; }   // folded phase must not wrap
    }
  }
  if (!(k > 1.0e-150)) { flags |= PV_NEVER; }
  c.ph_lo = lo; c.ph_hi = hi;
  const double hx = (n_ss > 1) ? fabs(0.5 * t_exp * c.invP) * (1.0 + 1.0e-9) : 0.0;
  c.ex_lo = lo - hx; c.ex_hi = hi + hx;
  if (!(c.ex_hi < 0.49 && c.ex_lo > -0.49)) { flags |= PV_ALWAYS; }   // also catches a non-finite exposure width
  c.win_mid = 0.5 * (c.ex_lo + c.ex_hi);
  c.win_half = 0.5 * (c.ex_hi - c.ex_lo);
  if (flags & PV_ALWAYS) { c.win_mid = 0.0; c.win_half = CUDART_INF; }
  if (flags & PV_NEVER) { c.win_mid = 0.0; c.win_half = -CUDART_INF; }
  c.flags = flags;
}

}  // namespace pt
