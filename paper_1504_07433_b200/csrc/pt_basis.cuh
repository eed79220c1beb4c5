// pt_basis.cuh — device implementation of the three Mandel–Agol basis functions λe, λd*, ηd in fp64.
//
// Formulation: the closed forms of Mandel & Agol (2002), rearranged so that no sub-expression is formed
// by cancellation near a case boundary, with the complete elliptic integrals K, E, Π evaluated by TWO Bulirsch `cel`
// sequences that share one AGM ladder (R. Bulirsch, Numer. Math. 13 (1969) 305: cel(kc,p,a,b) is linear in (a,b), so
// cK·K + cE·E = cel(kc,1,cK+cE,cK+cE·mc) and Π(n|m) = cel(kc,1-n,1,1)).  The partial-overlap and planet-inside cases
// select *coefficients*, then run the same loop, so a warp that straddles ingress does not serialise the expensive part.
// Nothing in this file is shared with oracle/ (which uses Carlson's R_F/R_D/R_J and the textbook forms).
#pragma once
#include <cuda_runtime.h>

#include "pt_math.cuh"

#ifndef PT_CEL_UNROLL
#define PT_CEL_UNROLL 1
#endif
namespace pt {
constexpr int kCelUnroll = PT_CEL_UNROLL;   // unroll factor of the AGM ladder loop

struct Basis {
  double le, ld, ed;
};


// cK·K(m) + cE·E(m) + cP·cel(kc, 1-n, a2, b2·sp) with mc = 1-m = kc² and sp = sqrt(1-n) > 0 the square root of the second
// sequence's p-argument.  (a2, b2) = (1, 1/sp) makes the second integral Π(n|m); (0, n/sp) makes it Π(n|m) - K(m).
__device__ __forceinline__ double cel_pair(double mc, double sp, double cK, double cE, double cP, double a2, double b2) {
  double qc = sqrt_fast(mc);
  // sequence 1 (p = 1): its p-iterate equals the ladder's `em`, and e/p equals the previous qc, so it needs 1/em only
  double a1 = cK + cE;
  double b1 = fma(cE, mc, cK);
  // sequence 2: p2 = sqrt(1-n); b2 arrives already divided by p2
  double p2 = sp;
  double e = qc, em = 1.0;
#pragma unroll kCelUnroll
  for (int it = 0; it < 16; ++it) {
    const double rr = rcp_fast(em * p2);   // one reciprocal serves both sequences
    const double rem = rr * p2;
    const double rp2 = rr * em;
    // sequence 1
    double f = a1;
    a1 = fma(b1, rem, a1);
    b1 = fma(f, qc, b1);
    b1 += b1;
    // sequence 2
    f = a2;
    a2 = fma(b2, rp2, a2);
    const double g2 = e * rp2;
    b2 = fma(f, g2, b2);
    b2 += b2;
    p2 += g2;
    // ladder
    const double g = em;
    em += qc;
    if (fabs(g - qc) <= 0x1p-27 * g) break;   // 7.5e-9: the next step squares it
    qc = 2.0 * sqrt_fast(e);
    e = qc * em;
  }
  const double d1 = 2.0 * em * em, d2 = em * (em + p2);
  const double rr = rcp_fast(d1 * d2);
  const double s1 = fma(a1, em, b1) * (d2 * rr);
  const double s2 = fma(a2, em, b2) * (d1 * rr);
  return kC[C_HALFPI] * fma(cP, s2, s1);
}

// Basis functions at radius ratio p > 0 and separation z >= 0 (planet in front of the star).
__device__ __forceinline__ Basis ma_basis(double p, double z) {
  Basis r;
  z = fmax(z, 0x1p-500);   // 3e-151: keeps every operand of the fast reciprocals normal; changes nothing above it
  // d = z-p, s = z+p and the four contact distances 1-d, 1+d, s-1, s+1.  Each is formed so that the operand pair that
  // nearly cancels at "its" contact is subtracted exactly first (Sterbenz), e.g. s-1 = z + (p-1) for p in [1/2, 2]:
  // a plain (z+p)-1 loses z entirely when z << p ~ 1 (and mc = (s-1)(s+1)/(4zp) then has O(1) relative error).
  const double d = z - p, s = z + p;
  const double pm1 = p - 1.0;
  const bool pmid = (p >= 0.5) & (p <= 2.0);
  const double sm1 = pmid ? z + pm1 : (p < 0.5 ? (z - 1.0) + p : s - 1.0);   // s - 1
  const double opd = pmid ? z - pm1 : 1.0 + d;                               // 1 + d
  const double omd = (p < 1.0) ? (1.0 - z) + p : 1.0 - d;                    // 1 - d
  const double sp1 = s + 1.0;
  if (omd <= 0.0) { r.le = 0.0; r.ld = 0.0; r.ed = 0.0; return r; }                  // no overlap (z >= 1+p)
  if (opd <= 0.0) { r.le = 1.0; r.ld = kC[C_TWOTHIRDS]; r.ed = 0.5; return r; }           // star covered (z <= p-1)
  const double p2 = p * p, z2 = z * z;
  const double eta2 = 0.5 * p2 * fma(2.0, z2, p2);
  const double oma = omd * opd;                // 1 - a
  const bool partial = sm1 > 0.0;

  if (partial) {
    const double T = sqrt_fast(oma * sm1 * sp1);
    const double pp1 = pm1 * (p + 1.0);                  // p² - 1 without cancellation for p ~ 1
    const double kap0 = atan2_pos(T, z2 + pp1);
    const double kap1 = atan2_pos(T, z2 - pp1);
    r.le = (fma(p2, kap0, kap1) - 0.5 * T) * kC[C_INVPI];
    r.ed = (fma(2.0 * eta2, kap0, kap1) - 0.25 * (1.0 + 5.0 * p2 + z2) * T) * kC[C_HALF_INVPI];
  } else {
    r.le = p2;
    r.ed = eta2;
  }

  if (sm1 == 0.0) {  // inner contact z = 1-p: elementary closed form (exact equality only; table nodes land here)
    r.ld = (2.0 / 3.0 * kC[C_INVPI]) * acos(1.0 - 2.0 * p) - (4.0 / 9.0 * kC[C_INVPI]) * (3.0 + 2.0 * p - 8.0 * p2) * sqrt(p * (1.0 - p));  // rare branch: library sqrt/acos are fine here
    return r;
  }

  double mc, sp, cK, cE, cP, pref, add;
  double a2 = 1.0, b2;
  if (fabs(d) < 0x1p-332) {  // 1e-100  // z = p: the Π term drops out
    add = kC[C_THIRD];
    cP = 0.0;
    sp = 1.0;
    b2 = 1.0;
    if (!partial) {  // p < 1/2, m = 4p²
      mc = (1.0 - 2.0 * p) * (1.0 + 2.0 * p);
      cE = 4.0 * (2.0 * p2 - 1.0);
      cK = mc;
      pref = kC[C_2INV9PI];
    } else {  // p > 1/2, m = 1/(4p²)
      const double i4p2 = rcp_fast(4.0 * p2);
      mc = (2.0 * p - 1.0) * (2.0 * p + 1.0) * i4p2;
      cE = 16.0 * p * (2.0 * p2 - 1.0);
      cK = -(1.0 - 4.0 * p2) * (3.0 - 8.0 * p2) * rcp_fast(p);
      pref = kC[C_INV9PI];
    }
  } else {
    const double rd = rcp_fast(d);
    const double ad = fabs(d);
    const double q = -d * s;  // p² - z²
    const double w7 = z2 + 7.0 * p2 - 4.0;
    add = d < 0.0 ? kC[C_TWOTHIRDS] : 0.0;
    cP = 3.0 * s * rd;        // -3q/a
    if (partial) {
      const double a = d * d, b = s * s;
      const double pz = p * z;
      const double rpz = rsqrt_fast(pz);
      mc = 0.25 * sm1 * sp1 * (rpz * rpz);
      sp = fabs(rd);          // sqrt(1/a)
      b2 = ad;                // 1/sp
      cE = 4.0 * pz * w7;
      pref = kC[C_INV9PI] * rpz;
      const double bm1 = sm1 * sp1;                      // b - 1
      if (oma < 0.5 * a) {
        // |n| = (1-a)/a < 1/2: write cK·K + cP·Π = (cK+cP)·K + cP·(Π-K) with cK+cP formed without cancellation.
        // For p -> 1, z -> 0 (planet as large as the star, concentric) cK -> 3, cP -> -3, Π -> K while the prefactor
        // 1/sqrt(pz) diverges: the plain form loses ~1e-16/sqrt(z) there.
        cK = fma(-bm1, 2.0 * b + a - 3.0, -3.0 * q * fma(a, bm1, oma) * (rd * rd));
        a2 = 0.0;
        b2 = -oma * (rd * rd) * ad;                      // n/sp, n = (a-1)/a
      } else {
        cK = fma(-bm1, 2.0 * b + a - 3.0, -3.0 * q * (b - 2.0));
      }
    } else {
      const double roma = rsqrt_fast(oma);
      const double rs = rcp_fast(s);
      mc = -sm1 * sp1 * (roma * roma);
      sp = s * fabs(rd);      // sqrt(b/a)
      b2 = ad * rs;           // 1/sp
      cE = oma * w7;
      pref = kC[C_2INV9PI] * roma;
      const double pz4 = 4.0 * p * z;                    // b - a
      if (pz4 < 0.5 * d * d) {
        // |n| = (b-a)/a < 1/2: same rewrite; cK = (1-a)(1-b) + 3q, so cK + cP = (1-a)[(1-b) - 3q/a]
        cK = oma * fma(-3.0 * q, rd * rd, -sm1 * sp1);
        a2 = 0.0;
        b2 = -pz4 * (rd * rd) * (ad * rs);               // n/sp, n = (a-b)/a
      } else {
        cK = 1.0 - 5.0 * z2 + p2 + q * q;
      }
    }
  }
  // λd* is the integral of a non-negative function: close to the outer contact, where its O(1) elliptic-integral terms
  // cancel down to less than their rounding error (a few 1e-16), the sum can come out negative — clamped, so that a
  // physical limb-darkening law never yields a flux above 1
  r.ld = fmax(fma(pref, cel_pair(mc, sp, cK, cE, cP, a2, b2), add), 0.0);
  return r;
}

}  // namespace pt
