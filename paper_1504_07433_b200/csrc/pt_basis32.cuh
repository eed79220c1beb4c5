// pt_basis32.cuh — the fp32-arithmetic variant of the orbit stage and the basis functions (BASELINE.json: "fp32 variant:
// 2e-6 absolute").  Everything up to the folded phase stays fp64 (pt_orbit.cuh: a time of ~1e3 d has a
// resolution of 1e-4 d in fp32); from the phase on — orbit, case split, λe, λd*, ηd, limb-darkening combine — the
// arithmetic is fp32 on the FP32 pipe (twice the FP64 rate on B200, and single-instruction MUFU reciprocals and roots).
// The same formulation as pt_basis.cuh (cancellation-free contact distances, atan2 for the κ's, two Bulirsch `cel`
// sequences on one AGM ladder).  λd* is a difference of O(1) elliptic-integral terms that cancels down to O(k²): its
// absolute error in fp32 is ~1e-7 x the size of those terms whatever k is, which near the inner contact of a small planet
// exceeds the gate; the kernel therefore returns an error bound with the value, and a caller that needs it re-evaluates
// that sample in fp64 (pt_basis.cuh).
#pragma once
#include <cuda_runtime.h>

#include "pt_basis.cuh"
#include "pt_orbit.cuh"

namespace pt {

#ifndef PT_F32_NTHR
#define PT_F32_NTHR 1.2f   // |n| below which cK K + cP Π is evaluated as (cK+cP) K + cP (Π-K): in fp32 the rewrite pays up to
                           // |n| ~ 1.2 (worst λd* error over k: 9.0e-7 with 0.5 as in fp64, 7.8e-7 with 1.2, 8.0e-7 with 1.5, 8.6e-7 with 2)
#endif

struct Basis32 {
  float le, ld, ed;
  float ld_err;            // bound on the absolute error of ld
};

__device__ __forceinline__ float rcp32(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt32(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt32(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// sin and cos for |x| <= ~8 (one Cody–Waite step by π/2 with a three-part constant, minimax-like Taylor kernels on |r| <= π/4).
__device__ __forceinline__ void sincos32(float x, float* sn, float* cs) {
  const float kf = rintf(x * 0.636619772f);
  const int k = (int)kf;
  float r = fmaf(-kf, 1.57079625f, x);          // π/2 hi
  r = fmaf(-kf, 7.54978942e-8f, r);             // π/2 mid
  r = fmaf(-kf, 5.39030253e-15f, r);            // π/2 lo
  const float r2 = r * r;
  float ps = fmaf(r2, 2.75573192e-6f, -1.98412698e-4f);
  ps = fmaf(ps, r2, 8.33333333e-3f);
  ps = fmaf(ps, r2, -1.66666667e-1f);
  const float s = fmaf(ps * r2, r, r);
  float pc = fmaf(r2, 2.48015873e-5f, -1.38888889e-3f);
  pc = fmaf(pc, r2, 4.16666667e-2f);
  pc = fmaf(pc, r2, -0.5f);
  const float c = fmaf(pc, r2, 1.0f);
  const float ss = (k & 1) ? c : s, cc = (k & 1) ? s : c;
  *sn = (k & 2) ? -ss : ss;
  *cs = ((k + 1) & 2) ? -cc : cc;
}

// atan2(y, x) for y >= 0: the angle in [0, π] (pt_math.cuh: atan2_pos, in fp32: odd polynomial on |t| <= tan(π/8)).
__device__ __forceinline__ float atan2_pos32(float y, float x) {
  const float ax = fabsf(x);
  const bool swap = y > ax;
  const float mn = swap ? ax : y, mx = swap ? y : ax;
  const bool big = mn > 0.414213562f * mx;
  const float num = big ? mn - mx : mn;
  const float den = big ? mn + mx : mx;
  const float t = num * rcp32(den);
  const float u = t * t;
  float p = fmaf(u, -0.0666666667f, 0.0769230769f);              // atan t = t + t u P(u): series through t^15 (next term < 4e-8 t)
  p = fmaf(p, u, -0.0909090909f);
  p = fmaf(p, u, 0.111111111f);
  p = fmaf(p, u, -0.142857143f);
  p = fmaf(p, u, 0.2f);
  p = fmaf(p, u, -0.333333333f);
  float a = fmaf(t * u, p, t);
  a = big ? a + 0.785398163f : a;
  a = swap ? 1.57079633f - a : a;
  return x < 0.0f ? 3.14159265f - a : a;
}

// cK·K(m) + cE·E(m) + cP·cel(kc, 1-n, a2, b2·sp) in fp32 (pt_basis.cuh: cel_pair); *mag receives the sum of the magnitudes of
// the two sequences' results, for the error bound of the caller.
__device__ __forceinline__ float cel_pair32(float mc, float sp, float cK, float cE, float cP, float a2, float b2, float* mag) {
  float qc = sqrt32(mc);
  float a1 = cK + cE;
  float b1 = fmaf(cE, mc, cK);
  float p2 = sp;
  float e = qc, em = 1.0f;
#pragma unroll 1
  for (int it = 0; it < 12; ++it) {
    const float rr = rcp32(em * p2);
    const float rem = rr * p2;
    const float rp2 = rr * em;
    float f = a1;
    a1 = fmaf(b1, rem, a1);
    b1 = fmaf(f, qc, b1);
    b1 += b1;
    f = a2;
    a2 = fmaf(b2, rp2, a2);
    const float g2 = e * rp2;
    b2 = fmaf(f, g2, b2);
    b2 += b2;
    p2 += g2;
    const float g = em;
    em += qc;
    if (fabsf(g - qc) <= 2.0e-4f * g) break;     // the next step squares it: below fp32 resolution
    qc = 2.0f * sqrt32(e);
    e = qc * em;
  }
  const float d1 = 2.0f * em * em, d2 = em * (em + p2);
  const float rr = rcp32(d1 * d2);
  const float s1 = fmaf(a1, em, b1) * (d2 * rr);
  const float s2 = fmaf(a2, em, b2) * (d1 * rr);
  *mag = 1.57079633f * (fabsf(s1) + fabsf(cP * s2));
  return 1.57079633f * fmaf(cP, s2, s1);
}

// Basis functions at radius ratio p > 0 and separation z >= 0 in fp32 (pt_basis.cuh: ma_basis, same case analysis).
__device__ __forceinline__ Basis32 ma_basis32(float p, float z) {
  Basis32 r;
  r.ld_err = 0.0f;
  z = fmaxf(z, 1.0e-30f);
  const float d = z - p, s = z + p;
  const float pm1 = p - 1.0f;
  const bool pmid = (p >= 0.5f) & (p <= 2.0f);
  const float sm1 = pmid ? z + pm1 : (p < 0.5f ? (z - 1.0f) + p : s - 1.0f);
  const float opd = pmid ? z - pm1 : 1.0f + d;
  const float omd = (p < 1.0f) ? (1.0f - z) + p : 1.0f - d;
  const float sp1 = s + 1.0f;
  if (omd <= 0.0f) { r.le = 0.0f; r.ld = 0.0f; r.ed = 0.0f; return r; }
  if (opd <= 0.0f) { r.le = 1.0f; r.ld = 0.666666667f; r.ed = 0.5f; return r; }
  const float p2 = p * p, z2 = z * z;
  const float eta2 = 0.5f * p2 * fmaf(2.0f, z2, p2);
  const float oma = omd * opd;
  const bool partial = sm1 > 0.0f;
  if (partial) {
    const float T = sqrt32(oma * sm1 * sp1);
    const float pp1 = pm1 * (p + 1.0f);
    const float kap0 = atan2_pos32(T, z2 + pp1);
    const float kap1 = atan2_pos32(T, z2 - pp1);
    r.le = (fmaf(p2, kap0, kap1) - 0.5f * T) * 0.318309886f;
    r.ed = (fmaf(2.0f * eta2, kap0, kap1) - 0.25f * (1.0f + 5.0f * p2 + z2) * T) * 0.159154943f;
  } else {
    r.le = p2;
    r.ed = eta2;
  }
  if (sm1 == 0.0f) {   // inner contact in fp32: the elementary closed form
    r.ld = 0.212206591f * acosf(1.0f - 2.0f * p) - 0.141471061f * (3.0f + 2.0f * p - 8.0f * p2) * sqrtf(p * (1.0f - p));
    r.ld_err = 4.0e-7f;
    return r;
  }
  float mc, sp, cK, cE, cP, pref, add;
  float a2 = 1.0f, b2;
  if (d == 0.0f) {
    add = 0.333333333f; cP = 0.0f; sp = 1.0f; b2 = 1.0f;
    if (!partial) {
      mc = (1.0f - 2.0f * p) * (1.0f + 2.0f * p);
      cE = 4.0f * (2.0f * p2 - 1.0f);
      cK = mc;
      pref = 0.0707355303f;
    } else {
      const float i4p2 = rcp32(4.0f * p2);
      mc = (2.0f * p - 1.0f) * (2.0f * p + 1.0f) * i4p2;
      cE = 16.0f * p * (2.0f * p2 - 1.0f);
      cK = -(1.0f - 4.0f * p2) * (3.0f - 8.0f * p2) * rcp32(p);
      pref = 0.0353677651f;
    }
  } else {
    const float rd = rcp32(d);
    const float ad = fabsf(d);
    const float q = -d * s;
    const float w7 = z2 + 7.0f * p2 - 4.0f;
    add = d < 0.0f ? 0.666666667f : 0.0f;
    cP = 3.0f * s * rd;
    if (partial) {
      const float a = d * d, b = s * s;
      const float pz = p * z;
      const float rpz = rsqrt32(pz);
      mc = 0.25f * sm1 * sp1 * (rpz * rpz);
      sp = fabsf(rd);
      b2 = ad;
      cE = 4.0f * pz * w7;
      pref = 0.0353677651f * rpz;
      const float bm1 = sm1 * sp1;
      if (oma < PT_F32_NTHR * a) {
        cK = fmaf(-bm1, 2.0f * b + a - 3.0f, -3.0f * q * fmaf(a, bm1, oma) * (rd * rd));
        a2 = 0.0f;
        b2 = -oma * (rd * rd) * ad;
      } else {
        cK = fmaf(-bm1, 2.0f * b + a - 3.0f, -3.0f * q * (b - 2.0f));
      }
    } else {
      const float roma = rsqrt32(oma);
      const float rs = rcp32(s);
      mc = -sm1 * sp1 * (roma * roma);
      sp = s * fabsf(rd);
      b2 = ad * rs;
      cE = oma * w7;
      pref = 0.0707355303f * roma;
      const float pz4 = 4.0f * p * z;
      if (pz4 < PT_F32_NTHR * d * d) {
        cK = oma * fmaf(-3.0f * q, rd * rd, -sm1 * sp1);
        a2 = 0.0f;
        b2 = -pz4 * (rd * rd) * (ad * rs);
      } else {
        cK = 1.0f - 5.0f * z2 + p2 + q * q;
      }
    }
  }
  float mag;
  const float v = cel_pair32(mc, sp, cK, cE, cP, a2, b2, &mag);
  r.ld = fmaxf(fmaf(pref, v, add), 0.0f);
  r.ld_err = fabsf(pref) * mag;       // x a few fp32 ulps: the caller scales it
  return r;
}

// fp32 copies of the constants of one parameter vector that the fp32 path reads (filled by tile_setup, pt_flux.cuh).
struct PvF32 {
  float a, cosi, ci2, e, sinw, cosw, rt1me2, sin_e, cos_e, khat;
  float coef[3];
  int use;                 // 1: this parameter vector is evaluated in fp32 (else fp64 arithmetic, fp32 storage)
};
static_assert(sizeof(PvF32) % 8 == 0, "records are copied as doubles");

// Worst absolute errors of ma_basis32 against the fp64 functions, measured over k in [0.005, 0.7] and z in [0, 1+k] with
// 4e5 points per k, a quarter of them within 1e-7 ... 1e-2 of the inner contact (profiles/r2_fp32_variant.md): λe 9e-8,
// λd* 7.8e-7 (k ~ 0.17 within 1e-4 of the inner contact; 2-3e-7 over the bulk), ηd 8e-8.  A parameter vector whose
// limb-darkening coefficients would carry them beyond 1.75e-6 in flux (gate: 2e-6), or with k > 0.7, keeps fp64
// arithmetic: the decision is uniform per parameter vector, so no warp diverges over it (NaN parameters compare false).
// Large a/R* or e amplify the fp32 rounding of the orbit beyond the gate as well.  One function, so that every kernel
// takes the same decision for a row: from the raw parameters (k, u1, u2, a/R*, e) of a single-passband row.
__device__ __forceinline__ bool f32_ok(double k, double u1, double u2, double a, double e) {
  const double cj = u1 + 2.0 * u2;
  const double gN = 1.0 / (1.0 - u1 / 3.0 - u2 / 6.0);
  const double c0 = gN * (1.0 - cj), c1 = gN * cj, c2 = gN * u2;
  return k <= 0.7 && a <= 50.0 && e <= 0.85 && (fabs(c0) * 9.0e-8 + fabs(c1) * 8.0e-7 + fabs(c2) * 8.0e-8) <= 1.75e-6;
}

// Eccentric anomaly from mean anomaly M in (-π, π] in fp32: the starter of pt_orbit.cuh, Newton steps with a full (cheap)
// fp32 sincos, and a first-order update of (sin E, cos E) for the last step (|dE| < 3e-4: the neglected term is < 5e-8).
__device__ __forceinline__ void kepler_newton32(float M, float e, float sin_e, float cos_e, float* sinE, float* cosE) {
  float E, sE, cE;
  if (e <= 0.8f) {
    float sM, cM;
    sincos32(M, &sM, &cM);
    const float sMe = fmaf(sM, cos_e, cM * sin_e);
    E = fmaf(e * sM, rcp32(1.0f - sMe + sM), M);
  } else {
    E = M + copysignf(e, M);
  }
  sincos32(E, &sE, &cE);
#pragma unroll 1
  for (int it = 0; it < 24; ++it) {
    const float f = E - fmaf(e, sE, M);
    const float dE = f * rcp32(fmaf(-e, cE, 1.0f));
    E -= dE;
    if (fabsf(dE) < 3.0e-4f) {
      const float ns = fmaf(-cE, dE, sE);
      cE = fmaf(sE, dE, cE);
      sE = ns;
      break;
    }
    sincos32(E, &sE, &cE);
  }
  *sinE = sE; *cosE = cE;
}

// Signed projected separation in fp32 from the pinned fp64 folded phase (cycles) — pt_orbit.cuh: orbit_z_signed.
// M_tr is added in fp64 (one DFMA) so that the mean anomaly is rounded to fp32 once.
__device__ __forceinline__ float orbit_z_signed32(const PvF32& c, double Mtr, bool circular, double ph) {
  if (circular) {
    const float phf = (float)ph;
    if (fabsf(phf) <= 0.125f) {
      const float r = 6.28318531f * phf, r2 = r * r;
      float ps = fmaf(r2, 2.75573192e-6f, -1.98412698e-4f);
      ps = fmaf(ps, r2, 8.33333333e-3f);
      ps = fmaf(ps, r2, -1.66666667e-1f);
      const float sn = fmaf(ps * r2, r, r);
      return c.a * sqrt32(fmaxf(fmaf(1.0f - c.ci2, sn * sn, c.ci2), 1.0e-30f));
    }
    float sn, cs;
    sincos32(6.28318531f * phf, &sn, &cs);
    const float cc = c.cosi * cs;
    const float z = c.a * sqrt32(fmaxf(fmaf(sn, sn, cc * cc), 1.0e-30f));
    return cs > 0.0f ? z : -z;
  }
  double Md = fma(kC[C_TWOPI], ph, Mtr);
  if (Md > kC[C_PI]) Md -= kC[C_TWOPI];
  if (Md <= -kC[C_PI]) Md += kC[C_TWOPI];
  float sE, cE;
  kepler_newton32((float)Md, c.e, c.sin_e, c.cos_e, &sE, &cE);
  const float x = cE - c.e, y = c.rt1me2 * sE;
  const float Aa = c.cosw * x - c.sinw * y;
  const float Bb = c.sinw * x + c.cosw * y;
  const float Bc = Bb * c.cosi;
  const float z = c.a * sqrt32(fmaxf(fmaf(Aa, Aa, Bc * Bc), 1.0e-30f));
  return Bb > 0.0f ? z : -z;
}

// Combined decrement coef0 λe + coef1 λd* + coef2 ηd of an in-transit sample in fp32.
__device__ __forceinline__ float ma_dec32(const PvF32& c, float z) {
  const Basis32 b = ma_basis32(c.khat, z);
  return fmaf(c.coef[2], b.ed, fmaf(c.coef[1], b.ld, c.coef[0] * b.le));
}

}  // namespace pt
