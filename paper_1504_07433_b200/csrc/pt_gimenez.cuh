// pt_gimenez.cuh — the Giménez transit model (Eq. 1-12) with precomputed coefficient tables
// and its interpolation in z.
//
//   f = 1 - Σ_{n=0}^{N} C_n α_n(b,c),  b = k/(1+k), c = z/(1+k)                                                     Eq. 1, 2, 9
//   α_n = b² (1-c²)^{ν+1} Σ_{j=0}^{N_J} A_{n,j} G_j(ν+2, ν+1; 1-b)² G_j(ν+2, 1; c²),  ν = (n+2)/2                   Eq. 3, 10, 11
// G_j(p,q;x) are Kopal's Jacobi polynomials 2F1(-j, j+p; q; x) (R20).  Here they are the standard Jacobi
// polynomials they are multiples of, run up by the three-term recurrence the paper describes (Eq. 12):
//   G_j(ν+2, ν+1; x) = j! Γ(ν+1)/Γ(j+ν+1) P_j^{(ν,1)}(1-2x),      G_j(ν+2, 1; x) = P_j^{(0,ν+1)}(1-2x),
//   P_{j+1} = ((r1 + r2 y) P_j - r3 P_{j-1}),  r = (a2, a3, a4)/a1 of the classical recurrence, P_{-1} = 0, P_0 = 1.
// The coefficient table the paper asks for ("A_{n,j} and j_n can be precomputed into two-dimensional lookup tables") holds
// per (n, j): B_{n,j} = A_{n,j} (j! Γ(ν+1)/Γ(j+ν+1))² — the normalisation of the first polynomial folded into A — and the two
// triples r of the two polynomial sequences.  It is built on the device once (gimenez_coef_kernel) into memory the caller
// owns.  None of this is shared with the oracle, which evaluates the polynomials by an explicit finite sum in __float128.
#pragma once
#include <cuda_runtime.h>

#include "pt_flux.cuh"

namespace pt {

constexpr int kGimCoef = 8;          // doubles per (n, j): B, r1[3], r2[3], spare
constexpr int kGimMaxLdc = 8;        // limb-darkening coefficients per passband
constexpr int kGimMaxNj = 256;
constexpr int kGimMaxPb = 64;

__global__ void gimenez_coef_kernel(int n_ldc, int n_j, double* __restrict__ coef) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (n_ldc + 1) * (n_j + 1)) return;
  const int n = idx / (n_j + 1), j = idx - n * (n_j + 1);
  const double nu = 0.5 * (double)(n + 2);
  double* c = coef + (size_t)idx * kGimCoef;
  // B = (-1)^j (2j+ν+2) Γ(ν+1) j! / (ν (j+1) Γ(j+ν+1))
  const double lg = lgamma(nu + 1.0) + lgamma((double)j + 1.0) - lgamma((double)j + nu + 1.0);
  const double B = (2.0 * j + nu + 2.0) / (nu * (double)(j + 1)) * exp(lg);
  c[0] = (j & 1) ? -B : B;
  for (int q = 0; q < 2; ++q) {
    const double al = q == 0 ? nu : 0.0, be = q == 0 ? 1.0 : nu + 1.0;
    const double s = 2.0 * j + al + be;
    const double a1 = 2.0 * (j + 1.0) * (j + al + be + 1.0) * s;
    const double a2 = (s + 1.0) * (al * al - be * be);
    const double a3 = s * (s + 1.0) * (s + 2.0);
    const double a4 = 2.0 * (j + al) * (j + be) * (s + 2.0);
    c[1 + 3 * q] = a2 / a1; c[2 + 3 * q] = a3 / a1; c[3 + 3 * q] = a4 / a1;
  }
  c[7] = 0.0;
}

// α_0 .. α_N at (k, z), 0 <= z < 1 + k, k > 0.
__device__ __forceinline__ void gimenez_alphas(const double* __restrict__ coef, int n_ldc, int n_j, double k, double z, double* an) {
  const double r1k = rcp_fast(1.0 + k);
  const double b = k * r1k, c = z * r1k;
  const double y1 = 2.0 * b - 1.0;                 // 1 - 2(1-b)
  const double c2 = c * c;
  const double y2 = 1.0 - 2.0 * c2;
  const double w = (1.0 - c) * (1.0 + c);          // 1 - c²
  const double sw = sqrt(w);
  double pw = w * w;                               // w^{ν+1} = sqrt(w)^{n+4}
  for (int n = 0; n <= n_ldc; ++n) {
    const double* cf = coef + (size_t)n * (n_j + 1) * kGimCoef;
    double p1m = 0.0, p1 = 1.0, p2m = 0.0, p2 = 1.0, s = 0.0;
    for (int j = 0; j <= n_j; ++j) {
      const double2* cj = (const double2*)(cf + (size_t)j * kGimCoef);     // the same address in every lane: a broadcast
      const double2 qa = cj[0], qb = cj[1], qc = cj[2], qd = cj[3];          // read-only: global (L1) or shared memory
      s = fma(qa.x * p1 * p1, p2, s);                                         // B P1² P2
      const double n1 = fma(fma(qb.x, y1, qa.y), p1, -qb.y * p1m);            // r1 = (qa.y, qb.x, qb.y)
      const double n2 = fma(fma(qc.y, y2, qc.x), p2, -qd.x * p2m);            // r2 = (qc.x, qc.y, qd.x)
      p1m = p1; p1 = n1; p2m = p2; p2 = n2;
    }
    an[n] = b * b * pw * s;
    pw *= sw;
  }
}

struct GimArgs {
  const double* coef;
  int n_ldc, n_j;
  const double* times;
  int64_t n_t, t_stride_pv;
  const double* params;
  int64_t n_pv;
  int n_pb, n_ss;
  double t_exp;
  double* flux;
  int32_t* status;
  // interpolation in z: per parameter vector (n_ldc+1) x (n_in + n_out) nodes in `work`
  double* work;
  int n_in, n_out;
};

// Row [t0, P, a/R*, i, e, w, k, u_1..u_N per passband] -> orbit constants, k, C_{n,q} (Eq. 7, 8) in shared memory.
__device__ __forceinline__ void gimenez_setup(const GimArgs& A, const double* row, PvConst& c, double* C) {
  bool ok = true;
  for (int i = 0; i < 7 + A.n_pb * A.n_ldc; ++i) ok &= isfinite(row[i]);
  const double k = row[6];
  if (!(k >= 0.0)) ok = false;
  for (int q = 0; q < A.n_pb && ok; ++q) {
    double su = 0.0, den = 1.0;
    for (int n = 1; n <= A.n_ldc; ++n) { const double u = row[7 + q * A.n_ldc + n - 1]; su += u; den -= (double)n * u / (double)(n + 2); }
    if (den == 0.0) { ok = false; break; }
    C[q * (A.n_ldc + 1)] = (1.0 - su) / den;
    for (int n = 1; n <= A.n_ldc; ++n) C[q * (A.n_ldc + 1) + n] = row[7 + q * A.n_ldc + n - 1] / den;
  }
  c.khat = ok ? k : 0.0;
  pv_setup_orbit(c, row, ok, A.n_ss, A.t_exp);
}

// MODE 0: every in-transit subsample through the series.  MODE 1: linear interpolation in the per-vector z-tables of `work`.
template <int MODE>
__global__ void __launch_bounds__(256) gimenez_kernel(const __grid_constant__ GimArgs A, int blocks_per_pv, int coef_in_smem) {
  extern __shared__ double2 s_coef2[];                  // the coefficient table, when it fits (MODE 0)
  __shared__ PvConst c;
  __shared__ double C[kGimMaxPb * (kGimMaxLdc + 1)];
  const double* coef = A.coef;
  if (MODE == 0 && coef_in_smem) {
    const int n2 = (A.n_ldc + 1) * (A.n_j + 1) * kGimCoef / 2;
    for (int i = threadIdx.x; i < n2; i += blockDim.x) s_coef2[i] = __ldg((const double2*)A.coef + i);
    coef = reinterpret_cast<const double*>(s_coef2);
  }
  const int64_t pv = blockIdx.x / blocks_per_pv;
  const int chunk = (int)(blockIdx.x % blocks_per_pv);
  const int64_t rowlen = 7 + (int64_t)A.n_pb * A.n_ldc;
  const double* row = A.params + pv * rowlen;
  if (threadIdx.x == 0) {
    gimenez_setup(A, row, c, C);
    if ((c.flags & PV_BAD) && chunk == 0 && A.status) { atomicOr(&A.status[0], PT_ST_BAD_PARAM); atomicAdd(&A.status[1], 1); }
  }
  __syncthreads();
  const double* tt = A.times + pv * A.t_stride_pv;
  double* fo = A.flux + pv * A.n_pb * A.n_t;
  const bool bad = c.flags & PV_BAD;
  const double k = c.khat;
  const int nt = A.n_in + A.n_out;
  const double* tab = MODE == 1 ? A.work + (size_t)pv * (A.n_ldc + 1) * nt : nullptr;
  const bool use_tab = MODE == 1 && k < 1.0 && k > 1.0e-150;
  const double zi_scale = use_tab ? (double)(A.n_in - 1) / (1.0 - k) : 0.0;      // nodes per unit z, inner / outer grid
  const double zo_scale = use_tab ? (double)(A.n_out - 1) / (2.0 * k) : 0.0;
  for (int64_t e = (int64_t)chunk * blockDim.x + threadIdx.x; e < A.n_t; e += (int64_t)blocks_per_pv * blockDim.x) {
    if (bad) { for (int q = 0; q < A.n_pb; ++q) fo[(int64_t)q * A.n_t + e] = nan64(); continue; }
    double acc[kGimMaxLdc + 1];
#pragma unroll
    for (int n = 0; n <= kGimMaxLdc; ++n) acc[n] = 0.0;
    const double t = __ldg(tt + e);
    bool any = false;
    if (in_window(t, c.t0, c.invP, c.win_mid, c.win_half)) {
      for (int s = 0; s < A.n_ss; ++s) {
        const double ts = (A.n_ss > 1) ? __dadd_rn(t, subsample_offset(s, A.n_ss, A.t_exp)) : t;
        const double zs = orbit_z_signed(c, fold_phase(ts, c.t0, c.P, c.invP, c.flags & PV_SLOWDIV));
        if (zs >= 0.0 && zs < 1.0 + k && k > 1.0e-150) {
          any = true;
          double an[kGimMaxLdc + 1];
          if (use_tab) {
            // the segment that holds z, its cell and the weight; the last cell is closed at its upper end
            const bool inner = zs < 1.0 - k;
            const double r = inner ? zs * zi_scale : (zs - (1.0 - k)) * zo_scale;
            const int nn = inner ? A.n_in : A.n_out;
            int i0 = (int)r;
            i0 = min(max(i0, 0), nn - 2);
            const double f = r - (double)i0;
            const double* tn = tab + (inner ? 0 : A.n_in) + i0;
            for (int n = 0; n <= A.n_ldc; ++n) {
              const double v0 = __ldg(tn + (size_t)n * nt), v1 = __ldg(tn + (size_t)n * nt + 1);
              an[n] = fma(f, v1 - v0, v0);
            }
          } else {
            gimenez_alphas(coef, A.n_ldc, A.n_j, k, zs, an);
          }
          for (int n = 0; n <= A.n_ldc; ++n) acc[n] += an[n];
        }
      }
    }
    const double inv = 1.0 / (double)A.n_ss;
    for (int q = 0; q < A.n_pb; ++q) {
      double al = 0.0;
      if (any) for (int n = 0; n <= A.n_ldc; ++n) al = fma(C[q * (A.n_ldc + 1) + n], acc[n], al);
      fo[(int64_t)q * A.n_t + e] = any ? 1.0 - al * inv : 1.0;
    }
  }
}

// Tables of the interpolated mode: node i of the inner grid at z = i (1-k)/(n_in-1), node i of the outer grid at
// z = (1-k) + i 2k/(n_out-1); the last outer node (z = 1+k) is 0.
__global__ void __launch_bounds__(256) gimenez_table_kernel(const __grid_constant__ GimArgs A) {
  const int nt = A.n_in + A.n_out;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= A.n_pv * nt) return;
  const int64_t pv = idx / nt;
  const int i = (int)(idx - pv * nt);
  const double k = __ldg(A.params + pv * (7 + (int64_t)A.n_pb * A.n_ldc) + 6);
  double an[kGimMaxLdc + 1];
  for (int n = 0; n <= A.n_ldc; ++n) an[n] = 0.0;
  if (k > 1.0e-150 && k < 1.0) {
    const double z = i < A.n_in ? (double)i * ((1.0 - k) / (double)(A.n_in - 1))
                                : (1.0 - k) + (double)(i - A.n_in) * ((2.0 * k) / (double)(A.n_out - 1));
    if (z < 1.0 + k && i != nt - 1) gimenez_alphas(A.coef, A.n_ldc, A.n_j, k, z, an);
  }
  for (int n = 0; n <= A.n_ldc; ++n) A.work[((size_t)pv * (A.n_ldc + 1) + n) * nt + i] = an[n];
}

}  // namespace pt
