// pt_flux.cuh — the fused flux kernel: S0-S7 (and S9) of the hot path in one persistent launch.
//
// Every warp is an autonomous pipeline; the block is only a container (no block barrier once the pipelines run).  A warp
// takes tiles (parameter vector pv, run of `tile_len` exposures) from counters in the launch's scheduler slot — heaviest
// rows first when the population is small enough to rank (LPT order), else in index order or per parameter vector — and
// pushes the work through three stages, each of which runs with (nearly) all 32 lanes busy because the stages are
// decoupled by per-warp queues in shared memory:
//
//   stream   every exposure of the tile: 16-byte time loads, a 6-instruction phase-window test, flux = 1 written with
//            16-byte streaming stores for the exposures that cannot be in transit; the others go to the EXPOSURE queue
//   z-stage  G = min(n_ss,32) lanes per queued exposure: pinned subsample time + phase fold (H1, H2), orbit -> signed z
//            (Newton–Kepler for e > 0).  Subsamples with 0 <= z < 1+k̂ are compacted (ballot + popc, order kept) into
//            the ITEM queue; an exposure without any such subsample is finished here (flux = 1).  n_ss == 1: the basis
//            functions are evaluated in this round (an in-window exposure is almost always in transit)
//   basis    32 queued subsamples, possibly of different exposures, tiles and parameter vectors: λe, λd*, ηd by the closed
//            forms / one shared `cel` ladder (pt_basis.cuh) or the bilinear table lookup; the supersample sum is a
//            segmented warp-shuffle reduction over the lanes that belong to one exposure, in 64-bit fixed point so that
//            the result does not depend on how an exposure's subsamples were split over batches (integer addition is
//            associative: bit-reproducible whatever the queue history); the last subsample of an exposure applies the
//            limb-darkening combine per passband and stores.
//
// This is the "binning" BASELINE.json asks for: the expensive stage only ever sees in-transit subsamples, 32 at a time,
// and inside/partial lanes differ only in the coefficients they feed to the shared elliptic-integral loop.  Queues
// survive tile changes (items carry the index of a small per-warp ring of parameter-vector records), so small tiles —
// needed to balance a small problem over 148 SMs — do not leave ragged batches behind.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "../../include/pt.h"
#include "pt_basis.cuh"
#include "pt_orbit.cuh"
#include "pt_basis32.cuh"

namespace pt {

constexpr int kThreads = 256;
constexpr int kWarpsPerBlock = kThreads / 32;
#ifndef PT_MIN_BLOCKS
#define PT_MIN_BLOCKS 3   // resident blocks per SM the flux kernel is compiled for (register cap 65536/(256*PT_MIN_BLOCKS))
#endif
constexpr int kMaxPassbands = 1024;
#ifndef PT_UNROLL
#define PT_UNROLL 4
#endif
constexpr int kUnroll = PT_UNROLL;      // 32-exposure groups a warp streams per iteration (independent loads in flight)
constexpr int kExpQ = PT_UNROLL > 4 ? 1024 : 512;      // exposure ring: >= 32*kUnroll*2 + 32 entries, power of two, uint16 tile-local indices
constexpr int kItemQ = 64;      // item ring: at most 31 left over + 32 new per z-round
constexpr int kSlots = 64;      // pending-exposure records (supersampled path): <= 31 + 32 alive
constexpr int kPvRing = 4;      // parameter-vector records a warp keeps alive (single-passband path)
constexpr int kCoefCache = 24;  // passbands whose combine coefficients are cached per warp (multi-passband path)
constexpr int kMaxTileLen = 32768;
constexpr int kRemBias = 1 << 24;
constexpr int kSchedHead = 8;   // words of a scheduler slot in front of the per-parameter-vector tickets
constexpr unsigned long long kSlotUnsorted = 1ULL;   // flag word: the shared time axis is not ascending / not finite
// words of a scheduler slot: [0] tile / work ticket, [1] warps (blocks) that have finished, [2] flags, [3] prep blocks that
// have finished (fused likelihood in front of the epoch kernel)
enum { kW_Ticket = 0, kW_Done = 1, kW_Flags = 2, kW_PrepDone = 3 };
constexpr uint32_t kUnitChunks = 0x80000000u;        // ucnt flag: units are chunks of kChunkLen exposures, not transit epochs
constexpr int kChunkLen = 256;
// -DPT_DEBUG_CHECKS: capacity invariants of the per-warp queues are checked and a violation traps (the test suite is run
// once against such a build; compute-sanitizer is not available on the GPU pool).
#ifdef PT_DEBUG_CHECKS
#define PT_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define PT_CHECK(cond) do { } while (0)
#endif
#ifndef PT_ST
#define PT_ST __stcs   // flux stores: write-once data, evict-first
#endif
#ifndef PT_EXPAND_INLINE
#define PT_EXPAND_INLINE __forceinline__
#endif

struct PvRec;

struct FluxArgs {
  const double* times;
  int64_t n_t, t_stride_pv;
  const double* params;
  int64_t n_pv;
  int n_pb, n_ss;
  double t_exp;
  void* flux;
  int32_t* status;
  // views (exact per-passband-k mode launches the single-passband kernel once per passband of a wider row)
  int64_t row_stride;          // doubles per parameter row
  int pb_first;                // first passband of the row this launch looks at
  int64_t flux_pv_stride;      // flux elements between parameter vectors
  int64_t flux_off;            // flux element offset of this launch's first passband
  int pbk;                     // 1: every passband at its own radius ratio, basis functions per passband (n_ss == 1 kernels)
  // fused likelihood (OutT = Chi2): observed flux and 1/sigma [n_pb][n_t] shared by all parameter vectors, chi2 [n_pv]
  const double* obs;
  const double* isig;
  double* chi2;
  const double* base_part;     // partial sums of the all-out-of-transit chi2 (chi2_base_kernel), n_base_part of them
  int n_base_part;
  // tiling
  int tile_len;            // exposures per tile (multiple of 256, <= kMaxTileLen)
  int tiles_per_pv;
  int64_t n_tiles;
  unsigned long long* sched;   // scheduler slot: [0] global tile ticket, [1] warps that have finished, [2] flags (kSlotUnsorted),
                               // [kSchedHead + pv] per-pv tickets
  const PvRec* pvcache;        // single passband, few parameter vectors: records precomputed by prep_kernel (else NULL)
  const uint32_t* order;       // global mode: row order of the tiles written by prep_kernel (heaviest rows first / rows sorted
                               // by k̂ for the table), or NULL = index order
  int per_pv;                  // 1: warps stay on one parameter vector and take its tiles from its own counter (n_pv small)
  int prep;                    // 1: launched as a programmatic dependent of prep_kernel: wait for it before reading the slot
  int range;                   // 1: one shared time axis; if prep_kernel found it ascending and finite, out-of-window
                               // stretches are found by search and written as pure fills (no per-exposure window test)
  // epoch kernel (pt_epoch.cuh): units of evaluation work per parameter vector, written by prep_kernel
  const double* un0;           // [n_pv] first transit epoch on the axis (units in epoch mode)
  const uint32_t* ucnt;        // [n_pv] number of units; kUnitChunks set: the row is cut into chunks of kChunkLen exposures
  int unit_chunks;             // work units per row: unit (row, c) owns the epochs [c cnt/C, (c+1) cnt/C) and the gaps in front of them
  int f32a;                    // 1: fp32 ARITHMETIC from the folded phase on (PT_F32; float output, single passband) where
                               // the parameter vector allows it (pt_basis32.cuh: f32_ok)
  int base_added;              // fused likelihood: prep_kernel already left the baseline in chi2[]
  // supersample accumulation (fixed point)
  int fx_bits;             // 61 - ceil(log2 n_ss): a sum of n_ss values below 2^eb fits an int64 at scale 2^(fx_bits-eb)
  double fx_scale;         // 2^fx_bits (basis values are <= 1)
  double fx_inv;           // 1 / (fx_scale * n_ss)
  double inv_nss;          // 1 / n_ss
  // interpolation table (mode 1)
  const void* tb;
  int tb_dtype, n_k, n_z, n_fn;
  double k_min, dk, dz, inv_dz;
};

__device__ __forceinline__ double nan64() { return __longlong_as_double(0x7ff8000000000000LL); }

// One parameter vector as a warp sees it while a tile of it is being streamed, and for as long as queued subsamples of
// that tile are alive.
struct PvRec {
  PvConst c;               // orbit constants, k̂, phase window (pt_orbit.cuh)
  const double* tb;        // times of the tile
  int64_t e0, pv;          // first exposure of the tile in its row; parameter vector (fused likelihood)
  char* ob;                // flux of the tile: row pv, passband 0, first exposure of the tile
  double coef[3];          // single passband: g(1-c)/N, g c/N, g u2/N
  double acc_scale;        // single passband: fixed-point scale of the combined decrement, and its inverse / n_ss
  double acc_inv;
  double ik2;              // 1/k̂² (0 when k̂ == 0)
  const double* row;       // parameter row (multi-passband combine beyond the coefficient cache)
  double w_c0, w_half;     // cheap window test: x' = t*invP + w_c0, |x' - rint(x')| < w_half + 2^-50 |x'|
  double fk;               // table: fractional k index
  int ik;                  // table: lower k index
  int use_table;
  PvF32 f;                 // fp32 copies for the fp32-arithmetic variant (f.use)
};

struct Slot {              // a supersampled exposure with subsamples still in the item queue
  long long acc[3];        // fixed-point sums (single passband: acc[0] = combined decrement)
  int remaining;           // subsamples not yet evaluated (+ kRemBias while the exposure is still being expanded)
  uint16_t e;              // tile-local exposure index
  uint16_t ring;           // PvRec index
};

// Range mode (ascending shared time axis): the transit epochs of the current tile that are still to be looked at, and the
// current batch of up to 32 of them — exposures [lo[i], hi[i]) of the tile can be in transit at epoch i of the batch.
struct RangeState {
  double n, nend;          // next epoch, last epoch (n > nend: none left)
  double T0, idt;          // first time of the tile, (n_e - 1) / (last - first): the search's first guess
  int lo[32], hi[32];
};

struct WarpState {
  RangeState rg;
  PvRec pv[kPvRing];
  uint16_t expq[kExpQ];
  double coefc[3 * kCoefCache];
  double kpb[kCoefCache];       // per-passband radius ratios (exact per-passband-k mode)
};

// The supersampled path's part of a warp's shared state (the n_ss == 1 kernels do not allocate it).
struct SsState {
  Slot slots[kSlots];
  double item_z[kItemQ];
  uint16_t item_tag[kItemQ];    // slot index of the queued subsample
};

// Ring positions of one warp.  They are warp-uniform and live in registers: every stage is inlined at its single call
// site in the kernel's work loop.
struct WarpCtr {
  int qhead, qcount;            // exposure ring
  int ihead, icount;            // item ring
  int slot_next;                // next slot to hand out (mod kSlots)
  int cur;                      // PvRec of the tile being streamed
};

// Output tag of the fused likelihood (S§8(f) NEXT-1): no flux is stored; every finished in-window exposure
// adds its chi2 correction to chi2[pv] instead.
struct Chi2 { double unused; };
template <typename OutT> constexpr bool kIsChi2 = std::is_same<OutT, Chi2>::value;

template <typename OutT> struct Vec2;
template <> struct Vec2<Chi2> { typedef double2 type; };
template <> struct Vec2<double> { typedef double2 type; };
template <> struct Vec2<float> { typedef float2 type; };

// flux = 1 for one exposure / an aligned pair of exposures, all passbands (streaming stores: the output is write-once).
template <bool NPB1, typename OutT>
__device__ __forceinline__ void store_one(OutT* __restrict__ out, int64_t n_t, int n_pb) {
  if constexpr (kIsChi2<OutT>) {
    return;   // flux 1 is what the chi2 baseline assumes: nothing to add
  } else {
    if (NPB1) PT_ST(out, (OutT)1.0);
    else for (int j = 0; j < n_pb; ++j) PT_ST(out + (int64_t)j * n_t, (OutT)1.0);
  }
}
template <bool NPB1, typename OutT>
__device__ __forceinline__ void store_one_pair(OutT* __restrict__ out, int64_t n_t, int n_pb) {
  if constexpr (kIsChi2<OutT>) {
    return;
  } else {
    typename Vec2<OutT>::type v;
    v.x = (OutT)1.0; v.y = (OutT)1.0;
    if (NPB1) PT_ST((typename Vec2<OutT>::type*)out, v);
    else for (int j = 0; j < n_pb; ++j) PT_ST((typename Vec2<OutT>::type*)(out + (int64_t)j * n_t), v);
  }
}

// Limb-darkening combine (Eq. 13 with the k-correction of P:L179) of one exposure's mean basis functions, and the
// stores.  Single passband: the decrement arrives already combined in `le`.
// One passband's result of a finished exposure: the flux store, or (fused likelihood) the chi2 correction
//   ((o - F) w)² - ((o - 1) w)² = (1-F) w² (2 (o-1) + (1-F)),   o = observed flux, w = 1/sigma,
// formed without cancellation from the decrement 1-F.
template <typename OutT>
__device__ __forceinline__ void emit(const FluxArgs& A, const PvRec& r, OutT* out, uint32_t e, int j, double dec, double& chi) {
  if constexpr (kIsChi2<OutT>) {
    const int64_t idx = (int64_t)j * A.n_t + r.e0 + e;
    const double o = __ldg(A.obs + idx), w = __ldg(A.isig + idx);
    chi = fma(dec * w * w, fma(2.0, o - 1.0, dec), chi);
  } else {
    PT_ST(out + (int64_t)j * A.n_t, (OutT)(1.0 - dec));
  }
}

// Limb-darkening combine (Eq. 13 with the k-correction of P:L179) of one exposure's mean basis functions, and the
// stores.  Single passband: the decrement arrives already combined in `le`.
template <bool NPB1, typename OutT>
__device__ __forceinline__ void finish_exposure(const FluxArgs& A, const WarpState& ws, const PvRec& r, uint32_t e,
                                                double le, double ld, double ed, double* chi_acc = nullptr) {
  OutT* out = (OutT*)r.ob + e;
  double chi = 0.0;
  if (NPB1) {
    emit<OutT>(A, r, out, e, 0, le, chi);
  } else {
    const int n_pb = A.n_pb;
    const int nc = n_pb < kCoefCache ? n_pb : kCoefCache;
    for (int j = 0; j < nc; ++j)
      emit<OutT>(A, r, out, e, j, fma(ws.coefc[3 * j + 2], ed, fma(ws.coefc[3 * j + 1], ld, ws.coefc[3 * j] * le)), chi);
    for (int j = nc; j < n_pb; ++j) {   // beyond the cache: coefficients from the parameter row
      const double k = __ldg(r.row + 6 + 3 * j), u1 = __ldg(r.row + 7 + 3 * j), u2 = __ldg(r.row + 8 + 3 * j);
      const double cj = u1 + 2.0 * u2;
      const double gN = k * k * r.ik2 / (1.0 - u1 / 3.0 - u2 / 6.0);
      emit<OutT>(A, r, out, e, j, fma(gN * u2, ed, fma(gN * cj, ld, gN * (1.0 - cj) * le)), chi);
    }
  }
  if constexpr (kIsChi2<OutT>) {
    if (chi_acc) *chi_acc += chi;          // caller sums over the tile (all of it one parameter vector)
    else atomicAdd(A.chi2 + r.pv, chi);
  }
}

// Table loads carry an L2 evict_last policy: the (k,z) table (60-160 MB) is re-read by every parameter vector while
// gigabytes of write-once flux stream through the same L2 (those go out with evict-first stores).
#ifndef PT_TABLE_POLICY
#define PT_TABLE_POLICY "createpolicy.fractional.L2::evict_last.b64 %0, 1.0;"
#endif
__device__ __forceinline__ unsigned long long l2_keep_policy() {
  unsigned long long pol;
  asm volatile(PT_TABLE_POLICY : "=l"(pol));
  return pol;
}
__device__ __forceinline__ float ldg_keep(const float* p, unsigned long long pol) {
  float v;
  asm volatile("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ double ldg_keep(const double* p, unsigned long long pol) {
  double v;
  asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ float4 ldg_keep4(const float* p, unsigned long long pol) {
  float4 v;
  asm volatile("ld.global.nc.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol));
  return v;
}

// Bilinear lookup of the three functions: lo = t00 + fz (t01 - t00), hi = t10 + fz (t11 - t10),
// v = lo + fk (hi - lo).  A padded fp32 table ([k][z][4], 16-byte nodes) is read with one 16-byte load per corner.
template <typename TT>
__device__ __forceinline__ Basis table_lookup(const FluxArgs& A, int ik, double fk, double z) {
  const unsigned long long pol = l2_keep_policy();
  const double rz = z * A.inv_dz;     // 1 ulp from z/dz: moves fz by 1e-16 rz, the value by < 1e-16 (bilinear is continuous across cells)
  int iz = (int)floor(rz);
  iz = min(max(iz, 0), A.n_z - 2);
  const double fz = rz - (double)iz;
  const TT* r0 = (const TT*)A.tb + ((size_t)ik * A.n_z + iz) * A.n_fn;
  const TT* r1 = r0 + (size_t)A.n_z * A.n_fn;
  double v[3];
  if (sizeof(TT) == 4 && A.n_fn == 4 && (reinterpret_cast<uintptr_t>(A.tb) & 15) == 0) {
    const float4 c00 = ldg_keep4((const float*)r0, pol), c01 = ldg_keep4((const float*)r0 + 4, pol);
    const float4 c10 = ldg_keep4((const float*)r1, pol), c11 = ldg_keep4((const float*)r1 + 4, pol);
    const double t00[3] = {(double)c00.x, (double)c00.y, (double)c00.z}, t01[3] = {(double)c01.x, (double)c01.y, (double)c01.z};
    const double t10[3] = {(double)c10.x, (double)c10.y, (double)c10.z}, t11[3] = {(double)c11.x, (double)c11.y, (double)c11.z};
#pragma unroll
    for (int f = 0; f < 3; ++f) {
      const double lo = fma(fz, t01[f] - t00[f], t00[f]);
      const double hi = fma(fz, t11[f] - t10[f], t10[f]);
      v[f] = fma(fk, hi - lo, lo);
    }
  } else {
#pragma unroll
    for (int f = 0; f < 3; ++f) {
      const double t00 = (double)ldg_keep(r0 + f, pol), t01 = (double)ldg_keep(r0 + A.n_fn + f, pol);
      const double t10 = (double)ldg_keep(r1 + f, pol), t11 = (double)ldg_keep(r1 + A.n_fn + f, pol);
      const double lo = fma(fz, t01 - t00, t00);
      const double hi = fma(fz, t11 - t10, t10);
      v[f] = fma(fk, hi - lo, lo);
    }
  }
  Basis b;
  b.le = v[0]; b.ld = v[1]; b.ed = v[2];
  return b;
}

template <int MODE>
__device__ __forceinline__ Basis eval_basis(const FluxArgs& A, const PvRec& r, double z) {
  if (MODE == 1 && r.use_table)
    return (A.tb_dtype == PT_F64) ? table_lookup<double>(A, r.ik, r.fk, z) : table_lookup<float>(A, r.ik, r.fk, z);
  return ma_basis(r.c.khat, z);
}

// The fp32-arithmetic variant exists in the kernels that store fp32 flux; whether a parameter vector takes it is decided
// once per vector (PvRec::f.use), so the branch below is uniform over a tile.
template <typename OutT> constexpr bool kF32Capable = std::is_same<OutT, float>::value;

// Signed separation of a sample at pinned folded phase ph, and whether it is in transit (0 <= z < 1 + k̂).
template <typename OutT>
__device__ __forceinline__ double sample_z(const PvRec& r, double ph, bool& in) {
  if constexpr (kF32Capable<OutT>) {
    if (r.f.use) {
      const float zf = orbit_z_signed32(r.f, r.c.Mtr, r.c.flags & PV_CIRCULAR, ph);
      in = zf >= 0.0f && zf < 1.0f + r.f.khat;
      return (double)zf;
    }
  }
  const double zs = orbit_z_signed(r.c, ph);
  in = zs >= 0.0 && zs < 1.0 + r.c.khat;
  return zs;
}

// Combined decrement coef0 λe + coef1 λd* + coef2 ηd of an in-transit sample (single passband).
template <int MODE, typename OutT>
__device__ __forceinline__ double sample_dec(const FluxArgs& A, const PvRec& r, double z) {
  if constexpr (kF32Capable<OutT>) {
    if (r.f.use) return (double)ma_dec32(r.f, (float)z);
  }
  const Basis b = eval_basis<MODE>(A, r, z);
  return fma(r.coef[2], b.ed, fma(r.coef[1], b.ld, r.coef[0] * b.le));
}

// 2^s as a double, s clamped to the normal range.
__device__ __forceinline__ double pow2i(int s) {
  s = min(max(s, -1000), 1000);
  return __longlong_as_double((long long)(s + 1023) << 52);
}

// S0: per-tile setup, executed redundantly by all lanes of the warp (same cost as one lane; lane 0 writes).
// Row validation, k̂ (summed in index order, R9), orbit constants and phase window (pv_setup_orbit), combine
// coefficients coef = g (1-c)/N, g c/N, g u2/N with g = k_j²/k̂², table indices, window-test constants.
template <int MODE, bool NPB1, typename OutT>
__device__ __noinline__ void tile_setup(const FluxArgs& A, WarpState& ws, int ring, int64_t pv, int chunk, int reuse) {
  const int lane = threadIdx.x & 31;
  PvRec& r = ws.pv[ring];
  const int n_pb = NPB1 ? 1 : A.n_pb;
  if (reuse >= 0) {   // same parameter vector as the previous tile of this warp: copy its record, move the tile pointers
    const int64_t e0 = (int64_t)chunk * A.tile_len;
    if (reuse != ring) {
      const double* src = reinterpret_cast<const double*>(&ws.pv[reuse]);
      double* dst = reinterpret_cast<double*>(&r);
      for (int i = lane; i < (int)(sizeof(PvRec) / sizeof(double)); i += 32) dst[i] = src[i];
      __syncwarp();
    }
    if (lane == 0) {
      r.tb = A.times + pv * A.t_stride_pv + e0;
      r.ob = kIsChi2<OutT> ? nullptr : (char*)A.flux + (pv * A.flux_pv_stride + A.flux_off + e0) * (int64_t)sizeof(OutT);
      r.e0 = e0;
      r.pv = pv;
    }
    __syncwarp();
    return;
  }
  if (NPB1 && A.pvcache) {   // the record was computed once for the whole launch (prep_kernel): copy, set the tile pointers
    const int64_t e0 = (int64_t)chunk * A.tile_len;
    const double* src = reinterpret_cast<const double*>(A.pvcache + pv);
    double* dst = reinterpret_cast<double*>(&r);
    for (int i = lane; i < (int)(sizeof(PvRec) / sizeof(double)); i += 32) dst[i] = __ldg(src + i);
    __syncwarp();
    if (lane == 0) {
      r.tb = A.times + pv * A.t_stride_pv + e0;
      r.ob = kIsChi2<OutT> ? nullptr : (char*)A.flux + (pv * A.flux_pv_stride + A.flux_off + e0) * (int64_t)sizeof(OutT);
      r.e0 = e0;
    }
    __syncwarp();
    return;
  }
  const double* row = A.params + pv * A.row_stride;
  const double* pbp = row + 6 + 3 * A.pb_first;   // this launch's passbands: (k, u1, u2) triples
  bool ok = true;
  double ksum = 0.0, N0 = 1.0;
  for (int j = 0; j < n_pb; ++j) {
    const double k = __ldg(pbp + 3 * j), u1 = __ldg(pbp + 3 * j + 1), u2 = __ldg(pbp + 3 * j + 2);
    const double N = 1.0 - u1 / 3.0 - u2 / 6.0;
    if (!(isfinite(k) && isfinite(u1) && isfinite(u2)) || !(k >= 0.0) || N == 0.0) ok = false;
    ksum = (!NPB1 && A.pbk) ? fmax(ksum, k) : ksum + k;
    if (j == 0) N0 = N;
  }
  // k̂: the mean radius ratio; per-passband-k mode: the largest one (window and in-transit test must cover all)
  const double khat = (NPB1 || A.pbk) ? ksum : ksum / (double)n_pb;
  PvConst& c = r.c;          // all lanes store the same values
  c.khat = khat;
  pv_setup_orbit(c, row, ok, A.n_ss, A.t_exp);
  const int64_t e0 = (int64_t)chunk * A.tile_len;
  const double ik2 = NPB1 ? 1.0 : (khat > 1.0e-150 ? rcp_fast(khat * khat) : (khat > 0.0 ? 1.0 / (khat * khat) : 0.0));   // single passband: unused
  if (lane == 0) {
    r.tb = A.times + pv * A.t_stride_pv + e0;
    r.ob = kIsChi2<OutT> ? nullptr : (char*)A.flux + (pv * A.flux_pv_stride + A.flux_off + e0) * (int64_t)sizeof(OutT);
    r.e0 = e0;
    r.pv = pv;
    r.row = row;
    r.ik2 = ik2;
    r.use_table = 0;
      r.f.use = 0;
  }
  if (c.flags & PV_BAD) {
    if (chunk == 0 && lane == 0 && A.status) {
      atomicOr(&A.status[0], PT_ST_BAD_PARAM);
      atomicAdd(&A.status[1], 1);
    }
    __syncwarp();
    return;
  }
  if (NPB1) {
    const double u1 = __ldg(pbp + 1), u2 = __ldg(pbp + 2);
    const double cj = u1 + 2.0 * u2;
    const double gN = 1.0 / N0;                           // k²/k̂² = 1 for a single passband
    const double c0 = gN * (1.0 - cj), c1 = gN * cj, c2 = gN * u2;
    // fixed-point scale of the combined decrement c0 λe + c1 λd + c2 ηd (each basis value <= 1): 2^eb > |c0|+|c1|+|c2|
    const double B = fabs(c0) + fabs(c1) + fabs(c2);
    int eb = (int)((__double_as_longlong(B) >> 52) & 0x7ff) - 1022;
    if (!(B > 0.0) || !isfinite(B)) eb = 0;
    if (lane == 0) {
      r.coef[0] = c0; r.coef[1] = c1; r.coef[2] = c2;
      r.acc_scale = pow2i(A.fx_bits - eb);
      r.acc_inv = pow2i(eb - A.fx_bits) * A.inv_nss;
      r.f.use = (A.f32a && MODE == 0 && f32_ok(khat, u1, u2, c.a, c.e)) ? 1 : 0;
      r.f.a = (float)c.a; r.f.cosi = (float)c.cosi; r.f.ci2 = (float)(c.cosi * c.cosi); r.f.e = (float)c.e;
      r.f.sinw = (float)c.sinw; r.f.cosw = (float)c.cosw; r.f.rt1me2 = (float)c.rt1me2; r.f.sin_e = (float)c.sin_e;
      r.f.cos_e = (float)c.cos_e; r.f.khat = (float)khat;
      r.f.coef[0] = (float)c0; r.f.coef[1] = (float)c1; r.f.coef[2] = (float)c2;
    }
  } else {
    for (int j = lane; j < n_pb && j < kCoefCache; j += 32) {
      const double k = __ldg(pbp + 3 * j), u1 = __ldg(pbp + 3 * j + 1), u2 = __ldg(pbp + 3 * j + 2);
      const double cj = u1 + 2.0 * u2;
      const double gN = (A.pbk ? 1.0 : k * k * ik2) / (1.0 - u1 / 3.0 - u2 / 6.0);
      ws.coefc[3 * j + 0] = gN * (1.0 - cj);
      ws.coefc[3 * j + 1] = gN * cj;
      ws.coefc[3 * j + 2] = gN * u2;
      ws.kpb[j] = k;
    }
  }
  if (MODE == 1) {
    const double rk = (khat - A.k_min) / A.dk;
    const bool use_table = (khat >= A.k_min) && (khat <= A.k_min + (A.n_k - 1) * A.dk);
    const int ik = min(max((int)floor(rk), 0), A.n_k - 2);
    if (lane == 0) {
      r.use_table = use_table ? 1 : 0;
      r.ik = ik;
      r.fk = rk - (double)ik;
    }
    if (!use_table && !(c.flags & PV_NEVER) && chunk == 0 && lane == 0 && A.status) {
      atomicOr(&A.status[0], PT_ST_K_OUT_OF_TABLE);
      atomicAdd(&A.status[1], 1);
    }
  }
  // cheap window test (see in_window2): x' = t*invP + c0 approximates (t-t0)/P - mid with an error below
  // 2^-53 (2|x'| + 2|t0/P| + 2|mid|); the test widens the half-width by 2^-50 (|x'| + |t0/P| + |mid| + 1).
  const double t0p = c.t0 * c.invP;
  if (lane == 0) {
    r.w_c0 = -t0p - c.win_mid;
    r.w_half = c.win_half + 0x1p-50 * (fabs(t0p) + fabs(c.win_mid) + 1.0);
  }
  __syncwarp();
}

// Cheap window test on an exposure time: can any subsample of it be in transit?  It is only ever used to SKIP exposures
// whose flux is exactly 1, so it must never say "no" wrongly; the half-width carries the error bound of the cheap fold
// (tile_setup) on top of the 1e-7-cycle margin built into the window.  |x'| >= 2^51: the widened half-width exceeds 2,
// so the test passes whatever the rounding did; NaN/inf times fail it (flux 1, as in the oracle, where every comparison
// with NaN is false).  6 FP64-pipe instructions per exposure.
__device__ __forceinline__ bool in_window2(double t, double invP, double c0, double half) {
  const double x = fma(t, invP, c0);
  const double magic = 6755399441055744.0;   // 1.5 * 2^52
  const double r = __dsub_rn(__dadd_rn(x, magic), magic);
  const double d = x - r;
  return fabs(d) < fma(fabs(x), 0x1p-50, half);
}

// ---------------------------------------------------------------------------------------------------- basis stage
// Evaluate the first n (<= 32) queued subsamples, one per lane.
#ifndef PT_BASIS_INLINE
#define PT_BASIS_INLINE __forceinline__
#endif
template <int MODE, bool NPB1, bool SS1, typename OutT>
__device__ PT_BASIS_INLINE void basis_round(const FluxArgs& A, WarpState& ws, SsState& ss, WarpCtr& C, int n) {
  const int lane = threadIdx.x & 31;
  const bool act = lane < n;
  const int ihead = C.ihead;
  const int idx = (ihead + lane) & (kItemQ - 1);
  if (SS1) {
    return;   // the n_ss == 1 path evaluates its samples in the z-round and never queues items
  } else {
    constexpr int NACC = NPB1 ? 1 : 3;
    const int sid = act ? (int)ss.item_tag[idx] : -1 - lane;   // inactive lanes: unique ids, never equal to a neighbour's
    long long v[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) v[a] = 0;
    int ring = 0;
    if (act) {
      ring = ss.slots[sid].ring;
      const PvRec& r = ws.pv[ring];
      if (NPB1) {
        v[0] = __double2ll_rn(sample_dec<MODE, OutT>(A, r, ss.item_z[idx]) * r.acc_scale);
      } else {
        const Basis b = eval_basis<MODE>(A, r, ss.item_z[idx]);
        v[0] = __double2ll_rn(b.le * A.fx_scale);
        v[NACC - 2] = __double2ll_rn(b.ld * A.fx_scale);
        v[NACC - 1] = __double2ll_rn(b.ed * A.fx_scale);
      }
    }
    // segmented inclusive scan over runs of equal slot id (an exposure's subsamples are contiguous in the queue)
    const int G = A.n_ss < 32 ? A.n_ss : 32;
    for (int o = 1; o < G; o <<= 1) {
      const int so = __shfl_up_sync(0xffffffffu, sid, o);
      const bool take = (lane >= o) && (so == sid);
#pragma unroll
      for (int a = 0; a < NACC; ++a) {
        const long long t = __shfl_up_sync(0xffffffffu, v[a], o);
        if (take) v[a] += t;
      }
    }
    const int sprev = __shfl_up_sync(0xffffffffu, sid, 1);
    const int snext = __shfl_down_sync(0xffffffffu, sid, 1);
    const unsigned heads = __ballot_sync(0xffffffffu, lane == 0 || sprev != sid);
    const bool tail = act && (lane == 31 || snext != sid);
    if (tail) {
      const int head = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
      Slot& s = ss.slots[sid];
      const int rem = s.remaining - (lane - head + 1);
      if (rem == 0) {
        const PvRec& r = ws.pv[ring];
        if (NPB1) {
          finish_exposure<true, OutT>(A, ws, r, s.e, (double)(s.acc[0] + v[0]) * r.acc_inv, 0.0, 0.0);
        } else {
          finish_exposure<false, OutT>(A, ws, r, s.e, (double)(s.acc[0] + v[0]) * A.fx_inv,
                                       (double)(s.acc[NACC - 2] + v[NACC - 2]) * A.fx_inv,
                                       (double)(s.acc[NACC - 1] + v[NACC - 1]) * A.fx_inv);
        }
#ifdef PT_DEBUG_CHECKS
        s.remaining = 0;
#endif
      } else {
        PT_CHECK(rem > 0);
        s.remaining = rem;
#pragma unroll
        for (int a = 0; a < NACC; ++a) s.acc[a] += v[a];
      }
    }
  }
  __syncwarp();
  C.ihead = (ihead + n) & (kItemQ - 1);
  C.icount -= n;
}

// ---------------------------------------------------------------------------------------------------- z-stage
// Expand the first nb (<= EPW = 32/G) queued exposures of the current tile into subsamples, G = min(n_ss,32) lanes each:
// pinned subsample time and phase fold (H1, H2), orbit, in-transit test; compacts the in-transit subsamples into
// the item queue.  One call is one z-round; for n_ss > 32 an exposure takes several calls (`ms0`, `msid` carry the
// subsample offset and the slot across them) so that the kernel can run basis rounds in between from its single call site.
// Per-lane constants of the z-stage, computed once per kernel: group (exposure) and subsample index of the lane, and the
// pinned subsample offset (H2) when one round covers all subsamples.
struct LaneCtx {
  int grp, g;
  double off0;
};

template <int MODE, bool NPB1, bool SS1, typename OutT>
__device__ PT_EXPAND_INLINE void expand(const FluxArgs& A, WarpState& ws, SsState& ss, WarpCtr& C, const LaneCtx& L, int nb, int& ms0, int& msid,
                                        double& chi_acc) {
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  const int cur = C.cur;
  const PvRec& r = ws.pv[cur];
  const int n_pb = NPB1 ? 1 : A.n_pb;
  const int n_ss = SS1 ? 1 : A.n_ss;
  const int G = n_ss < 32 ? n_ss : 32;
  const int grp = L.grp, g = L.g;
  const bool act = grp < nb;
  const int qhead = C.qhead;
  const uint32_t e = act ? ws.expq[(qhead + grp) & (kExpQ - 1)] : 0u;
  const double t = act ? __ldg(r.tb + e) : 0.0;
  const bool slow_div = r.c.flags & PV_SLOWDIV;
  OutT* ob = (OutT*)r.ob;
  if (SS1) {
    // n_ss == 1: an exposure in the window is almost always in transit, so a second compaction would buy nothing; the
    // basis functions are evaluated right here, one exposure per lane, and the item queue stays empty.
    if (act) {
      bool in_tr;
      const double zs = sample_z<OutT>(r, fold_phase(t, r.c.t0, r.c.P, r.c.invP, slow_div), in_tr);
      if (in_tr) {
        if (!NPB1 && MODE == 0 && A.pbk) {
          // exact per-passband-k mode (S§8(f) NEXT-2): one orbit evaluation, the basis functions once per passband at k_j
          double chi = 0.0;
          for (int j = 0; j < n_pb; ++j) {
            double kj, c0, c1, c2;
            if (j < kCoefCache) {
              kj = ws.kpb[j]; c0 = ws.coefc[3 * j]; c1 = ws.coefc[3 * j + 1]; c2 = ws.coefc[3 * j + 2];
            } else {
              const double u1 = __ldg(r.row + 7 + 3 * j), u2 = __ldg(r.row + 8 + 3 * j);
              const double cj = u1 + 2.0 * u2, gN = 1.0 / (1.0 - u1 / 3.0 - u2 / 6.0);
              kj = __ldg(r.row + 6 + 3 * j); c0 = gN * (1.0 - cj); c1 = gN * cj; c2 = gN * u2;
            }
            Basis b;
            b.le = 0.0; b.ld = 0.0; b.ed = 0.0;
            if (kj > 1.0e-150) b = ma_basis(kj, zs);
            emit<OutT>(A, r, (OutT*)r.ob + e, e, j, fma(c2, b.ed, fma(c1, b.ld, c0 * b.le)), chi);
          }
        } else {
          if (NPB1) {
            finish_exposure<true, OutT>(A, ws, r, e, sample_dec<MODE, OutT>(A, r, zs), 0.0, 0.0, &chi_acc);
          } else {
            const Basis b = eval_basis<MODE>(A, r, zs);
            finish_exposure<false, OutT>(A, ws, r, e, b.le, b.ld, b.ed, &chi_acc);
          }
        }
      } else {
        store_one<NPB1, OutT>(ob + e, A.n_t, n_pb);
      }
    }
    C.qhead = (qhead + nb) & (kExpQ - 1);
    C.qcount -= nb;
    return;
  } else {
    const bool multi = n_ss > 32;             // one exposure per round, several sub-rounds of 32 subsamples
    const unsigned gmask = (G == 32 ? 0xffffffffu : ((1u << G) - 1u)) << (grp * G);
    const unsigned below = (grp * G >= 32) ? 0xffffffffu : ((1u << (grp * G)) - 1u);   // lanes of earlier groups
    const int s0 = multi ? ms0 : 0;
    int sid = multi ? msid : -1;
    {
      const int s = s0 + g;
      bool p = false;
      double zs = 0.0;
      if (act && s < n_ss) {
        const double ts = __dadd_rn(t, multi ? subsample_offset(s, n_ss, A.t_exp) : L.off0);
        zs = sample_z<OutT>(r, fold_phase(ts, r.c.t0, r.c.P, r.c.invP, slow_div), p);
      }
      const unsigned m = __ballot_sync(0xffffffffu, p);
      int nalloc = 0;
      if (!multi) {
        const int cnt = __popc(m & gmask);
        const bool has = act && cnt > 0;
        const unsigned hm = __ballot_sync(0xffffffffu, has && g == 0);
        sid = (C.slot_next + __popc(hm & below)) & (kSlots - 1);
        nalloc = __popc(hm);
        if (act && g == 0) {
          if (has) {
            Slot& sl = ss.slots[sid];
            PT_CHECK(sl.remaining == 0);
            sl.acc[0] = 0; sl.acc[1] = 0; sl.acc[2] = 0;
            sl.remaining = cnt; sl.e = (uint16_t)e; sl.ring = (uint16_t)cur;
          } else {
            store_one<NPB1, OutT>(ob + e, A.n_t, n_pb);
          }
        }
      } else if (m) {
        if (sid < 0) {
          sid = C.slot_next & (kSlots - 1);
          nalloc = 1;
          if (lane == 0) {
            Slot& sl = ss.slots[sid];
            PT_CHECK(sl.remaining == 0);
            sl.acc[0] = 0; sl.acc[1] = 0; sl.acc[2] = 0;
            sl.remaining = kRemBias; sl.e = (uint16_t)e; sl.ring = (uint16_t)cur;
          }
          __syncwarp();
        }
        if (lane == 0) ss.slots[sid].remaining += __popc(m);
      }
      if (p) {
        const int pos = (C.ihead + C.icount + __popc(m & lt)) & (kItemQ - 1);
        ss.item_z[pos] = zs;
        ss.item_tag[pos] = (uint16_t)sid;
      }
      __syncwarp();
      C.icount += __popc(m);
      PT_CHECK(C.icount <= kItemQ);
      C.slot_next = (C.slot_next + nalloc) & (kSlots - 1);
    }
    if (multi) {
      ms0 = s0 + 32;
      msid = sid;
      if (ms0 < n_ss) return;                 // more sub-rounds of this exposure to come
      ms0 = 0;
      msid = -1;
      if (sid < 0) {
        if (lane == 0) store_one<NPB1, OutT>(ob + e, A.n_t, n_pb);
      } else if (lane == 0) {
        Slot& sl = ss.slots[sid];
        const int rem = sl.remaining - kRemBias;
        sl.remaining = rem;
        if (rem == 0) {   // every subsample was already evaluated by the basis rounds in between
          if (NPB1) finish_exposure<true, OutT>(A, ws, r, e, (double)sl.acc[0] * r.acc_inv, 0.0, 0.0);
          else finish_exposure<false, OutT>(A, ws, r, e, (double)sl.acc[0] * A.fx_inv, (double)sl.acc[1] * A.fx_inv,
                                            (double)sl.acc[2] * A.fx_inv);
        }
      }
    }
    __syncwarp();
    C.qhead = (qhead + nb) & (kExpQ - 1);
    C.qcount -= nb;
  }
}

// Per-pv scheduling: find the next parameter vector after `pv` (cyclically) that still has tiles and take one.
// Lanes look at 32 counters at a time (plain loads: a stale value only costs a wasted ticket), then one ticket is drawn
// from the first candidate; a counter only ever grows, so an exhausted parameter vector stays exhausted.
__device__ __forceinline__ bool next_pv(const FluxArgs& A, int64_t& pv, int& chunk) {
  const int lane = threadIdx.x & 31;
  const int64_t n_pv = A.n_pv;
  const unsigned long long tpp = (unsigned long long)A.tiles_per_pv;
  for (int64_t off = 1; off < n_pv; off += 32) {
    const int64_t cand = (pv + off + lane) % n_pv;
    const bool in_range = off + lane < n_pv;
    const unsigned long long seen = in_range ? *((volatile unsigned long long*)(A.sched + kSchedHead + cand)) : tpp;
    unsigned avail = __ballot_sync(0xffffffffu, seen < tpp);
    while (avail) {
      const int src = __ffs(avail) - 1;
      avail &= avail - 1u;
      const int64_t target = (pv + off + src) % n_pv;
      unsigned long long got = 0;
      if (lane == 0) got = atomicAdd(A.sched + kSchedHead + target, 1ULL);
      got = __shfl_sync(0xffffffffu, got, 0);
      if (got < tpp) {
        pv = target;
        chunk = (int)got;
        return true;
      }
    }
  }
  return false;
}

// flux = 1 for exposures [a, b) of the tile, all passbands: the out-of-transit stretches of range mode.  V == 2: a and b
// are even and the rows 16-byte aligned, every lane stores aligned pairs; 512 contiguous bytes per warp instruction.
template <int V, bool NPB1, typename OutT>
__device__ __forceinline__ void fill_ones(OutT* __restrict__ ob, uint32_t a, uint32_t b, int64_t n_t, int n_pb) {
  if constexpr (kIsChi2<OutT>) {
    return;   // flux 1 is what the chi2 baseline assumes
  } else {
    const uint32_t lane = threadIdx.x & 31;
    const int np = NPB1 ? 1 : n_pb;
    const uint32_t n = b - a;                       // warp-uniform: the trip count is too, only the tail is predicated
    for (int j = 0; j < np; ++j) {
      if (V == 2) {
        typedef typename Vec2<OutT>::type V2;
        V2 v;
        v.x = (OutT)1.0; v.y = (OutT)1.0;
        V2* p = (V2*)(ob + (int64_t)j * n_t + a) + lane;
#pragma unroll 4
        for (uint32_t i = n >> 6; i > 0; --i) { PT_ST(p, v); p += 32; }
        if (2u * lane < (n & 63u)) PT_ST(p, v);
      } else {
        OutT* p = ob + (int64_t)j * n_t + a + lane;
#pragma unroll 4
        for (uint32_t i = n >> 5; i > 0; --i) { PT_ST(p, (OutT)1.0); p += 32; }
        if (lane < (n & 31u)) PT_ST(p, (OutT)1.0);
      }
    }
  }
}

// First index i in [0, n] with t[i] >= x (STRICT = false) or t[i] > x (STRICT = true) in the ascending array t[0..n),
// given four consecutive values v[0..3] = t[s..s+3] that were loaded around the index a uniform cadence predicts (the
// caller issues those loads for both ends of a range at once: one memory latency per batch of epochs).  If the answer is
// not bracketed by the probe (an unevenly sampled axis), gallop outwards from it and bisect: O(log n) for any ascending axis.
template <bool STRICT>
__device__ __forceinline__ int search_sorted(const double* __restrict__ t, int n, double x, int s, const double (&v)[4]) {
  int c = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) c += (STRICT ? v[i] <= x : v[i] < x) ? 1 : 0;
  if ((c > 0 || s == 0) && (c < 4 || s + 4 >= n)) return min(s + c, n);
  int lo, hi;
  if (c == 0) {                      // the answer is < s: gallop down
    hi = s;
    lo = s - 1;
    int step = 1;
    while (lo >= 0) {
      const double w = __ldg(t + lo);
      if (STRICT ? w <= x : w < x) break;
      hi = lo; lo -= step; step <<= 1;
    }
    lo = max(lo, -1) + 1;
  } else {                           // the answer is > s + 3: gallop up
    lo = s + 4;
    hi = s + 4;
    int step = 1;
    while (hi < n) {
      const double w = __ldg(t + hi);
      if (!(STRICT ? w <= x : w < x)) break;
      lo = hi + 1; hi += step; step <<= 1;
    }
    hi = min(hi, n);
  }
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    const double w = __ldg(t + mid);
    if (STRICT ? w <= x : w < x) lo = mid + 1; else hi = mid;
  }
  return lo;
}
// Start of the four-value probe for x: one below the index a uniform cadence predicts, clamped so that s..s+3 is in range
// (n >= 4; shorter tiles never take range mode).
__device__ __forceinline__ int probe_start(double x, int n, double T0, double idt) {
  const double gf = (x - T0) * idt;
  const int g = gf > 1.0 ? (gf < (double)(n - 1) ? (int)gf : n - 1) : 1;
  return min(g - 1, n - 4);
}

// ---------------------------------------------------------------------------------------------------- the kernel
// MODE 0: exact.  MODE 1: interpolated (exact basis functions for a parameter vector whose k̂ is off the table).
// V: exposures per lane and load/store in the stream stage (2 = 16-byte ld/st, needs even row lengths/strides and
// 16-byte aligned bases).  NPB1: single passband.  SS1: n_ss == 1 (no supersample accumulation).
template <int MODE, int V, bool NPB1, bool SS1, typename OutT>
__global__ void __launch_bounds__(kThreads, PT_MIN_BLOCKS) flux_kernel(const __grid_constant__ FluxArgs A) {
  __shared__ WarpState s_ws[kWarpsPerBlock];
  __shared__ SsState s_ss[SS1 ? 1 : kWarpsPerBlock];
  SsState& ss = s_ss[SS1 ? 0 : (threadIdx.x >> 5)];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  WarpState& ws = s_ws[warp];
#ifdef PT_DEBUG_CHECKS
  if (!SS1) for (int i = lane; i < kSlots; i += 32) ss.slots[i].remaining = 0;
  __syncwarp();
#endif
  WarpCtr C;
  C.qhead = 0; C.qcount = 0; C.ihead = 0; C.icount = 0; C.slot_next = 0; C.cur = 0;
  const int n_pb = NPB1 ? 1 : A.n_pb;
  const int n_ss = SS1 ? 1 : A.n_ss;
  const int EPW = 32 / (n_ss < 32 ? n_ss : 32);
  constexpr uint32_t kSuper = 32u * kUnroll * V;
  LaneCtx L;
  {
    const int G = n_ss < 32 ? n_ss : 32;
    L.grp = lane / G;
    L.g = lane - L.grp * G;
    L.off0 = (n_ss > 1 && n_ss <= 32) ? subsample_offset(L.g, n_ss, A.t_exp) : 0.0;
  }
  const int64_t gw = (int64_t)blockIdx.x * kWarpsPerBlock + warp, nw = (int64_t)gridDim.x * kWarpsPerBlock;

  // Tiles are dealt dynamically from counters in the launch's scheduler slot; the next ticket is always drawn before the
  // current tile is processed, so the atomic's latency is hidden.
  //   global mode: one counter over all (pv, chunk) tiles; a warp starts with tile `gw`.
  //   per-pv mode (few parameter vectors, several tiles each): one counter per parameter vector; a warp stays on its
  //     parameter vector (setup done once, later tiles only move the tile pointers) and moves on to the next one that has
  //     tiles left when it is exhausted, so fast parameter vectors lend their warps to slow ones.
  // The last warp to finish zeroes the slot for the next launch that uses it.
  // Row order of the tiles (global mode): prep_kernel ranks the rows — by decreasing expected in-window fraction for the
  // exact model (longest processing time first: the launch ends on light tiles), by k̂ for the interpolated model (tiles
  // in flight then share a few k-rows of the table, which stay in L1/L2 while gigabytes of flux stream past).
  // The slot (order, records, flags) is written by prep_kernel, whose programmatic dependent this grid is.
  if (A.prep) asm volatile("griddepcontrol.wait;" ::: "memory");
  const bool sorted_axis = A.range && !(*((volatile const unsigned long long*)(A.sched + kW_Flags)) & kSlotUnsorted);
  const int tpp = A.tiles_per_pv;
  int64_t pv_cur = 0, last_pv = -1;
  int chunk_cur = 0, last_ring = -1;
  bool have;
  if (!A.per_pv) {
    have = gw < A.n_tiles;
    pv_cur = gw / tpp;
    chunk_cur = (int)(gw - pv_cur * tpp);
    if (A.order && have) pv_cur = (int64_t)__ldg(A.order + pv_cur);
  } else {
    pv_cur = gw % A.n_pv;
    unsigned long long f0 = 0;
    if (lane == 0) f0 = atomicAdd(A.sched + kSchedHead + pv_cur, 1ULL);
    f0 = __shfl_sync(0xffffffffu, f0, 0);
    have = f0 < (unsigned long long)tpp;
    chunk_cur = (int)f0;
    if (!have) have = next_pv(A, pv_cur, chunk_cur);
  }

  // The warp's work loop is a small state machine so that every stage has exactly ONE call site (one copy of its code:
  // the stages are large, and two inlined copies of the basis functions need not round identically).  Priority: a full
  // basis round, then a z-round, then the next piece of streaming / the next tile.
  enum { PH_NEWTILE, PH_STREAM, PH_EXIT };
  int phase = have ? PH_NEWTILE : PH_EXIT;
  bool drain_all = false;        // empty the item queue (ragged last round) before going on
  int keep = EPW;                // z-rounds run while the exposure ring holds at least this many entries
  int ms0 = 0, msid = -1;        // n_ss > 32: sub-round state of the exposure being expanded
  double chi_acc = 0.0;          // fused likelihood, n_ss == 1: this lane's chi2 corrections of the current tile
  uint32_t base = 0, n_e = 0;
  // range mode: position in / size of the current batch of epochs (the rest of the state lives in ws.rg)
  bool rng_on = false;
  int rng_i = 0, rng_cnt = 0;
  unsigned long long fetched = 0;
  const double* __restrict__ tb = nullptr;
  OutT* __restrict__ ob = nullptr;
  double w_invP = 0.0, w_c0 = 0.0, w_half = 0.0;

  for (;;) {
    if (!SS1) {
      const int ic = C.icount;
      if (ic >= 32 || (drain_all && ic > 0)) {
        basis_round<MODE, NPB1, SS1, OutT>(A, ws, ss, C, min(ic, 32));
        continue;
      }
      drain_all = false;
    }
    {
      const int qc = C.qcount;
      if (qc >= keep) {
        expand<MODE, NPB1, SS1, OutT>(A, ws, ss, C, L, min(qc, EPW), ms0, msid, chi_acc);
        continue;
      }
    }
    if (phase == PH_STREAM) {
      if (base >= n_e) {
        // tile finished (the exposure ring is empty: keep was 1).  Multi-passband: the coefficient cache belongs to this
        // parameter vector, so the item queue is emptied too.
        if (!NPB1 && !SS1 && C.icount > 0) { drain_all = true; continue; }
        if (kIsChi2<OutT> && SS1) {   // one atomic per tile: lane sums, then a shuffle tree
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) chi_acc += __shfl_xor_sync(0xffffffffu, chi_acc, o);
          if (lane == 0 && chi_acc != 0.0) atomicAdd(A.chi2 + pv_cur, chi_acc);
          chi_acc = 0.0;
        }
        const unsigned long long nf = __shfl_sync(0xffffffffu, fetched, 0);
        if (!A.per_pv) {
          const int64_t tile = nw + (int64_t)nf;
          have = tile < A.n_tiles;
          pv_cur = tile / tpp;
          chunk_cur = (int)(tile - pv_cur * tpp);
          if (A.order && have) pv_cur = (int64_t)__ldg(A.order + pv_cur);
        } else if (nf < (unsigned long long)tpp) {
          chunk_cur = (int)nf;
        } else {
          have = next_pv(A, pv_cur, chunk_cur);
        }
        phase = have ? PH_NEWTILE : PH_EXIT;
        continue;
      }
      if (rng_on) {
        // ---- range mode: exposures between the in-window ranges are pure fills (no time loads, no arithmetic)
        const PvRec& r = ws.pv[C.cur];
        do {
          if (rng_i == rng_cnt) {
            const double n0 = ws.rg.n, nend = ws.rg.nend;
            if (!(n0 <= nend)) {                                   // no epoch left: the rest of the tile is out of transit
              fill_ones<V, NPB1, OutT>(ob, base, n_e, A.n_t, n_pb);
              base = n_e;
              break;
            }
            // next batch of epochs, one per lane: [t0 + (n + ex_lo) P, t0 + (n + ex_hi) P] widened by the rounding of this
            // very expression (ex_lo/ex_hi already carry the 1e-7-cycle margin of the window, pt_orbit.cuh)
            const double n = n0 + (double)lane;
            int lo = (int)n_e, hi = (int)n_e;
            if (n <= nend) {
              const double padn = 0x1p-49 * (fabs(n) + fabs(r.c.t0 * r.c.invP) + 1.0);
              const double tlo = fma(r.c.P, n + (r.c.ex_lo - padn), r.c.t0);
              const double thi = fma(r.c.P, n + (r.c.ex_hi + padn), r.c.t0);
              const double T0 = ws.rg.T0, idt = ws.rg.idt;
              const int sl = probe_start(tlo, (int)n_e, T0, idt), sh = probe_start(thi, (int)n_e, T0, idt);
              double vl[4], vh[4];
#pragma unroll
              for (int i = 0; i < 4; ++i) { vl[i] = __ldg(tb + sl + i); vh[i] = __ldg(tb + sh + i); }   // 8 independent loads
              lo = search_sorted<false>(tb, (int)n_e, tlo, sl, vl) & ~(V - 1);
              hi = min((search_sorted<true>(tb, (int)n_e, thi, sh, vh) + (V - 1)) & ~(V - 1), (int)n_e);
            }
            __syncwarp();
            ws.rg.lo[lane] = lo; ws.rg.hi[lane] = hi;
            if (lane == 0) ws.rg.n = n0 + 32.0;
            __syncwarp();
            const double left = nend - n0 + 1.0;
            rng_cnt = left < 32.0 ? (int)left : 32;
            rng_i = 0;
          }
          const int lo = max(ws.rg.lo[rng_i], (int)base);
          const int hi = ws.rg.hi[rng_i];
          if (hi <= lo) { ++rng_i; continue; }                     // no exposure at this epoch (or swallowed by the previous range)
          fill_ones<V, NPB1, OutT>(ob, base, (uint32_t)lo, A.n_t, n_pb);
          const int cnt = min(hi - lo, 32);
          if (lane < cnt) {
            ws.expq[(C.qhead + C.qcount + lane) & (kExpQ - 1)] = (uint16_t)(lo + lane);
            if ((lane & 15) == 0) asm volatile("prefetch.global.L1 [%0];" ::"l"(tb + lo + lane));   // times the z-round reads next
          }
          __syncwarp();
          C.qcount += cnt;
          PT_CHECK(C.qcount <= kExpQ);
          base = (uint32_t)(lo + cnt);
          if ((int)base >= hi) ++rng_i;
        } while (C.qcount < EPW);
        if (base >= n_e) keep = 1;
        continue;
      }
      // ---- stream super-groups of kUnroll x 32 lanes x V exposures until a z-round is due or the tile ends
      do {
      unsigned inw = 0;                                          // bit (u*V+v): exposure (u,v) of this lane is in the window
      if (base + kSuper <= n_e) {                                // warp-uniform
        double t[kUnroll][V];
        if (base + 2 * kSuper <= n_e) {                          // next super-group's times -> L1 while this one is processed
#pragma unroll
          for (int u = 0; u < kUnroll; ++u)
            asm volatile("prefetch.global.L1 [%0];" ::"l"(tb + base + kSuper + (u * 32 + lane) * V));
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {                      // all loads first: kUnroll independent requests per lane
          const uint32_t e = base + (u * 32 + lane) * V;
          if (V == 2) { const double2 tv = __ldg((const double2*)(tb + e)); t[u][0] = tv.x; t[u][V - 1] = tv.y; }
          else t[u][0] = __ldg(tb + e);
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
          const uint32_t e = base + (u * 32 + lane) * V;
          unsigned pair = 0;
#pragma unroll
          for (int v = 0; v < V; ++v) pair |= in_window2(t[u][v], w_invP, w_c0, w_half) ? (1u << v) : 0u;
          inw |= pair << (u * V);
          if (V == 2 && pair == 0) store_one_pair<NPB1, OutT>(ob + e, A.n_t, n_pb);
          else {
#pragma unroll
            for (int v = 0; v < V; ++v) if (!((pair >> v) & 1u)) store_one<NPB1, OutT>(ob + e + v, A.n_t, n_pb);
          }
        }
      } else {                                                   // ragged end of the tile: rolled, one exposure at a time
#pragma unroll 1
        for (int uv = 0; uv < kUnroll * V; ++uv) {
          const uint32_t e = base + ((uv / V) * 32 + lane) * V + (uv % V);
          if (e < n_e) {
            if (in_window2(__ldg(tb + e), w_invP, w_c0, w_half)) inw |= 1u << uv;
            else store_one<NPB1, OutT>(ob + e, A.n_t, n_pb);
          }
        }
      }
      // append the in-window exposures to the exposure ring, one 32-lane row (u) at a time: a transit is a run of
      // consecutive exposures, so only one or two rows have any; per row two ballots give every lane its place, in
      // time order, without divergence
      unsigned rows = __reduce_or_sync(0xffffffffu, inw);
      if (rows) {
        const unsigned lt = (1u << lane) - 1u;
        int tail = C.qhead + C.qcount;
        do {
          const int u = (__ffs(rows) - 1) / V;
          rows &= ~(((1u << V) - 1u) << (u * V));
          const unsigned pair = (inw >> (u * V)) & ((1u << V) - 1u);
          const unsigned b0 = __ballot_sync(0xffffffffu, pair & 1u);
          const unsigned b1 = (V == 2) ? __ballot_sync(0xffffffffu, pair & 2u) : 0u;
          const int off = tail + __popc(b0 & lt) + __popc(b1 & lt);
          const uint32_t e0 = base + (u * 32 + lane) * V;
          if (pair & 1u) ws.expq[off & (kExpQ - 1)] = (uint16_t)e0;
          if (V == 2 && (pair & 2u)) ws.expq[(off + (int)(pair & 1u)) & (kExpQ - 1)] = (uint16_t)(e0 + 1);
          tail += __popc(b0) + __popc(b1);
        } while (rows);
        __syncwarp();
        C.qcount = tail - C.qhead;
        PT_CHECK(C.qcount <= kExpQ);
      }
      base += kSuper;
      } while (base < n_e && C.qcount < EPW);
      if (base >= n_e) keep = 1;      // end of the tile: the exposure ring holds this tile's indices, so it is emptied
      continue;
    }
    if (phase == PH_NEWTILE) {
      // the PvRec this tile will use must not be referenced by queued subsamples any more
      const int ring = NPB1 ? ((C.cur + 1) & (kPvRing - 1)) : 0;
      if (!SS1 && C.icount > 0) {
        bool clash = true;
        if (NPB1) clash = ((int)ss.slots[ss.item_tag[C.ihead]].ring == ring);
        if (clash) { drain_all = true; continue; }
      }
      fetched = 0;
      if (lane == 0) fetched = atomicAdd(A.per_pv ? A.sched + kSchedHead + pv_cur : A.sched, 1ULL);
      tile_setup<MODE, NPB1, OutT>(A, ws, ring, pv_cur, chunk_cur, (pv_cur == last_pv) ? last_ring : -1);
      last_pv = pv_cur;
      last_ring = ring;
      C.cur = ring;
      const PvRec& r = ws.pv[ring];
      n_e = (uint32_t)min((int64_t)A.tile_len, A.n_t - (int64_t)chunk_cur * A.tile_len);
      tb = r.tb;
      ob = (OutT*)r.ob;
      base = 0;
      keep = EPW;
      if (r.c.flags & PV_BAD) {
        if constexpr (kIsChi2<OutT>) {
          if (chunk_cur == 0 && lane == 0 && !A.base_added) atomicAdd(A.chi2 + pv_cur, nan64());
        } else {
          for (int j = 0; j < n_pb; ++j)
            for (uint32_t e = lane; e < n_e; e += 32) ob[(int64_t)j * A.n_t + e] = (OutT)nan64();
        }
        base = n_e;       // nothing to stream
        keep = 1;
      } else if (kIsChi2<OutT> && chunk_cur == 0 && !A.base_added) {
        // chi2 of this parameter vector starts from the all-out-of-transit value: partial sums in fixed order
        double b = 0.0;
        for (int i = lane; i < A.n_base_part; i += 32) b += A.base_part[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) b += __shfl_xor_sync(0xffffffffu, b, o);
        if (lane == 0) atomicAdd(A.chi2 + pv_cur, b);
      }
      w_invP = r.c.invP; w_c0 = r.w_c0; w_half = r.w_half;
      // range mode for this tile?  Needs the ascending axis and no more transit epochs than a few per hundred exposures
      // (else the per-exposure window test is the cheaper way); a row that is always in the window streams as before
      rng_on = false;
      if (sorted_axis && base + 4 <= n_e && !(r.c.flags & PV_ALWAYS)) {
        if (r.c.flags & PV_NEVER) {
          rng_on = true;
          if (lane == 0) { ws.rg.n = 0.0; ws.rg.nend = -1.0; }
        } else {
          const double T0 = __ldg(tb), T1 = __ldg(tb + (n_e - 1));
          const double x0 = (T0 - r.c.t0) * r.c.invP, x1 = (T1 - r.c.t0) * r.c.invP;
          const double pad = 0x1p-49 * (fabs(x0) + fabs(x1) + 2.0);
          const double n0 = ceil(x0 - r.c.ex_hi - pad), n1 = floor(x1 - r.c.ex_lo + pad);
          if (n1 - n0 + 1.0 <= 0.0625 * (double)n_e + 2.0) {       // false for NaN/inf (they never reach here: the axis is finite)
            rng_on = true;
            if (lane == 0) {
              ws.rg.n = n0; ws.rg.nend = n1;
              ws.rg.T0 = T0;
              ws.rg.idt = (T1 > T0) ? (double)(n_e - 1) / (T1 - T0) : 0.0;
            }
          }
        }
        __syncwarp();
        rng_i = 0; rng_cnt = 0;
      }
      phase = PH_STREAM;
      continue;
    }
    // PH_EXIT
    if (!SS1 && C.icount > 0) { drain_all = true; continue; }
    break;
  }
  if (lane == 0) {
    const unsigned long long done = atomicAdd(A.sched + 1, 1ULL);
    if (done == (unsigned long long)nw - 1ULL) {   // every warp has taken its last ticket: nobody reads the slot any more
      const int64_t nwords = kSchedHead + (A.per_pv ? A.n_pv : 0);
      for (int64_t i = 0; i < nwords; ++i) A.sched[i] = 0ULL;
    }
  }
}

// ---------------------------------------------------------------------------------------------------- prep kernel
// Everything the flux kernel wants to find ready in its scheduler slot, in one small launch in front of it (the flux kernel
// is its programmatic dependent: it starts launching at once and waits for this grid before it reads the slot).  Blocks
// take one of four roles by index:
//   records   a warp per parameter vector runs the per-tile setup once and stores the record (single passband, at most
//             kPvCacheMax vectors with several tiles each: the flux kernel then only copies it per tile); raises the
//             status flags that the flux kernel's own setup would have raised
//   axis      is the shared time axis ascending and finite?  (range mode; kSlotUnsorted is set otherwise)
//   order     row order of the tiles by counting sort on a 12-bit key: decreasing expected in-window fraction
//             sqrt((1+k)² - b²)/(π a) + t_exp/P for the exact model (the estimate only orders tiles), k̂ for the table
//   baseline  fused likelihood: partial sums of the all-out-of-transit chi2, fixed order; chi2[] zeroed
struct PrepArgs {
  PvRec* rec;
  uint32_t* order;
  int order_by_k;
  int n_rec_blocks, n_axis_blocks, n_order_blocks, n_base_blocks;
  double* base_part;
  // units of the epoch kernel (pt_epoch.cuh): per-row first epoch and unit count (records role)
  double* un0;
  uint32_t* ucnt;
  int want_units;
  int n_blocks;              // blocks of this launch
};
constexpr int kOrderBins = 4096;

// Units of evaluation work of one parameter vector on the shared ascending axis [T_first, T_last] (epoch kernel): the
// transit epochs n0 .. n0 + cnt - 1 whose window [t0 + (n + ex_lo) P, t0 + (n + ex_hi) P] can hold an exposure, or — a row
// that is always in the window, or whose windows are so dense that looking for them costs more than evaluating every
// exposure — chunks of kChunkLen exposures (kUnitChunks).  Rows that never transit or are bad have no units.
__device__ __forceinline__ void pv_units(const PvConst& c, double T_first, double T_last, int64_t n_t, double* n0, uint32_t* cnt) {
  *n0 = 0.0; *cnt = 0u;
  if (c.flags & (PV_BAD | PV_NEVER)) return;
  const uint32_t chunks = kUnitChunks | (uint32_t)((n_t + kChunkLen - 1) / kChunkLen);
  if (c.flags & PV_ALWAYS) { *cnt = chunks; return; }
  const double x0 = (T_first - c.t0) * c.invP, x1 = (T_last - c.t0) * c.invP;
  const double pad = 0x1p-49 * (fabs(x0) + fabs(x1) + 2.0);
  const double a = ceil(x0 - c.ex_hi - pad), b = floor(x1 - c.ex_lo + pad);
  const double m = b - a + 1.0;
  if (!(m == m) || fabs(m) > 1.0e300) { *cnt = chunks; return; }   // non-finite axis ends: the row is cut into chunks
  if (!(m >= 1.0)) return;                                  // no epoch on the axis
  if (m > 0.125 * (double)n_t + 2.0 || m > 1.0e9) { *cnt = chunks; return; }
  *n0 = a; *cnt = (uint32_t)m;
}

template <int MODE>
__global__ void __launch_bounds__(kThreads) prep_kernel(const __grid_constant__ FluxArgs A, const __grid_constant__ PrepArgs Q) {
  __shared__ WarpState s_ws[kWarpsPerBlock];          // records role; the other roles overlay their scratch on it
  __shared__ int s_last;
  static_assert(sizeof(s_ws) >= kOrderBins * sizeof(int) + kThreads * sizeof(int), "order scratch must fit");
  static_assert(sizeof(s_ws) >= kThreads * sizeof(double), "reduction scratch must fit");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  asm volatile("griddepcontrol.launch_dependents;");   // the flux kernel may start launching: it waits before it reads
  int b = blockIdx.x;
  if (b < Q.n_rec_blocks) {
    const int64_t pv = (int64_t)b * kWarpsPerBlock + warp;
    if (pv < A.n_pv) {
      WarpState& ws = s_ws[warp];
      tile_setup<MODE, true, double>(A, ws, 0, pv, 0, -1);
      const double* src = reinterpret_cast<const double*>(&ws.pv[0]);
      double* dst = reinterpret_cast<double*>(Q.rec + pv);
      for (int i = lane; i < (int)(sizeof(PvRec) / sizeof(double)); i += 32) dst[i] = src[i];
      if (Q.want_units && lane == 0) {
        double n0; uint32_t cnt;
        pv_units(ws.pv[0].c, __ldg(A.times), __ldg(A.times + A.n_t - 1), A.n_t, &n0, &cnt);
        Q.un0[pv] = n0; Q.ucnt[pv] = cnt;
      }
    }
  } else if ((b -= Q.n_rec_blocks) < Q.n_axis_blocks) {
    // adjacent pairs (j, j+1): NaN fails the comparison; the ends must be finite
    bool bad = false;
    const int64_t n = A.n_t;
    for (int64_t j = (int64_t)b * kThreads + threadIdx.x; j + 1 < n; j += (int64_t)Q.n_axis_blocks * kThreads)
      bad |= !(__ldg(A.times + j) <= __ldg(A.times + j + 1));
    if (b == 0 && threadIdx.x == 0) bad |= !(fabs(__ldg(A.times)) < CUDART_INF) || !(fabs(__ldg(A.times + n - 1)) < CUDART_INF);
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(A.sched + kW_Flags, kSlotUnsorted);
  } else if ((b -= Q.n_axis_blocks) < Q.n_order_blocks) {
    int* hist = reinterpret_cast<int*>(s_ws);            // kOrderBins counters, then kThreads partial sums
    int* part = hist + kOrderBins;
    const int n = (int)A.n_pv;
    for (int i = threadIdx.x; i < kOrderBins; i += kThreads) hist[i] = 0;
    __syncthreads();
    auto key_of = [&](int i) -> int {
      const double* row = A.params + (int64_t)i * A.row_stride;
      const double k = __ldg(row + 6 + 3 * A.pb_first);
      float q;
      if (Q.order_by_k) {
        q = (float)((k - A.k_min) / (A.dk * (double)(A.n_k - 1)));              // position of k in the table's range
      } else {
        const double P = __ldg(row + 1), a = __ldg(row + 2), ci = cos(__ldg(row + 3));
        const double bb = a * ci, c2 = (1.0 + k) * (1.0 + k) - bb * bb;
        q = 1.0f - (float)(sqrt(fmax(c2, 0.0)) / (3.14159 * a) + ((A.n_ss > 1) ? fabs(A.t_exp / P) : 0.0));
        if (!(q == q) || q > 1.0f || q < 0.0f) q = 0.0f;   // odd rows (bad parameters, a < 1+k): treat as heavy
      }
      if (!(q == q)) q = 0.0f;
      return min(max((int)(q * (float)(kOrderBins - 1)), 0), kOrderBins - 1);
    };
    for (int i = threadIdx.x; i < n; i += kThreads) atomicAdd(&hist[key_of(i)], 1);
    __syncthreads();
    // exclusive scan of the histogram: each thread owns kOrderBins / kThreads consecutive bins
    constexpr int kPer = kOrderBins / kThreads;
    int sum = 0;
    for (int j = 0; j < kPer; ++j) sum += hist[threadIdx.x * kPer + j];
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
      int run = 0;
      for (int t = 0; t < kThreads; ++t) { const int v = part[t]; part[t] = run; run += v; }
    }
    __syncthreads();
    int run = part[threadIdx.x];
    for (int j = 0; j < kPer; ++j) { const int v = hist[threadIdx.x * kPer + j]; hist[threadIdx.x * kPer + j] = run; run += v; }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += kThreads) Q.order[atomicAdd(&hist[key_of(i)], 1)] = (uint32_t)i;
  } else {
    b -= Q.n_order_blocks;
    // chi2 of the all-out-of-transit model, sum over (passband, exposure) of ((obs - 1) / sigma)²: block b reduces a
    // contiguous range in a fixed order (strided per-thread sums, then a shared-memory tree) and writes one partial; the
    // flux kernel adds the partials, again in a fixed order, to every parameter vector.
    double* s_sum = reinterpret_cast<double*>(s_ws);
    const int64_t n = (int64_t)A.n_pb * A.n_t;
    const int64_t per = (n + Q.n_base_blocks - 1) / Q.n_base_blocks;
    const int64_t lo = (int64_t)b * per, hi = min(lo + per, n);
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += kThreads) {
      const double d = (__ldg(A.obs + i) - 1.0) * __ldg(A.isig + i);
      acc = fma(d, d, acc);
    }
    s_sum[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
      if ((int)threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
      __syncthreads();
    }
    if (threadIdx.x == 0) Q.base_part[b] = s_sum[0];
    if (!Q.want_units)
      for (int64_t i = (int64_t)b * kThreads + threadIdx.x; i < A.n_pv; i += (int64_t)Q.n_base_blocks * kThreads) A.chi2[i] = 0.0;
  }
  if (!Q.want_units || Q.n_base_blocks == 0) return;
  // ---- fused likelihood in front of the epoch kernel: the last block to get here leaves the out-of-transit baseline (the
  // partials in a fixed order) in chi2[]; bad rows are NaN
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    s_last = (atomicAdd(A.sched + kW_PrepDone, 1ULL) == (unsigned long long)(Q.n_blocks - 1)) ? 1 : 0;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  double B = 0.0;
  for (int i = 0; i < Q.n_base_blocks; ++i) B += ((volatile double*)Q.base_part)[i];
  for (int pv = threadIdx.x; pv < (int)A.n_pv; pv += kThreads) {
    const int fl = ((volatile int*)&Q.rec[pv].c.flags)[0];
    A.chi2[pv] = (fl & PV_BAD) ? nan64() : B;
  }
  if (threadIdx.x == 0) A.sched[kW_PrepDone] = 0ULL;
}

}  // namespace pt
