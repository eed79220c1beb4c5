// pt_epoch.cuh — the epoch kernel: the hot path (S1-S7, S9) for one passband on ONE SHARED, ASCENDING time axis
// (BASELINE.json configs[1] and configs[3]: a light curve sampled at a fixed cadence, evaluated for a whole population).
//
// On such an axis the exposures that can be in transit are known without looking at the others: parameter vector pv
// transits at the epochs n = n0 .. n0+cnt-1 (prep_kernel), and the exposures inside the conservative window of epoch n,
//     t0 + (n + ex_lo) P  <=  t  <=  t0 + (n + ex_hi) P          (ex_lo, ex_hi: pt_orbit.cuh, widened by the rounding of
//                                                                 this very expression)
// form one index range [lo_n, hi_n) that two searches find (a four-value probe where a uniform cadence predicts the
// answer, galloping + bisection otherwise).  Everything else has flux exactly 1.
//
// Work unit = (row pv, chunk c of C): the epochs [c cnt/C, (c+1) cnt/C) of the row TOGETHER WITH the stretch of the row in
// front of each of them: epoch j owns the exposures [hi_{j-1}, hi_j) — the gap before its window, written as pure 16-byte
// streaming stores (no time loads, no arithmetic), and its window, every exposure of which is evaluated.  hi_{-1} = 0 and
// the last epoch of the row also owns the tail, so the units partition the output exactly and nothing is searched twice.
// (A batch of epochs writes ones over its whole stretch, windows included, and overwrites the windows — same warp, ordered by
// a __syncwarp — instead of one short run per gap: 4 % more bytes, a tenth of the fill instructions; PT_FILL_THROUGH.  In the
// interpolated model the stretch goes out piece by piece, each in front of the round of the evaluation that needs it.)
// Units are dealt to the blocks of one persistent grid from a ticket counter, rows in the order prep_kernel left (by k̂
// for the table: neighbouring tickets read neighbouring table rows; heaviest first for the exact model).
//
//   interpolated model (MODE 1): a block of 16 warps per unit.  The block first STAGES THE TABLE IN SHARED MEMORY: the two
//     k-rows that bracket k̂ are read once, coalesced, over the z-range the row can reach, blended in k and combined with
//     the limb-darkening coefficients into ONE fp64 value per z-node, G[j] = Σ_f coef_f (T[ik][j][f] + fk (T[ik+1][j][f] -
//     T[ik][j][f])); a sample is then 1 - (G[iz] + fz (G[iz+1] - G[iz])) from shared memory — the same bilinear rule
//     (S§8(c)-2 step 8) with the k-blend done first.  No per-sample gather from L2 is left.
//   exact model (MODE 0): a block is a single autonomous warp (no barrier cost, 24 of them per SM).
//   Inside a unit every warp takes an equal run of consecutive epochs, in as few batches of up to 31 epochs as possible
//   (lane = epoch: probes, searches), fills the gaps, and packs the
//   in-window exposures of the batch (times n_ss subsamples) densely over the lanes in rounds of 32: pinned subsample time
//   and phase fold (H1, H2), orbit, in-transit test, basis functions or table lookup, limb-darkening combine;
//   n_ss > 1: segmented warp-shuffle sum in 64-bit fixed point (order-independent: bit-reproducible), carried across
//   rounds in a small ring of accumulators.
//   A row that is always in the window, or whose epochs are denser than one per eight exposures, is cut into chunks of
//   kChunkLen exposures instead of epochs (every exposure evaluated); a row that never transits is all fill; a bad row NaN.
//
// If prep_kernel finds the axis not ascending (or not finite), every row is cut into chunks: exact for any order of the
// times, only slow.
#pragma once
#include "pt_flux.cuh"

namespace pt {

#ifndef PT_FILL_THROUGH
#define PT_FILL_THROUGH 1     // 1: a batch writes ones over its whole stretch and overwrites the windows (0.737 -> 0.704 ms on configs[3]);
                               // 0: only the gaps are filled, every element is written exactly once
#endif
#ifndef PT_FILL_ROUNDS_INTERP
#define PT_FILL_ROUNDS_INTERP 1   // the stretch of a batch is written piece by piece in front of the rounds of its evaluation
                                  // (configs[3]: 0.80 ms with the whole stretch first, 0.67 ms piece by piece)
#endif
#ifndef PT_FILL_ROUNDS_EXACT
#define PT_FILL_ROUNDS_EXACT 0     // exact model: the whole stretch in front of the rounds (configs[1] 0.083 vs 0.079 ms)
#endif
#ifndef PT_EPOCH_DEPTH
#define PT_EPOCH_DEPTH 3          // rounds of time loads in flight ahead of the evaluation, interpolated model (1 / 2 / 3: 0.674 / 0.673 / 0.670 ms)
#endif
#ifndef PT_EPOCH_FILL_AHEAD
#define PT_EPOCH_FILL_AHEAD 1      // pieces of ones written ahead of the round being evaluated (1 / 2 / 3 / 4: 0.675 / 0.700 / 0.716 / 0.763 ms:
                                   // longer bursts of stores from one warp hold up everybody's loads)
#endif
#ifndef PT_EPOCH_WARPS
#define PT_EPOCH_WARPS 24   // single-warp blocks per SM of the exact model's epoch kernel
#endif
constexpr int kAccRing = 64;        // supersample accumulators in flight per warp (exposures are finished in order)
constexpr int kBcumMax = 4096;      // rows of a launch the epoch kernel takes (= the slot's record capacity)
constexpr int kOffTable = 256;      // subsample offsets tabulated per block (n_ss up to this; computed on the fly above)

struct EpochWarp {
  long long acc[kAccRing];
};

// flux = v for exposures [a, b) of a row (any parity): aligned pairs as 16-byte (fp32: 8-byte) streaming stores when the
// row allows it (V2), single elements at odd ends.
template <bool V2, typename OutT>
__device__ __forceinline__ void fill_span(OutT* __restrict__ row, uint32_t a, uint32_t b, OutT val) {
  if constexpr (kIsChi2<OutT>) {
    return;
  } else {
    if (a >= b) return;
    const uint32_t lane = threadIdx.x & 31;
    if (V2) {
      if (a & 1u) { if (lane == 0) PT_ST(row + a, val); ++a; }
      if ((b & 1u) && b > a) { --b; if (lane == 0) PT_ST(row + b, val); }
      typedef typename Vec2<OutT>::type V2T;
      V2T v; v.x = val; v.y = val;
      const uint32_t n = b - a;                     // even
      V2T* p = (V2T*)(row + a) + lane;
#pragma unroll 4
      for (uint32_t i = n >> 6; i > 0; --i) { PT_ST(p, v); p += 32; }
      if (2u * lane < (n & 63u)) PT_ST(p, v);
    } else {
      OutT* p = row + a + lane;
      const uint32_t n = b - a;
#pragma unroll 4
      for (uint32_t i = n >> 5; i > 0; --i) { PT_ST(p, val); p += 32; }
      if (lane < (n & 31u)) PT_ST(p, val);
    }
  }
}

// Index range [lo, hi) of the exposures t[0..n) inside the window of epoch `en` of the parameter vector with constants c:
// first index with t >= tlo, first index with t > thi.  The same expression (and the same exact searches) is evaluated by
// fill tiles on a slice of the axis and by eval batches on the whole axis: on an ascending axis the slice result is the
// whole-axis result clipped to the slice.  Split in two so that the eight probe loads of the next batch of epochs are in
// flight while the current one is being filled: under a saturated write stream a load takes microseconds.
// Every load of the time axis carries the L2 evict_last policy `pol`: gigabytes of write-once flux pass through the same L2.
struct Probe {
  double tlo, thi;
  int sl, sh;
  double vl[4], vh[4];
};
__device__ __forceinline__ void probe_issue(const PvConst& c, double en, const double* __restrict__ t, int n, double T0, double idt,
                                            unsigned long long pol, Probe& q) {
  const double padn = 0x1p-49 * (fabs(en) + fabs(c.t0 * c.invP) + 1.0);
  q.tlo = fma(c.P, en + (c.ex_lo - padn), c.t0);
  q.thi = fma(c.P, en + (c.ex_hi + padn), c.t0);
  q.sl = probe_start(q.tlo, n, T0, idt); q.sh = probe_start(q.thi, n, T0, idt);
#pragma unroll
  for (int i = 0; i < 4; ++i) { q.vl[i] = ldg_keep(t + q.sl + i, pol); q.vh[i] = ldg_keep(t + q.sh + i, pol); }   // 8 independent loads
}
__device__ __forceinline__ void probe_finish(const Probe& q, const double* __restrict__ t, int n, int* lo, int* hi) {
  *lo = search_sorted<false>(t, n, q.tlo, q.sl, q.vl);
  *hi = search_sorted<true>(t, n, q.thi, q.sh, q.vh);
}

// Result of one finished exposure e of row `row` (single passband): the flux store, or the chi2 correction (pt_flux.cuh: emit).
template <typename OutT>
__device__ __forceinline__ void emit1(const FluxArgs& A, OutT* __restrict__ row, uint32_t e, double dec, double& chi) {
  if constexpr (kIsChi2<OutT>) {
    const double o = __ldg(A.obs + e), w = __ldg(A.isig + e);
    chi = fma(dec * w * w, fma(2.0, o - 1.0, dec), chi);
  } else {
    PT_ST(row + e, (OutT)(1.0 - dec));
  }
}

// Combined decrement c0 λe + c1 λd* + c2 ηd from the closed forms, out of line: the interpolated kernel only needs it for a
// parameter vector whose k̂ is off the table, and must not pay its registers everywhere else.
__device__ __noinline__ double ma_dec_noinline(double khat, double z, double c0, double c1, double c2) {
  const Basis b = ma_basis(khat, z);
  return fma(c2, b.ed, fma(c1, b.ld, c0 * b.le));
}

// Stage the table for one parameter vector: G[j] = Σ_f coef_f (T[ik][j][f] + fk (T[ik+1][j][f] - T[ik][j][f])) for the z-nodes
// the row can reach (whole block, coalesced loads with the L2 evict_last policy).
template <int NT>
__device__ __forceinline__ void stage_table(const FluxArgs& A, const PvRec& r, double* __restrict__ G, unsigned long long pol) {
  const double khat = r.c.khat;
  const double zmin = (r.c.flags & PV_CIRCULAR) ? r.c.a * fabs(r.c.cosi) : 0.0;
  const int jlo = max(0, (int)floor(zmin * A.inv_dz) - 1);
  const int jhi = min(A.n_z - 1, (int)floor((1.0 + khat) * A.inv_dz) + 2);
  const double c0 = r.coef[0], c1 = r.coef[1], c2 = r.coef[2], fk = r.fk;
  const size_t r0 = (size_t)r.ik * A.n_z;
  if (A.tb_dtype == PT_F32 && A.n_fn == 4 && (reinterpret_cast<uintptr_t>(A.tb) & 15) == 0) {
    const float* t0 = (const float*)A.tb + r0 * 4;
    const float* t1 = t0 + (size_t)A.n_z * 4;
#pragma unroll 4
    for (int j = jlo + (int)threadIdx.x; j <= jhi; j += NT) {
      const float4 a = ldg_keep4(t0 + (size_t)j * 4, pol), b = ldg_keep4(t1 + (size_t)j * 4, pol);
      const double v0 = fma(fk, (double)b.x - (double)a.x, (double)a.x);
      const double v1 = fma(fk, (double)b.y - (double)a.y, (double)a.y);
      const double v2 = fma(fk, (double)b.z - (double)a.z, (double)a.z);
      G[j] = fma(c2, v2, fma(c1, v1, c0 * v0));
    }
  } else {
    const int nf = A.n_fn;
#pragma unroll 2
    for (int j = jlo + (int)threadIdx.x; j <= jhi; j += NT) {
      double a[3], b[3];
      if (A.tb_dtype == PT_F64) {
        const double* t0 = (const double*)A.tb + (r0 + j) * nf;
        const double* t1 = t0 + (size_t)A.n_z * nf;
#pragma unroll
        for (int f = 0; f < 3; ++f) { a[f] = ldg_keep(t0 + f, pol); b[f] = ldg_keep(t1 + f, pol); }
      } else {
        const float* t0 = (const float*)A.tb + (r0 + j) * nf;
        const float* t1 = t0 + (size_t)A.n_z * nf;
#pragma unroll
        for (int f = 0; f < 3; ++f) { a[f] = (double)ldg_keep(t0 + f, pol); b[f] = (double)ldg_keep(t1 + f, pol); }
      }
      const double v0 = fma(fk, b[0] - a[0], a[0]), v1 = fma(fk, b[1] - a[1], a[1]), v2 = fma(fk, b[2] - a[2], a[2]);
      G[j] = fma(c2, v2, fma(c1, v1, c0 * v0));
    }
  }
}

// ---------------------------------------------------------------------------------------------------- the kernel
// MODE 0: exact (NT = 32: a block is one autonomous warp).  MODE 1: interpolated (NT = 512; exact basis functions for a
// parameter vector whose k̂ is off the table).  V2: rows allow aligned pair stores.  SS1: n_ss == 1.
template <int MODE, int NT, bool V2, bool SS1, typename OutT>
__global__ void __launch_bounds__(NT, (NT == 32 ? PT_EPOCH_WARPS : 2)) epoch_kernel(const __grid_constant__ FluxArgs A) {
  extern __shared__ double s_G[];                       // MODE 1: the staged table of the current unit, n_z doubles
  __shared__ EpochWarp s_w[SS1 ? 1 : NT / 32];
  __shared__ double s_off[SS1 ? 1 : kOffTable];
  __shared__ PvRec s_rec;
  __shared__ unsigned long long s_tk;
  constexpr int nwp = NT / 32;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  EpochWarp& W = s_w[SS1 ? 0 : warp];
  const int n_ss = SS1 ? 1 : A.n_ss;
  if (!SS1) {   // before the wait: overlaps prep_kernel
    for (int i = tid; i < kOffTable && i < n_ss; i += NT) s_off[i] = subsample_offset(i, n_ss, A.t_exp);
    for (int i = lane; i < kAccRing; i += 32) W.acc[i] = 0;
    __syncthreads();
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");   // prep_kernel's slot (records, units, order, axis flag) is complete
  // an axis that is not ascending (or not finite) has no index ranges: every row is then cut into chunks and every exposure
  // evaluated (slow, but exact for any order of the times: an exposure outside the transit evaluates to flux 1)
  const bool unsorted = *((volatile const unsigned long long*)(A.sched + kW_Flags)) & kSlotUnsorted;
  const int C = A.unit_chunks;
  const unsigned long long n_units = (unsigned long long)A.n_pv * (unsigned long long)C;
  const int n_t = (int)A.n_t;
  const double T_first = __ldg(A.times), T_last = __ldg(A.times + (n_t - 1));
  const double idt_axis = (T_last > T_first) ? (double)(n_t - 1) / (T_last - T_first) : 0.0;
  const int G = n_ss < 32 ? n_ss : 32;
  const uint32_t ss_magic = SS1 ? 0u : (uint32_t)((65536 + G - 1) / G);   // floor(v / n_ss) = v * magic >> 16 for v < 64, n_ss < 32
  const unsigned long long pol = l2_keep_policy();

  unsigned long long ticket = blockIdx.x;
  while (ticket < n_units) {
    if (tid == 0) { s_tk = atomicAdd(A.sched + kW_Ticket, 1ULL); }   // the next ticket: its latency hides behind this unit
    const int64_t j = (int64_t)(ticket / (unsigned long long)C);
    const int c = (int)(ticket - (unsigned long long)j * C);
    const int64_t pv = A.order ? (int64_t)__ldg(A.order + j) : j;
    uint32_t ucnt = __ldg(A.ucnt + pv);
    if (unsorted && ucnt != 0u) ucnt = kUnitChunks | (uint32_t)((n_t + kChunkLen - 1) / kChunkLen);
    const double un0 = __ldg(A.un0 + pv);
    {
      const double* src = reinterpret_cast<const double*>(A.pvcache + pv);
      double* dst = reinterpret_cast<double*>(&s_rec);
      for (int i = tid; i < (int)(sizeof(PvRec) / sizeof(double)); i += NT) dst[i] = __ldg(src + i);
    }
    __syncthreads();
    const unsigned long long next_ticket = (unsigned long long)gridDim.x + s_tk;
    const PvRec& r = s_rec;
    const int flags = r.c.flags;
    const uint32_t cnt = ucnt & ~kUnitChunks;
    const bool chunk_units = ucnt & kUnitChunks;
    OutT* __restrict__ row = kIsChi2<OutT> ? nullptr : (OutT*)A.flux + pv * A.flux_pv_stride + A.flux_off;
    if ((flags & PV_BAD) || cnt == 0u) {
      // nothing to evaluate: this unit's share of the row is NaN (bad parameters) or 1 (no transit on the axis)
      if constexpr (!kIsChi2<OutT>) {
        const OutT val = (flags & PV_BAD) ? (OutT)nan64() : (OutT)1.0;
        const int64_t s0 = ((int64_t)c * n_t / C) & ~(int64_t)1, s1 = (c == C - 1) ? (int64_t)n_t : (((int64_t)(c + 1) * n_t / C) & ~(int64_t)1);
        const int64_t per = (((s1 - s0) + nwp - 1) / nwp + 1) & ~(int64_t)1;
        const int64_t a = min(s0 + (int64_t)warp * per, s1), b = min(a + per, s1);
        fill_span<V2, OutT>(row, (uint32_t)a, (uint32_t)b, val);
      }
    } else {
      const uint32_t E0 = (uint32_t)((unsigned long long)c * cnt / (unsigned long long)C);
      const uint32_t E1 = (uint32_t)((unsigned long long)(c + 1) * cnt / (unsigned long long)C);
      const bool use_tb = MODE == 1 && r.use_table;
      // batches of Be <= 31 epochs (lane = epoch; one more lane looks at the epoch in front of the batch).
      // Every warp takes an equal run of consecutive epochs — its stores walk through one contiguous piece of the row — cut
      // into as few batches as possible: a batch costs an exposed load (its probes; the times of a window then hit L1).
      const uint32_t nE = E1 - E0;
      const uint32_t nEw = (nE + nwp - 1u) / nwp;
      const uint32_t wE0 = min(E0 + (uint32_t)warp * nEw, E1), wE1 = min(wE0 + nEw, E1);
      const uint32_t nS = (nEw + 30u) / 31u;
      const uint32_t Be = nS ? (nEw + nS - 1u) / nS : 1u;
      if (MODE == 1 && use_tb && E1 > E0) {
        stage_table<NT>(A, r, s_G, pol);
        __syncthreads();
      }
      const double khat = r.c.khat;
      const bool slow_div = flags & PV_SLOWDIV;
      const double c0 = r.coef[0], c1 = r.coef[1], c2 = r.coef[2];
      double chi = 0.0;
      for (uint32_t first = wE0; first < wE1; first += Be) {
        const int m = (int)min(Be, wE1 - first);
        // lane i < m: epoch first + i; lane m: the epoch in front of the batch (only its hi is used)
        int lo = 0, hi = 0;
        {
          const bool mine = lane < m, prev = (lane == m) && first > 0u;
          if (mine || prev) {
            const uint32_t ei = mine ? first + (uint32_t)lane : first - 1u;
            if (chunk_units) {
              lo = (int)ei * kChunkLen;
              hi = min(lo + kChunkLen, n_t);
            } else {
              Probe q;
              probe_issue(r.c, un0 + (double)ei, A.times, n_t, T_first, idt_axis, pol, q);
              probe_finish(q, A.times, n_t, &lo, &hi);
            }
          }
        }
        // gaps: [hi of the epoch in front, lo)
        int phi = __shfl_up_sync(0xffffffffu, hi, 1);
        const int phi0 = __shfl_sync(0xffffffffu, hi, m);
        if (lane == 0) phi = phi0;
#if PT_FILL_THROUGH
        // ones over the whole stretch of the batch, windows included; the evaluation overwrites the windows (same warp, ordered
        // by a __syncwarp): a few per cent more bytes, a tenth of the fill instructions.  The stretch is written piece by piece
        // in front of the rounds of the evaluation (`fill_to`), each piece ending with the window of the round's last sample.
        const int bend = (first + (uint32_t)m == cnt) ? n_t : __shfl_sync(0xffffffffu, hi, m - 1);
        int filled = phi0;
        constexpr bool kPerRound = (MODE == 1) ? (PT_FILL_ROUNDS_INTERP != 0) : (PT_FILL_ROUNDS_EXACT != 0);
        auto fill_to = [&](int need) {
          if constexpr (!kIsChi2<OutT>) {
            if (need > filled) {
              fill_span<V2, OutT>(row, (uint32_t)filled, (uint32_t)need, (OutT)1.0);
              filled = need;
              __syncwarp();
            }
          }
        };
        if (!kPerRound) fill_to(bend);
        (void)phi;
#else
        for (int i = 0; i < m; ++i) {
          const int a = __shfl_sync(0xffffffffu, phi, i), b = __shfl_sync(0xffffffffu, lo, i);
          PT_CHECK(a >= 0 && b <= n_t);                      // a > b never happens (the windows are disjoint) and would be a no-op
          if constexpr (!kIsChi2<OutT>) fill_span<V2, OutT>(row, (uint32_t)a, (uint32_t)b, (OutT)1.0);
        }
        if constexpr (!kIsChi2<OutT>) {
          if (first + (uint32_t)m == cnt) fill_span<V2, OutT>(row, (uint32_t)__shfl_sync(0xffffffffu, hi, m - 1), (uint32_t)n_t, (OutT)1.0);   // tail of the row
        }
        const int bend = 0;
        auto fill_to = [&](int) {};
        (void)bend;
#endif
        // in-window exposures of the batch, packed over the lanes
        const int rcnt = lane < m ? hi - lo : 0;
        int cum = rcnt;                                   // inclusive scan of the range lengths
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int v = __shfl_up_sync(0xffffffffu, cum, o);
          if (lane >= o) cum += v;
        }
        const int n_exp = __shfl_sync(0xffffffffu, cum, 31);
        const int ebase = lo - (cum - rcnt);              // exposure x of the batch, if it lies in this lane's range, is e = ebase + x
        auto range_of = [&](int x) -> int {               // the range i with cum[i-1] <= x < cum[i]
          int i = 0;
#pragma unroll
          for (int step = 16; step > 0; step >>= 1) {
            const int cv = __shfl_sync(0xffffffffu, cum, i + step - 1);
            if (cv <= x) i += step;
          }
          return i;
        };
        auto exposure_of = [&](int x) -> int { return __shfl_sync(0xffffffffu, ebase, range_of(x)) + x; };
        // end of the stretch that must hold its ones before the samples up to x_last (uniform) are stored
        auto stretch_end = [&](int x_last, bool last_round) -> int {
          if (!kPerRound) return bend;
          return last_round ? bend : __shfl_sync(0xffffffffu, hi, range_of(x_last));
        };
        auto decrement = [&](double zs) -> double {       // combined decrement of an in-transit sample
          if (MODE == 1 && use_tb) {
            const double rz = zs * A.inv_dz;
            int iz = (int)floor(rz);
            iz = min(max(iz, 0), A.n_z - 2);
            const double g0 = s_G[iz], g1 = s_G[iz + 1];
            return fma(rz - (double)iz, g1 - g0, g0);
          } else if (MODE == 1) {
            return ma_dec_noinline(khat, zs, c0, c1, c2);
          } else {
            if constexpr (kF32Capable<OutT>) {
              if (r.f.use) return (double)ma_dec32(r.f, (float)zs);
            }
            const Basis b = ma_basis(khat, zs);
            return fma(c2, b.ed, fma(c1, b.ld, c0 * b.le));
          }
        };
        if (SS1) {
          const int R = (n_exp + 31) >> 5;
          auto fetch = [&](int q, int& e, double& t, bool& act) {
            const int x = q * 32 + lane;
            act = x < n_exp;
            e = exposure_of(act ? x : n_exp - 1);
            PT_CHECK(e >= 0 && e < n_t);
            t = act ? ldg_keep(A.times + e, pol) : 0.0;
            if constexpr (kIsChi2<OutT>) {     // the observation this exposure will be compared with: towards L1 now
              if (act) {
                asm volatile("prefetch.global.L1 [%0];" ::"l"(A.obs + e));
                asm volatile("prefetch.global.L1 [%0];" ::"l"(A.isig + e));
              }
            }
          };
          // the times of the next kDepth rounds are in flight during this one (under a saturated store stream a load that
          // misses L1 takes microseconds; most of a window's times were brought into L1 by its probes)
          constexpr int kDepth = (MODE == 1) ? PT_EPOCH_DEPTH : 1;
          int eq[kDepth]; double tq[kDepth]; bool aq[kDepth];
#pragma unroll
          for (int d = 0; d < kDepth; ++d) {
            eq[d] = 0; tq[d] = 0.0; aq[d] = false;
            if (d < R) fetch(d, eq[d], tq[d], aq[d]);
          }
          for (int q = 0; q < R; ++q) {
            const int e = eq[0]; const double t = tq[0]; const bool act = aq[0];
#pragma unroll
            for (int d = 0; d + 1 < kDepth; ++d) { eq[d] = eq[d + 1]; tq[d] = tq[d + 1]; aq[d] = aq[d + 1]; }
            if (q + kDepth < R) fetch(q + kDepth, eq[kDepth - 1], tq[kDepth - 1], aq[kDepth - 1]);
#if PT_FILL_THROUGH
            fill_to(stretch_end(min((q + PT_EPOCH_FILL_AHEAD) * 32 - 1, n_exp - 1), q + PT_EPOCH_FILL_AHEAD >= R));
#endif
            if (act) {
              bool in;
              const double zs = sample_z<OutT>(r, fold_phase(t, r.c.t0, r.c.P, r.c.invP, slow_div), in);
              const double dec = in ? decrement(zs) : 0.0;
              if (in || !kIsChi2<OutT>) emit1<OutT>(A, row, (uint32_t)e, dec, chi);
            }
          }
          fill_to(bend);                                   // a batch without a single in-window exposure
        } else {
          // supersampled: items y = x n_ss + s, 32 per round; segmented fixed-point sum per exposure, carried in W.acc
          const long long n_items = (long long)n_exp * n_ss;
          for (long long y0 = 0; y0 < n_items; y0 += 32) {
            const int x0 = (n_items < 0x7fffffffLL) ? (int)((uint32_t)y0 / (uint32_t)n_ss) : (int)(y0 / n_ss);
            const int v = (int)(y0 - (long long)x0 * n_ss) + lane;          // < n_ss + 32
            const int dx = (n_ss >= 32) ? (v >= n_ss ? 1 : 0) : (int)(((uint32_t)v * ss_magic) >> 16);
            const int x = x0 + dx, sub = v - dx * n_ss;
            const bool act = x < n_exp;
            const int e = exposure_of(act ? x : n_exp - 1);
            PT_CHECK(e >= 0 && e < n_t && sub >= 0 && sub < n_ss);
#if PT_FILL_THROUGH
            {
              const long long yl = y0 + 31;
              const int xl = (n_items < 0x7fffffffLL) ? (int)((uint32_t)yl / (uint32_t)n_ss) : (int)(yl / n_ss);
              fill_to(stretch_end(min(xl, n_exp - 1), y0 + 32 >= n_items));
            }
#endif
            long long fx = 0;
            if (act) {
              const double t = ldg_keep(A.times + e, pol);
              const double ts = __dadd_rn(t, sub < kOffTable ? s_off[sub] : subsample_offset(sub, n_ss, A.t_exp));
              bool in;
              const double zs = sample_z<OutT>(r, fold_phase(ts, r.c.t0, r.c.P, r.c.invP, slow_div), in);
              if (in) fx = __double2ll_rn(decrement(zs) * r.acc_scale);
            }
            const int sid = act ? x : -1 - lane;
            for (int o = 1; o < G; o <<= 1) {
              const int so = __shfl_up_sync(0xffffffffu, sid, o);
              const long long tv = __shfl_up_sync(0xffffffffu, fx, o);
              if (lane >= o && so == sid) fx += tv;
            }
            const int snext = __shfl_down_sync(0xffffffffu, sid, 1);
            if (act && (lane == 31 || snext != sid)) {       // last subsample of this exposure in this round
              const long long sum = W.acc[x & (kAccRing - 1)] + fx;
              PT_CHECK(sub == n_ss - 1 || lane == 31 || snext < 0 || snext == x + 1);   // an unfinished exposure only at the end of a round
              if (sub == n_ss - 1) {
                W.acc[x & (kAccRing - 1)] = 0;
                emit1<OutT>(A, row, (uint32_t)e, (double)sum * r.acc_inv, chi);
              } else {
                W.acc[x & (kAccRing - 1)] = sum;
              }
            }
            __syncwarp();
          }
          fill_to(bend);
        }
      }
      if constexpr (kIsChi2<OutT>) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) chi += __shfl_xor_sync(0xffffffffu, chi, o);
        if (lane == 0 && chi != 0.0) atomicAdd(A.chi2 + pv, chi);
      }
    }
    __syncthreads();                                      // the record and the staged table are free again
    ticket = next_ticket;
  }
  if (tid == 0) {
    const unsigned long long done = atomicAdd(A.sched + kW_Done, 1ULL);
    if (done == (unsigned long long)gridDim.x - 1ULL) {   // every block has taken its last ticket: nobody reads the slot any more
      for (int i = 0; i < kSchedHead; ++i) A.sched[i] = 0ULL;
    }
  }
}

}  // namespace pt
