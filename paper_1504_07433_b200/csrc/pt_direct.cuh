// pt_direct.cuh — the direct kernel: exact model, one passband, no supersampling, where most exposures ARE in or near a
// transit (BASELINE.json configs[4]: per-row times drawn around the transit; the `dense` bench workload).
//
// Nothing is gained there by separating the exposures that can be in transit from those that cannot (the general kernel's
// queues, pt_flux.cuh) or by looking for epochs (pt_epoch.cuh): every lane simply evaluates its own exposures — 16-byte
// time load, cheap phase-window test (an exposure outside the window is 1 without the orbit), pinned phase fold, orbit,
// case split and basis functions, combine, 16-byte flux store.  The kernel is one short loop, and that is its point: the
// general kernel's code is ~90 KB of SASS through which its autonomous warps wander independently, and the profiler shows
// 15 % (fp64) to 44 % (fp32 variant) of the stall samples on instruction fetch; this loop fits the instruction caches.
// For the same reason the loop of the fp32 variant (SEL 3) contains the fp32 arithmetic only; the few rows that keep fp64
// arithmetic (PvRec::f.use == 0) call one out-of-line function per exposure.  (Measured alternatives: both arithmetics
// inline in the general kernel 0.46 ms on `dense`; two launches, fp32 rows then fp64 rows (SEL 1, SEL 2), 0.41 ms — the 3 %
// of fp64 rows alone take 0.11 ms because a handful of warps run them with nothing to hide their latency; SEL 3: see
// DESIGN.md.  With fp64 output the general kernel is the faster one — 0.51 against 0.57 ms, its queues keep the lanes
// fuller — so SEL 0 is not instantiated by the library.)
// Persistent grid of autonomous warps; tiles (row, run of tile_len exposures) from a ticket counter in the scheduler slot.
#pragma once
#include "pt_flux.cuh"

namespace pt {

#ifndef PT_DIRECT_ONE_COPY
#define PT_DIRECT_ONE_COPY 1
#endif
#ifndef PT_DIRECT_BLOCKS
#define PT_DIRECT_BLOCKS 3
#endif

// fp64 flux of one in-window exposure, out of line: the fp32 kernel needs it for the few rows that keep fp64 arithmetic and
// must not carry its code in the loop.
__device__ __noinline__ double flux64_noinline(const PvRec& r, double ph) {
  const double zs = orbit_z_signed(r.c, ph);
  if (!(zs >= 0.0 && zs < 1.0 + r.c.khat)) return 1.0;
  const Basis b = ma_basis(r.c.khat, zs);
  return 1.0 - fma(r.coef[2], b.ed, fma(r.coef[1], b.ld, r.coef[0] * b.le));
}

template <int V, typename OutT, int SEL>
__global__ void __launch_bounds__(kThreads, PT_DIRECT_BLOCKS) direct_kernel(const __grid_constant__ FluxArgs A) {
  __shared__ WarpState s_ws[kWarpsPerBlock];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  WarpState& ws = s_ws[warp];
  const unsigned long long gw = (unsigned long long)blockIdx.x * kWarpsPerBlock + warp, nw = (unsigned long long)gridDim.x * kWarpsPerBlock;
  const int tpp = A.tiles_per_pv;
  if (A.prep) asm volatile("griddepcontrol.wait;" ::: "memory");   // prep_kernel's records are complete
  int64_t last_pv = -1;
  unsigned long long tile = gw;
  while (tile < (unsigned long long)A.n_tiles) {
    unsigned long long fetched = 0;
    if (lane == 0) fetched = atomicAdd(A.sched + kW_Ticket, 1ULL);   // the next ticket: its latency hides behind this tile
    const int64_t pv = (int64_t)(tile / (unsigned long long)tpp);
    const int chunk = (int)(tile - (unsigned long long)pv * tpp);
    if (SEL == 1 || SEL == 2) {
      // which launch does this row belong to?  The rule of tile_setup from the raw parameters, before the (long) setup
      const double* row = A.params + pv * A.row_stride;
      const bool f32row = A.f32a && f32_ok(__ldg(row + 6), __ldg(row + 7), __ldg(row + 8), __ldg(row + 2), __ldg(row + 4));
      if (f32row != (SEL == 1)) { tile = nw + __shfl_sync(0xffffffffu, fetched, 0); continue; }
    }
    tile_setup<0, true, OutT>(A, ws, 0, pv, chunk, (pv == last_pv) ? 0 : -1);
    last_pv = pv;
    const PvRec& r = ws.pv[0];
    const int n_e = (int)min((int64_t)A.tile_len, A.n_t - (int64_t)chunk * A.tile_len);
    const double* __restrict__ tb = r.tb;
    OutT* __restrict__ ob = (OutT*)r.ob;
    const int flags = r.c.flags;
    const bool mine = (SEL == 0 || SEL == 3) || (SEL == 1 ? r.f.use != 0 : r.f.use == 0);
    if (flags & PV_BAD) {
      if (SEL != 1) for (int e = lane; e < n_e; e += 32) ob[e] = (OutT)nan64();
    } else if (mine) {
      const double invP = r.c.invP, w_c0 = r.w_c0, w_half = r.w_half;
      const bool slow_div = flags & PV_SLOWDIV;
      // flux of one exposure
      auto flux_of = [&](double t) -> OutT {
        if (!in_window2(t, invP, w_c0, w_half)) return (OutT)1.0;
        const double ph = fold_phase(t, r.c.t0, r.c.P, invP, slow_div);
        if constexpr (SEL == 3) {
          if (!r.f.use) return (OutT)flux64_noinline(r, ph);
        }
        if constexpr (SEL == 1 || SEL == 3) {
          const float zf = orbit_z_signed32(r.f, r.c.Mtr, flags & PV_CIRCULAR, ph);
          if (!(zf >= 0.0f && zf < 1.0f + r.f.khat)) return (OutT)1.0;
          return (OutT)(1.0f - ma_dec32(r.f, zf));
        } else {
          const double zs = orbit_z_signed(r.c, ph);
          if (!(zs >= 0.0 && zs < 1.0 + r.c.khat)) return (OutT)1.0;
          const Basis b = ma_basis(r.c.khat, zs);
          return (OutT)(1.0 - fma(r.coef[2], b.ed, fma(r.coef[1], b.ld, r.coef[0] * b.le)));
        }
      };
      if (V == 2) {
        typedef typename Vec2<OutT>::type V2T;
        const int n2 = n_e & ~1;
        V2T ones; ones.x = (OutT)1.0; ones.y = (OutT)1.0;
        double2 nx = make_double2(0.0, 0.0);
        if (2 * lane < n2) nx = __ldg((const double2*)(tb + 2 * lane));
        for (int e0 = 0; e0 < n2; e0 += 64) {
          const int e = e0 + 2 * lane;
          const double2 tv = nx;
          if (e + 64 < n2) nx = __ldg((const double2*)(tb + e + 64));      // the next round's times are in flight
          const bool any = (e < n2) && (in_window2(tv.x, invP, w_c0, w_half) || in_window2(tv.y, invP, w_c0, w_half));
          if (!__any_sync(0xffffffffu, any)) {                             // nothing of this round can be in transit
            if (e < n2) PT_ST((V2T*)(ob + e), ones);
            continue;
          }
          if (e >= n2) continue;
          V2T o;
#if PT_DIRECT_ONE_COPY
          // one copy of the evaluation in the instruction stream, run twice (the loop is kept rolled on purpose)
          double ta = tv.x;
          o.y = (OutT)0;
#pragma unroll 1
          for (int k = 0; k < 2; ++k) {
            const OutT v = flux_of(ta);
            o.x = o.y; o.y = v; ta = tv.y;
          }
#else
          o.x = flux_of(tv.x);
          o.y = flux_of(tv.y);
#endif
          PT_ST((V2T*)(ob + e), o);
        }
        if ((n_e & 1) && lane == 0) PT_ST(ob + n2, flux_of(__ldg(tb + n2)));
      } else {
        for (int e = lane; e < n_e; e += 32) PT_ST(ob + e, flux_of(__ldg(tb + e)));
      }
    }
    tile = nw + __shfl_sync(0xffffffffu, fetched, 0);
  }
  if (lane == 0) {
    const unsigned long long done = atomicAdd(A.sched + kW_Done, 1ULL);
    if (done == nw - 1ULL) {   // every warp has taken its last ticket: nobody reads the slot any more
      for (int i = 0; i < kSchedHead; ++i) A.sched[i] = 0ULL;
    }
  }
}

}  // namespace pt
