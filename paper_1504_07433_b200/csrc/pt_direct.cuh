// pt_direct.cuh — the direct kernel: exact model, one passband, no supersampling, per-row times (BASELINE.json configs[4]:
// per-row times drawn around the transit; the `dense` bench workload) — the kernel of the fp32-arithmetic variant there.
//
// A tile (row, run of tile_len exposures; tickets from the scheduler slot, records from prep_kernel when a row has more
// than one tile) is worked through in passes of kDirectSub exposures:
//   pass 1  16-byte time loads, kDirectUnroll of them in flight per lane; the cheap phase-window test; ones for the
//           exposures outside the window (pairs: one 16-byte / 8-byte store); the exposures inside — in exposure order — are
//           appended to a list in shared memory (ballot + popc).  A round with nothing inside the window costs one vote.
//   pass 2  the list 32 at a time, every lane busy: time (an L1 hit), pinned phase fold, orbit, case split and basis
//           functions, combine, store.  What does not fill a round waits for the next pass of the tile.
// The kernel is short on purpose: the general kernel's code (pt_flux.cuh) is ~90 KB of SASS through which its autonomous
// warps wander independently, and the profiler showed 15 % (fp64) to 44 % (fp32 variant inline) of its stall samples on
// instruction fetch.  Here there is ONE copy of the evaluation (pass 2), and the fp32 variant (SEL 3) contains the fp32
// arithmetic only; the few rows that keep fp64 arithmetic (PvRec::f.use == 0) call one out-of-line function per exposure.
// History: both arithmetics inline in the general kernel 0.46 ms on `dense`; a loop in which every lane
// evaluates its own two exposures 0.375 ms with two inlined copies of the evaluation, 0.322 ms with one rolled copy,
// 0.263 ms with the records from prep_kernel — but 0.19 ms on a sparse per-row population (3 % in the window) where this
// form takes 0.087 ms (and 0.270 ms on `dense`).  With fp64 arithmetic (SEL 0) it ties with the general kernel on both
// (0.457 / 0.105 ms against 0.460 / 0.102 ms), so the library keeps fp64 calls on the general kernel (PT_DIRECT_F64).
// Persistent grid of autonomous warps.
#pragma once
#include "pt_flux.cuh"

namespace pt {

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

constexpr int kDirectUnroll = 4;                 // 16-byte time loads in flight per lane in pass 1
constexpr int kDirectSub = 1024;                 // exposures looked at per pass (their in-window ones fit the list)
constexpr int kDirectList = kDirectSub + 32;     // + what the previous pass left over

// SEL 0: fp64 arithmetic.  SEL 3: fp32 arithmetic, the rows that keep fp64 arithmetic out of line.
// A tile is worked through in passes of kDirectSub exposures.  Pass 1: 16-byte time loads, the cheap phase-window test, ones
// for the exposures outside the window (pairs: 16-byte stores), the others — in exposure order — appended to a list in
// shared memory.  Pass 2: the list 32 at a time, every lane busy: time (an L1 hit), pinned phase fold, orbit, basis
// functions, combine, store.  What does not fill a round waits for the next pass of the tile.
template <int V, typename OutT, int SEL>
__global__ void __launch_bounds__(kThreads, PT_DIRECT_BLOCKS) direct_kernel(const __grid_constant__ FluxArgs A) {
  __shared__ WarpState s_ws[kWarpsPerBlock];
  __shared__ uint16_t s_list[kWarpsPerBlock][kDirectList];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  WarpState& ws = s_ws[warp];
  uint16_t* __restrict__ list = s_list[warp];
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
    tile_setup<0, true, OutT>(A, ws, 0, pv, chunk, (pv == last_pv) ? 0 : -1);
    last_pv = pv;
    const PvRec& r = ws.pv[0];
    const int n_e = (int)min((int64_t)A.tile_len, A.n_t - (int64_t)chunk * A.tile_len);
    const double* __restrict__ tb = r.tb;
    OutT* __restrict__ ob = (OutT*)r.ob;
    const int flags = r.c.flags;
    if (flags & PV_BAD) {
      for (int e = lane; e < n_e; e += 32) ob[e] = (OutT)nan64();
    } else {
      const double invP = r.c.invP, w_c0 = r.w_c0, w_half = r.w_half;
      const bool slow_div = flags & PV_SLOWDIV;
      // flux of one exposure inside the window
      auto flux_of = [&](double t) -> OutT {
        const double ph = fold_phase(t, r.c.t0, r.c.P, invP, slow_div);
        if constexpr (SEL == 3) {
          if (!r.f.use) return (OutT)flux64_noinline(r, ph);
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
      int n_list = 0;
      for (int s0 = 0; s0 < n_e; s0 += kDirectSub) {
        const int s1 = min(s0 + kDirectSub, n_e);
        // ---- pass 1
        if (V == 2) {
          typedef typename Vec2<OutT>::type V2T;
          V2T ones; ones.x = (OutT)1.0; ones.y = (OutT)1.0;
          for (int e0 = s0; e0 < s1; e0 += 64 * kDirectUnroll) {
            double2 tv[kDirectUnroll];
#pragma unroll
            for (int u = 0; u < kDirectUnroll; ++u) {                 // kDirectUnroll 16-byte loads in flight per lane
              const int e = e0 + 64 * u + 2 * lane;
              tv[u] = (e + 1 < s1) ? __ldg((const double2*)(tb + e)) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int u = 0; u < kDirectUnroll; ++u) {
              const int e = e0 + 64 * u + 2 * lane;
              bool in_x = false, in_y = false;
              if (e + 1 < s1) {
                in_x = in_window2(tv[u].x, invP, w_c0, w_half);
                in_y = in_window2(tv[u].y, invP, w_c0, w_half);
                if (!(in_x && in_y)) PT_ST((V2T*)(ob + e), ones);     // the one inside the window is overwritten in pass 2
              } else if (e < s1) {                                   // odd tail of the tile
                in_x = in_window2(__ldg(tb + e), invP, w_c0, w_half);
                if (!in_x) PT_ST(ob + e, (OutT)1.0);
              }
              if (__any_sync(0xffffffffu, in_x || in_y)) {            // else nothing of this round can be in transit
                const unsigned bx = __ballot_sync(0xffffffffu, in_x), by = __ballot_sync(0xffffffffu, in_y);
                const int pos = n_list + __popc(bx & lt) + __popc(by & lt);
                if (in_x) list[pos] = (uint16_t)e;
                if (in_y) list[pos + (in_x ? 1 : 0)] = (uint16_t)(e + 1);
                n_list += __popc(bx) + __popc(by);
              }
            }
          }
        } else {
          for (int e0 = s0; e0 < s1; e0 += 32) {
            const int e = e0 + lane;
            bool in_x = false;
            if (e < s1) {
              in_x = in_window2(__ldg(tb + e), invP, w_c0, w_half);
              if (!in_x) PT_ST(ob + e, (OutT)1.0);
            }
            const unsigned bx = __ballot_sync(0xffffffffu, in_x);
            if (in_x) list[n_list + __popc(bx & lt)] = (uint16_t)e;
            n_list += __popc(bx);
          }
        }
        PT_CHECK(n_list <= kDirectList);
        __syncwarp();
        // ---- pass 2: full rounds; everything at the end of the tile
        const bool last = s1 == n_e;
        int done = 0;
        while (n_list - done >= 32 || (last && done < n_list)) {
          const int i = done + lane;
          if (i < n_list) {
            const int e = list[i];
            PT_ST(ob + e, flux_of(__ldg(tb + e)));
          }
          done += 32;
        }
        __syncwarp();
        const int rem = n_list - done;        // < 32 exposures wait for the next pass
        if (rem > 0) {
          const uint16_t v = lane < rem ? list[done + lane] : (uint16_t)0;
          __syncwarp();
          if (lane < rem) list[lane] = v;
          __syncwarp();
        }
        n_list = rem > 0 ? rem : 0;
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
