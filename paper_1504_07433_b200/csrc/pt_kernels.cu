// pt_kernels.cu — sm_100a kernels and the C ABI of include/pt.h.
//
// The fused flux kernel (whole hot path in one persistent launch) lives in pt_flux.cuh; this file holds the orbit-only
// kernel, the table builder, the FP64 probe and the host side of the C ABI.
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <mutex>

#include "../../include/pt.h"
#include "pt_flux.cuh"
#include "pt_epoch.cuh"
#include "pt_direct.cuh"
#include "pt_gimenez.cuh"

#ifndef PT_REC_MIN_TILES
#define PT_REC_MIN_TILES 2   // tiles per row from which prep_kernel computes the records once (dense 4096 x 4096, six tiles per
                             // row: 0.510 -> 0.458 ms against a threshold of eight)
#endif

namespace pt {

static std::atomic<int64_t> g_launches{0};

// Scheduler slots of the flux kernel: tile counters, flag word, chi2 partials, row order and per-vector records, written by
// prep_kernel / the flux kernel of ONE launch.  The kernel leaves the counters and flags of its slot zeroed when it ends.
// Ordinary launches share the first kSchedRing slots round-robin per device; every launch records an event behind its
// flux kernel, and a slot is given to a new launch only once that event has completed — if all of them are still in
// flight, the new launch's stream is made to wait for the oldest one (cudaStreamWaitEvent: ordering on the device, no host
// synchronisation), so two launches can never share a live slot whatever the number of streams and launches in flight.
// A launch made while its stream is being captured into a CUDA graph gets one of the kSchedGraph slots behind the ring for
// good (the graph replays it; CUDA orders replays of one executable graph behind one another) and makes no CUDA call
// other than the kernel launches; when those slots are used up, capturing returns PT_ERR_CUDA.
constexpr int kSchedRing = 16;
constexpr int kSchedGraph = 8;
constexpr int kSchedSlots = kSchedRing + kSchedGraph;
constexpr int kSchedWords = 1024;   // [0] global ticket, [1] finished warps, [2] flags, [kSchedHead + pv] per-vector tickets;
                                    // the last kBaseBlocks words hold the chi2 baseline partials
constexpr int kPvCacheMax = 4096;   // parameter vectors whose records / row order a slot can hold (prep_kernel)
struct SchedSlot {
  unsigned long long w[kSchedWords];
  uint32_t order[kPvCacheMax];
  PvRec pv[kPvCacheMax];
  // epoch kernel (pt_epoch.cuh): first epoch and unit count per row, prefix of the batch counts in row order
  double un0[kPvCacheMax];
  uint32_t ucnt[kPvCacheMax];
};
__device__ SchedSlot g_sched[kSchedSlots];

// Work area of pt_gimenez_interp_static (the per-vector z-tables of pt_gimenez_interp): 4 MiB that every device which loads
// the library holds until the process ends.
constexpr int64_t kGimStaticWork = 1 << 19;   // doubles
static __device__ __align__(256) double g_gim_work[kGimStaticWork];

struct SlotHost {
  cudaEvent_t ev = nullptr;
  bool used = false;
};
struct DeviceSlots {
  SchedSlot* base = nullptr;
  SlotHost slot[kSchedRing];
  int next = 0, n_graph = 0;
};
static std::mutex g_slot_mutex;
static DeviceSlots g_dev_slots[64];

struct SlotTicket {
  SchedSlot* slot = nullptr;
  int dev = -1, idx = -1;
  bool capturing = false;
};

// Take a slot for a launch on `st` (see above).  Returns a null slot on a CUDA error or when the graph slots are used up.
static SlotTicket slot_acquire(cudaStream_t st) {
  SlotTicket t;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return t;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) return t;
  t.capturing = cs != cudaStreamCaptureStatusNone;
  std::lock_guard<std::mutex> lock(g_slot_mutex);
  DeviceSlots& D = g_dev_slots[dev];
  if (!D.base) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_sched) != cudaSuccess) return t;
    D.base = (SchedSlot*)p;
  }
  t.dev = dev;
  if (t.capturing) {
    if (D.n_graph >= kSchedGraph) return t;
    t.idx = kSchedRing + D.n_graph++;
    t.slot = D.base + t.idx;
    return t;
  }
  int pick = -1;
  for (int k = 0; k < kSchedRing; ++k) {
    const int i = (D.next + k) % kSchedRing;
    SlotHost& h = D.slot[i];
    if (!h.used || cudaEventQuery(h.ev) == cudaSuccess) { pick = i; break; }
  }
  (void)cudaGetLastError();            // cudaEventQuery's cudaErrorNotReady is not an error
  if (pick < 0) {                      // every slot in flight: order this launch behind the oldest one
    pick = D.next;
    if (cudaStreamWaitEvent(st, D.slot[pick].ev, 0) != cudaSuccess) return t;
  }
  D.next = (pick + 1) % kSchedRing;
  SlotHost& h = D.slot[pick];
  if (!h.ev && cudaEventCreateWithFlags(&h.ev, cudaEventDisableTiming) != cudaSuccess) return t;
  h.used = true;
  t.slot = D.base + pick; t.idx = pick;
  return t;
}

// Mark the end of the launch that holds the slot (after its last kernel has been enqueued on `st`).
static void slot_release(const SlotTicket& t, cudaStream_t st) {
  if (!t.slot || t.capturing) return;
  std::lock_guard<std::mutex> lock(g_slot_mutex);
  cudaEventRecord(g_dev_slots[t.dev].slot[t.idx].ev, st);
}

// S1-S2 alone: signed projected separation of every subsample.
__global__ void __launch_bounds__(kThreads) orbit_kernel(const double* __restrict__ times, int64_t n_t,
                                                         int64_t t_stride_pv, const double* __restrict__ params,
                                                         int n_pb, int n_ss, double t_exp, double* __restrict__ z_out,
                                                         int blocks_per_pv, int solver) {
  __shared__ PvConst c;
  __shared__ double ser[5];
  __shared__ int s_solver;
  const int64_t pv = blockIdx.x / blocks_per_pv;
  const int chunk = (int)(blockIdx.x % blocks_per_pv);
  const double* row = params + pv * (6 + 3 * (int64_t)n_pb);
  if (threadIdx.x == 0) {
    bool ok = true;
    double ksum = 0.0;
    for (int j = 0; j < n_pb; ++j) {
      const double k = row[6 + 3 * j], u1 = row[7 + 3 * j], u2 = row[8 + 3 * j];
      if (!(isfinite(k) && isfinite(u1) && isfinite(u2)) || !(k >= 0.0) || (1.0 - u1 / 3.0 - u2 / 6.0) == 0.0) ok = false;
      ksum += k;
    }
    c.khat = ksum / (double)n_pb;
    pv_setup_orbit(c, row, ok, n_ss, t_exp);
    // the routine for this parameter vector ("selects the most appropriate orbit calculation routine based on the
    // eccentricity"); a non-exact routine asked for by name is used even for e == 0 (w and Mtr are then set up as for e > 0)
    int sv = (c.flags & PV_BAD) ? SOLVER_EXACT : dispatch_solver(solver, c.e);
    if (sv == SOLVER_NEWTON) sv = SOLVER_EXACT;
    if (sv != SOLVER_EXACT) {
      if (c.flags & PV_CIRCULAR) {   // e == 0 through an eccentric routine: conjunction at true anomaly π/2 - w
        double w = row[5];
        sincos(w, &c.sinw, &c.cosw);
        c.rt1me2 = 1.0;
        const double ftr = 0.5 * kPi - atan2(c.sinw, c.cosw);
        c.Mtr = ftr - kTwoPi * rint(ftr * (1.0 / kTwoPi));
      }
      series_coefficients(c.e, sv == SOLVER_PS3 ? 3 : 5, ser);
    }
    s_solver = sv;
  }
  __syncthreads();
  const int sv = s_solver;
  const int64_t n = n_t * n_ss;
  const double* tt = times + pv * t_stride_pv;
  double* zo = z_out + pv * n;
  const bool bad = c.flags & PV_BAD;
  for (int64_t i = (int64_t)chunk * kThreads + threadIdx.x; i < n; i += (int64_t)blocks_per_pv * kThreads) {
    double z;
    if (bad) z = nan64();
    else {
      const int64_t e = i / n_ss;
      const int s = (int)(i - e * n_ss);
      const double t = __ldg(tt + e);
      const double ts = (n_ss > 1) ? __dadd_rn(t, subsample_offset(s, n_ss, t_exp)) : t;
      const double ph = fold_phase(ts, c.t0, c.P, c.invP, c.flags & PV_SLOWDIV);
      z = (sv == SOLVER_EXACT) ? orbit_z_signed(c, ph) : orbit_z_signed_alt(c, ser, ph, sv);
    }
    zo[i] = z;
  }
}

// S8: table nodes.
template <typename TT>
__global__ void __launch_bounds__(kThreads) table_kernel(double k_min, double dk, int n_k, double dz, int n_z, int n_fn,
                                                         TT* __restrict__ tb) {
  const int64_t n = (int64_t)n_k * n_z;
  for (int64_t idx = (int64_t)blockIdx.x * kThreads + threadIdx.x; idx < n; idx += (int64_t)gridDim.x * kThreads) {
    const int i = (int)(idx / n_z), j = (int)(idx - (int64_t)i * n_z);
    const double k = __dadd_rn(k_min, __dmul_rn((double)i, dk));
    const double z = __dmul_rn((double)j, dz);
    Basis b;
    if (k > 1.0e-150) b = ma_basis(k, z);
    else { b.le = 0.0; b.ld = 0.0; b.ed = 0.0; }
    TT* o = tb + idx * n_fn;
    o[0] = (TT)b.le; o[1] = (TT)b.ld; o[2] = (TT)b.ed;
    if (n_fn == 4) o[3] = (TT)0;
  }
}

constexpr int kBaseBlocks = 128;   // chi2 baseline partials (prep_kernel), kept in the tail of the slot's words

// FP64-pipe peak probe: 8 independent DFMA chains per thread.
__global__ void __launch_bounds__(kThreads) dfma_probe_kernel(int iters, double* __restrict__ sink) {
  double a0 = threadIdx.x * 1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999, c = 1e-6;
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  sink[(size_t)blockIdx.x * kThreads + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// FP32-pipe peak probe: 8 independent FFMA chains per thread.
__global__ void __launch_bounds__(kThreads) ffma_probe_kernel(int iters, float* __restrict__ sink) {
  float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const float m = 0.999999f, c = 1e-6f;
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
    a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
  }
  sink[(size_t)blockIdx.x * kThreads + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// ------------------------------------------------------------------------------------------------ host side
static int check_common(const void* times, const void* params, const void* out, int64_t n_t, int64_t t_stride_pv,
                        int64_t n_pv, int n_pb, int n_ss) {
  if (!times || !params || !out) return PT_ERR_NULL;
  if (n_t <= 0 || n_pv <= 0 || n_pb < 1 || n_ss < 1 || n_pb > kMaxPassbands) return PT_ERR_SIZE;
  if (t_stride_pv != 0 && t_stride_pv < n_t) return PT_ERR_SIZE;
  return PT_OK;
}

static bool table_ok(const pt_table* tb) {
  return tb && tb->d_data && tb->n_k >= 2 && tb->n_z >= 2 && (tb->n_fn == 3 || tb->n_fn == 4) && tb->dk > 0.0 && tb->dz > 0.0 &&
         (tb->dtype == PT_F64 || tb->dtype == PT_F32);
}

// Number of SMs of the current device (the persistent grid is sized from it), cached per device.
static int sm_count() {
  static std::atomic<int> cached[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  int n = cached[dev].load();
  if (n == 0) {
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    cached[dev].store(n);
  }
  return n;
}

// How a launch is cut up (pure host logic; exported as pt_plan for the CPU tests).
//   persistent grid: PT_MIN_BLOCKS blocks of 8 autonomous warps per SM; tiles of `tile_len` exposures of one parameter
//   vector, about kTilesPerWarp per warp so that heavy and light tiles average out.
//   mode 0  one global tile counter, rows in index order
//   mode 1  one counter per parameter vector (a warp keeps its parameter vector: the setup is reused)
//   mode 2  global counter, rows in order of decreasing expected work (LPT): heavy tiles first, the launch ends on light ones
constexpr int64_t kLptRows = 512;   // rows up to which the longest-processing-time-first order is used
struct Plan {
  int tile_len;
  int64_t tiles_per_pv;
  int mode;
  int64_t blocks;
};
#ifndef PT_LPT_TILE
#define PT_LPT_TILE 256
#endif
#ifndef PT_RANGE_MIN
#define PT_RANGE_MIN 131072   // exposures (n_pv x n_t) from which the axis check + range mode pay for the extra launch
#endif
static Plan plan_tiles(int64_t n_pv, int64_t n_t, int n_sm) {
  Plan p{};
  const int64_t warps = (int64_t)n_sm * PT_MIN_BLOCKS * kWarpsPerBlock;
  constexpr int64_t kTilesPerWarp = 8;
  const double total = (double)n_pv * (double)n_t;
  int64_t tl = (int64_t)(total / (double)(warps * kTilesPerWarp));
  tl = (tl + 255) / 256 * 256;
  if (tl < 256) tl = 256;
  if (tl > 16384) tl = 16384;
  if (total < (double)(64 * n_sm)) {
    // a tiny problem (configs[0]: 1000 exposures) is a latency, not a throughput: short tiles, so that it is one round of
    // many warps instead of many rounds of a few
    tl = ((int64_t)(total / (double)(2 * n_sm)) + 31) / 32 * 32;
    tl = tl < 32 ? 32 : (tl > 256 ? 256 : tl);
  }
  int64_t tpp = (n_t + tl - 1) / tl;
  const bool few = (n_pv <= kSchedWords - kSchedHead - kBaseBlocks && tpp >= 2);   // the slot's tail holds the chi2 partials
  p.mode = few ? 1 : 0;
  if (few && n_pv <= kLptRows && n_pv * tpp >= 2 * warps) {   // worth ranking the rows only with several tiles per warp
    p.mode = 2;
    if (tl < PT_LPT_TILE) { tl = PT_LPT_TILE; tpp = (n_t + tl - 1) / tl; }
  }
  if (tpp > 0x7fffffff || (double)tpp * (double)n_pv > 9.0e18) return p;   // tile_len == 0: too large
  p.tile_len = (int)tl;
  p.tiles_per_pv = tpp;
  const int64_t n_tiles = n_pv * tpp;
  p.blocks = (n_tiles + kWarpsPerBlock - 1) / kWarpsPerBlock;
  if (p.blocks > warps / kWarpsPerBlock) p.blocks = warps / kWarpsPerBlock;
  return p;
}

struct Chi2Args {
  const double* obs;
  const double* isig;
};
constexpr int kDtypeChi2 = 100;   // internal: d_flux is chi2[n_pv], `like` holds the observations

static int launch_flux(int mode, const pt_table* tb, const double* d_times, int64_t n_t, int64_t t_stride_pv,
                       const double* d_params, int64_t n_pv, int n_pb, int n_ss, double t_exp, int dtype, void* d_flux,
                       int32_t* d_status, cudaStream_t st, const Chi2Args* like = nullptr, int pb_view = -1, int n_pb_row = 0) {
  int rc = check_common(d_times, d_params, d_flux, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  if (dtype != PT_F64 && dtype != PT_F32 && dtype != PT_F32S && !(dtype == kDtypeChi2 && like)) return PT_ERR_DTYPE;
  const bool f32a = (dtype == PT_F32) && mode == 0 && n_pb == 1 && pb_view == -1;   // fp32 arithmetic where the kernels have it
  if (dtype == PT_F32S) dtype = PT_F32;                   // from here on: the storage type
  FluxArgs A{};
  A.times = d_times; A.n_t = n_t; A.t_stride_pv = t_stride_pv; A.params = d_params; A.n_pv = n_pv;
  A.n_pb = n_pb; A.n_ss = n_ss; A.t_exp = t_exp; A.flux = d_flux; A.status = d_status;
  A.row_stride = 6 + 3 * (int64_t)n_pb; A.pb_first = 0; A.flux_pv_stride = (int64_t)n_pb * n_t; A.flux_off = 0;
  A.pbk = (pb_view == -2) ? 1 : 0;
  A.f32a = f32a ? 1 : 0;
  if (pb_view >= 0) {   // single-passband view of passband `pb_view` in rows of n_pb_row passbands
    A.row_stride = 6 + 3 * (int64_t)n_pb_row; A.pb_first = pb_view;
    A.flux_pv_stride = (int64_t)n_pb_row * n_t; A.flux_off = (int64_t)pb_view * n_t;
  }
  if (mode == 1) {
    if (!table_ok(tb)) return PT_ERR_TABLE;
    A.tb = tb->d_data; A.tb_dtype = tb->dtype; A.n_k = tb->n_k; A.n_z = tb->n_z; A.n_fn = tb->n_fn;
    A.k_min = tb->k_min; A.dk = tb->dk; A.dz = tb->dz; A.inv_dz = 1.0 / tb->dz;
  }
  const pt::Plan plan = plan_tiles(n_pv, n_t, sm_count());
  if (plan.tile_len == 0) return PT_ERR_SIZE;
  A.tile_len = plan.tile_len; A.tiles_per_pv = (int)plan.tiles_per_pv; A.n_tiles = n_pv * plan.tiles_per_pv;
  A.per_pv = plan.mode == 1;
  int lg = 0;
  while (((int64_t)1 << lg) < (int64_t)n_ss) ++lg;
  A.fx_bits = 61 - lg;
  A.fx_scale = ldexp(1.0, A.fx_bits);
  A.fx_inv = 1.0 / (A.fx_scale * (double)n_ss);
  A.inv_nss = 1.0 / (double)n_ss;
  const dim3 grid((unsigned)plan.blocks);
  if (dtype == kDtypeChi2) {
    A.obs = like->obs; A.isig = like->isig; A.chi2 = (double*)d_flux; A.flux = nullptr;
  }
  const SlotTicket ticket = slot_acquire(st);
  SchedSlot* slot = ticket.slot;
  if (!slot) return PT_ERR_CUDA;
  A.sched = slot->w;
  // What prep_kernel is asked to leave in the slot (pt_flux.cuh):
  //   records  single passband, at most kPvCacheMax parameter vectors, at least two tiles each (the per-tile setup is 15 % of
  //            the flux kernel's instructions on configs[1] when done per tile, 18 % of the direct kernel's time on `dense`)
  //   axis     one shared time axis of a problem large enough for the extra launch to pay: is it ascending?
  //   order    global tile counter: heaviest rows first (mode 2), or rows by k̂ for the interpolated model
  //   baseline fused likelihood
  const bool want_rec = n_pb == 1 && pb_view < 0 && n_pv <= kPvCacheMax && A.n_tiles >= PT_REC_MIN_TILES * n_pv &&
                        (double)n_pv * (double)n_t >= 65536.0;   // a small problem does not pay for the extra launch
  const bool want_axis = t_stride_pv == 0 && n_t >= 2048 && (double)n_pv * (double)n_t >= (double)PT_RANGE_MIN;
  // epoch kernel: one passband on one shared axis that prep_kernel checks; it does the whole launch if the axis is ascending,
  // else the general kernel launched behind it does
  const bool want_epoch = want_axis && n_pb == 1 && pb_view < 0 && n_pv <= kPvCacheMax && n_t < 0x7fffff00LL &&
                          (mode == 0 || (size_t)tb->n_z * sizeof(double) <= 110000);
  const bool want_order = n_pv <= kPvCacheMax && n_pv >= 2 &&
                          (want_epoch || plan.mode == 2 || (mode == 1 && plan.mode == 0 && A.n_tiles >= 4 * (int64_t)grid.x * kWarpsPerBlock));
  // direct kernel: the fp32 variant where there are no epochs to look for (per-row times, or a small problem)
#ifndef PT_DIRECT_F64
#define PT_DIRECT_F64 0
#endif
  const bool direct64 = PT_DIRECT_F64 && dtype == PT_F64 && mode == 0 && n_pb == 1 && pb_view < 0 && t_stride_pv != 0;
  const bool use_direct = (f32a || direct64) && n_ss == 1 && !want_epoch;
  PrepArgs Q{};
  if (want_rec || want_epoch) { Q.rec = slot->pv; Q.n_rec_blocks = (int)((n_pv + kWarpsPerBlock - 1) / kWarpsPerBlock); }
  if (want_axis) { int nb = (int)((n_t + 8 * kThreads - 1) / (8 * kThreads)); Q.n_axis_blocks = nb > 64 ? 64 : nb; }
  if (want_order) { Q.order = slot->order; Q.order_by_k = (want_epoch ? mode == 1 : plan.mode == 0) ? 1 : 0; Q.n_order_blocks = 1; }
  if (dtype == kDtypeChi2) {
    // out-of-transit baseline into the tail of the slot's words, chi2[] zeroed
    const int64_t n_obs = (int64_t)n_pb * n_t;
    int nb = (int)((n_obs + 4095) / 4096);
    Q.n_base_blocks = nb > kBaseBlocks ? kBaseBlocks : (nb < 1 ? 1 : nb);
    Q.base_part = reinterpret_cast<double*>(A.sched + kSchedWords - kBaseBlocks);
    A.base_part = Q.base_part; A.n_base_part = Q.n_base_blocks;
  }
  const int n_prep = Q.n_rec_blocks + Q.n_axis_blocks + Q.n_order_blocks + Q.n_base_blocks;
  // epoch kernel: interpolated model = blocks of 16 warps that stage the table (n_z doubles of shared memory, two per SM);
  // exact model = single-warp blocks, 24 per SM.  About four units per block so that the ticket counter balances the load.
#ifndef PT_EPOCH_NT
#define PT_EPOCH_NT 512
#endif
  const int e_nt = (mode == 1) ? PT_EPOCH_NT : 32;
  const int64_t e_grid = (int64_t)sm_count() * ((mode == 1) ? 2 : PT_EPOCH_WARPS);
  const size_t e_smem = (mode == 1) ? (size_t)tb->n_z * sizeof(double) : 0;
  if (want_epoch) {
    Q.want_units = 1; Q.un0 = slot->un0; Q.ucnt = slot->ucnt; Q.n_blocks = n_prep;
    A.un0 = slot->un0; A.ucnt = slot->ucnt;
#ifndef PT_EPOCH_UNITS
#define PT_EPOCH_UNITS 4
#endif
    int64_t C = (PT_EPOCH_UNITS * e_grid + n_pv - 1) / n_pv;
    A.unit_chunks = (int)(C < 1 ? 1 : (C > 4096 ? 4096 : C));
    A.base_added = (dtype == kDtypeChi2) ? 1 : 0;
  }
  if (n_prep > 0) {
    // an ordinary launch: ordered behind whatever the caller enqueued before (the kernel that wrote d_params, the fill that
    // zeroed d_status), so it and its dependent below see the caller's data
    if (mode == 0) prep_kernel<0><<<n_prep, kThreads, 0, st>>>(A, Q);
    else prep_kernel<1><<<n_prep, kThreads, 0, st>>>(A, Q);
    g_launches.fetch_add(1);
    A.prep = 1;
    A.pvcache = (want_rec || want_epoch) ? slot->pv : nullptr;
    A.order = want_order ? slot->order : nullptr;
    A.range = want_axis ? 1 : 0;
  }
  // 16-byte loads/stores need even row lengths/strides and 16-byte aligned bases
  const bool v2 = (n_t % 2 == 0) && (t_stride_pv % 2 == 0) && (reinterpret_cast<uintptr_t>(d_times) % 16 == 0) &&
                  (dtype == kDtypeChi2 || reinterpret_cast<uintptr_t>(d_flux) % 16 == 0);
  const bool p1 = (n_pb == 1), s1 = (n_ss == 1);
  // behind prep_kernel the flux kernel is a programmatic dependent launch: its launch latency overlaps that kernel, and it
  // waits (griddepcontrol.wait) before it reads the slot
  cudaLaunchAttribute pdl_attr[1];
  pdl_attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl_attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cfg.attrs = pdl_attr; cfg.numAttrs = A.prep ? 1 : 0;
  if (use_direct) {
    const bool dv2 = v2 && reinterpret_cast<uintptr_t>(d_flux) % 16 == 0;
    cudaError_t d_err;
    if (direct64) d_err = dv2 ? cudaLaunchKernelEx(&cfg, direct_kernel<2, double, 0>, A) : cudaLaunchKernelEx(&cfg, direct_kernel<1, double, 0>, A);
    else d_err = dv2 ? cudaLaunchKernelEx(&cfg, direct_kernel<2, float, 3>, A) : cudaLaunchKernelEx(&cfg, direct_kernel<1, float, 3>, A);
    g_launches.fetch_add(1);
    const cudaError_t err2 = cudaGetLastError();
    slot_release(ticket, st);
    return (d_err == cudaSuccess && err2 == cudaSuccess) ? PT_OK : PT_ERR_CUDA;
  }
  if (want_epoch) {
    cudaLaunchConfig_t ecfg = cfg;
    ecfg.gridDim = dim3((unsigned)e_grid);
    ecfg.blockDim = dim3((unsigned)e_nt);
    ecfg.dynamicSmemBytes = e_smem;
    ecfg.numAttrs = 1;
    const bool ev2 = (n_t % 2 == 0) && (dtype == kDtypeChi2 || reinterpret_cast<uintptr_t>(d_flux) % 16 == 0);
    cudaError_t e_err = cudaSuccess;
#define PT_EPOCH(M, NTT, VV, S, T)                                                                                  \
  do {                                                                                                              \
    if (e_smem > 48 * 1024)                                                                                         \
      e_err = cudaFuncSetAttribute(epoch_kernel<M, NTT, VV, S, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e_smem); \
    if (e_err == cudaSuccess) e_err = cudaLaunchKernelEx(&ecfg, epoch_kernel<M, NTT, VV, S, T>, A);                 \
  } while (0)
#define PT_EPOCH_T(M, NTT, T)                                                \
  do {                                                                       \
    if (ev2) { if (s1) PT_EPOCH(M, NTT, true, true, T); else PT_EPOCH(M, NTT, true, false, T); } \
    else { if (s1) PT_EPOCH(M, NTT, false, true, T); else PT_EPOCH(M, NTT, false, false, T); }   \
  } while (0)
    if (mode == 0) {
      if (dtype == PT_F64) PT_EPOCH_T(0, 32, double); else if (dtype == PT_F32) PT_EPOCH_T(0, 32, float); else PT_EPOCH_T(0, 32, Chi2);
    } else {
      if (dtype == PT_F64) PT_EPOCH_T(1, PT_EPOCH_NT, double); else if (dtype == PT_F32) PT_EPOCH_T(1, PT_EPOCH_NT, float); else PT_EPOCH_T(1, PT_EPOCH_NT, Chi2);
    }
#undef PT_EPOCH_T
#undef PT_EPOCH
    g_launches.fetch_add(1);
    const cudaError_t err2 = cudaGetLastError();
    slot_release(ticket, st);
    return (e_err == cudaSuccess && err2 == cudaSuccess) ? PT_OK : PT_ERR_CUDA;
  }
#define PT_LAUNCH(M, VV, P, S, T) cudaLaunchKernelEx(&cfg, flux_kernel<M, VV, P, S, T>, A)
#define PT_LAUNCH_S(M, VV, P, T)                             \
  do {                                                       \
    if (s1) PT_LAUNCH(M, VV, P, true, T);                    \
    else PT_LAUNCH(M, VV, P, false, T);                      \
  } while (0)
#define PT_LAUNCH_T(M, T)                                    \
  do {                                                       \
    if (v2 && p1) PT_LAUNCH_S(M, 2, true, T);                \
    else if (v2) PT_LAUNCH_S(M, 2, false, T);                \
    else if (p1) PT_LAUNCH_S(M, 1, true, T);                 \
    else PT_LAUNCH_S(M, 1, false, T);                        \
  } while (0)
  if (mode == 0) {
    if (dtype == PT_F64) PT_LAUNCH_T(0, double); else if (dtype == PT_F32) PT_LAUNCH_T(0, float); else PT_LAUNCH_T(0, Chi2);
  } else {
    if (dtype == PT_F64) PT_LAUNCH_T(1, double); else if (dtype == PT_F32) PT_LAUNCH_T(1, float); else PT_LAUNCH_T(1, Chi2);
  }
#undef PT_LAUNCH_T
#undef PT_LAUNCH_S
#undef PT_LAUNCH
  g_launches.fetch_add(1);
  const cudaError_t err = cudaGetLastError();
  slot_release(ticket, st);
  return err == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

}  // namespace pt

using namespace pt;

extern "C" {

int pt_build_arch(void) {
#ifdef PT_BUILD_ARCH
  return PT_BUILD_ARCH;
#else
  return 0;
#endif
}

int64_t pt_launch_count(void) { return g_launches.load(); }

int pt_plan(int64_t n_pv, int64_t n_t, int32_t n_sm, int64_t* h_out) {
  if (!h_out) return PT_ERR_NULL;
  if (n_pv <= 0 || n_t <= 0 || n_sm <= 0) return PT_ERR_SIZE;
  const Plan p = plan_tiles(n_pv, n_t, n_sm);
  if (p.tile_len == 0) return PT_ERR_SIZE;
  h_out[0] = p.tile_len; h_out[1] = p.tiles_per_pv; h_out[2] = p.mode; h_out[3] = p.blocks;
  return PT_OK;
}

int pt_probe_dfma(int32_t blocks, int32_t iters, double* d_sink, void* stream) {
  if (!d_sink) return PT_ERR_NULL;
  if (blocks < 1 || iters < 1) return PT_ERR_SIZE;
  dfma_probe_kernel<<<(unsigned)blocks, kThreads, 0, (cudaStream_t)stream>>>(iters, d_sink);
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

int pt_probe_ffma(int32_t blocks, int32_t iters, float* d_sink, void* stream) {
  if (!d_sink) return PT_ERR_NULL;
  if (blocks < 1 || iters < 1) return PT_ERR_SIZE;
  ffma_probe_kernel<<<(unsigned)blocks, kThreads, 0, (cudaStream_t)stream>>>(iters, d_sink);
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

int pt_orbit_z(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
               int32_t n_pb, int32_t n_ss, double t_exp, double* d_z, void* stream) {
  return pt_orbit_z_solver(d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss, t_exp, PT_SOLVER_EXACT, d_z, stream);
}

int pt_orbit_z_solver(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                      int32_t n_pb, int32_t n_ss, double t_exp, int32_t solver, double* d_z, void* stream) {
  int rc = check_common(d_times, d_params, d_z, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  if (solver < PT_SOLVER_EXACT || solver > PT_SOLVER_FAST) return PT_ERR_SIZE;
  const int64_t n = n_t * n_ss;
  int64_t bpp = (n + (int64_t)kThreads * 8 - 1) / ((int64_t)kThreads * 8);
  const int64_t cap = ((int64_t)sm_count() * 16 + n_pv - 1) / n_pv;
  if (bpp > cap) bpp = cap;
  if (bpp < 1) bpp = 1;
  if (n_pv * bpp > 0x7fffffff) return PT_ERR_SIZE;
  orbit_kernel<<<(unsigned)(n_pv * bpp), kThreads, 0, (cudaStream_t)stream>>>(d_times, n_t, t_stride_pv, d_params, n_pb,
                                                                              n_ss, t_exp, d_z, (int)bpp, (int)solver);
  g_launches.fetch_add(1);
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

int pt_ma_quad_exact(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                     int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype, void* d_flux, int32_t* d_status,
                     void* stream) {
  return launch_flux(0, nullptr, d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss, t_exp, dtype, d_flux, d_status,
                     (cudaStream_t)stream);
}

int pt_ma_quad_exact_pbk(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                         int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype, void* d_flux, int32_t* d_status,
                         void* stream) {
  int rc = check_common(d_times, d_params, d_flux, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  if (n_ss == 1 && n_pb > 1)   // fused: one launch, the orbit once per sample, the basis functions once per passband
    return launch_flux(0, nullptr, d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss, t_exp, dtype, d_flux, d_status,
                       (cudaStream_t)stream, nullptr, -2, n_pb);
  for (int j = 0; j < n_pb && rc == PT_OK; ++j)
    rc = launch_flux(0, nullptr, d_times, n_t, t_stride_pv, d_params, n_pv, 1, n_ss, t_exp, dtype, d_flux, d_status,
                     (cudaStream_t)stream, nullptr, j, n_pb);
  return rc;
}

int pt_table_spacing(double k_min, double k_max, int32_t n_k, double z_max, int32_t n_z, double* h_dk, double* h_dz) {
  if (!h_dk || !h_dz) return PT_ERR_NULL;
  if (n_k < 2 || n_z < 2 || !(k_max > k_min) || !(k_min >= 0.0) || !(z_max > 0.0)) return PT_ERR_SIZE;
  *h_dk = (k_max - k_min) / (double)(n_k - 1);
  *h_dz = z_max / (double)(n_z - 1);
  return PT_OK;
}

int pt_ma_table_build(double k_min, double k_max, int32_t n_k, double z_max, int32_t n_z, int32_t dtype, int32_t n_fn,
                      void* d_table, void* stream) {
  if (!d_table) return PT_ERR_NULL;
  if (n_k < 2 || n_z < 2 || (n_fn != 3 && n_fn != 4) || !(k_max > k_min) || !(k_min >= 0.0) || !(z_max > 0.0))
    return PT_ERR_SIZE;
  if (dtype != PT_F64 && dtype != PT_F32) return PT_ERR_DTYPE;
  double dk, dz;
  pt_table_spacing(k_min, k_max, n_k, z_max, n_z, &dk, &dz);
  const int64_t n = (int64_t)n_k * n_z;
  int64_t blocks = (n + kThreads - 1) / kThreads;
  if (blocks > (int64_t)sm_count() * 64) blocks = (int64_t)sm_count() * 64;
  if (dtype == PT_F64)
    table_kernel<double><<<(unsigned)blocks, kThreads, 0, (cudaStream_t)stream>>>(k_min, dk, n_k, dz, n_z, n_fn, (double*)d_table);
  else
    table_kernel<float><<<(unsigned)blocks, kThreads, 0, (cudaStream_t)stream>>>(k_min, dk, n_k, dz, n_z, n_fn, (float*)d_table);
  g_launches.fetch_add(1);
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

int pt_ma_quad_interp(const pt_table* table, const double* d_times, int64_t n_t, int64_t t_stride_pv,
                      const double* d_params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype,
                      void* d_flux, int32_t* d_status, void* stream) {
  return launch_flux(1, table, d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss, t_exp, dtype, d_flux, d_status,
                     (cudaStream_t)stream);
}

int pt_ma_quad_chi2(const pt_table* table, const double* d_times, int64_t n_t, const double* d_params, int64_t n_pv,
                    int32_t n_pb, int32_t n_ss, double t_exp, const double* d_obs, const double* d_isig, double* d_chi2,
                    int32_t* d_status, void* stream) {
  if (!d_obs || !d_isig) return PT_ERR_NULL;
  const Chi2Args like{d_obs, d_isig};
  return launch_flux(table ? 1 : 0, table, d_times, n_t, 0, d_params, n_pv, n_pb, n_ss, t_exp, kDtypeChi2, d_chi2, d_status,
                     (cudaStream_t)stream, &like);
}

// ---- the Giménez model
int pt_gimenez_coef_size(int32_t n_ldc, int32_t n_j, int64_t* h_bytes) {
  if (!h_bytes) return PT_ERR_NULL;
  if (n_ldc < 1 || n_ldc > kGimMaxLdc || n_j < 0 || n_j > kGimMaxNj) return PT_ERR_SIZE;
  *h_bytes = (int64_t)(n_ldc + 1) * (n_j + 1) * kGimCoef * (int64_t)sizeof(double);
  return PT_OK;
}

int pt_gimenez_coef_build(int32_t n_ldc, int32_t n_j, double* d_coef, void* stream) {
  if (!d_coef) return PT_ERR_NULL;
  if (n_ldc < 1 || n_ldc > kGimMaxLdc || n_j < 0 || n_j > kGimMaxNj) return PT_ERR_SIZE;
  if (reinterpret_cast<uintptr_t>(d_coef) % 32 != 0) return PT_ERR_SIZE;
  const int n = (n_ldc + 1) * (n_j + 1);
  gimenez_coef_kernel<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(n_ldc, n_j, d_coef);
  g_launches.fetch_add(1);
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

static int gimenez_launch(int mode, const double* d_coef, int32_t n_ldc, int32_t n_j, int32_t n_in, int32_t n_out, double* d_work,
                          const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                          int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux, int32_t* d_status, void* stream) {
  if (!d_coef || !d_times || !d_params || !d_flux || (mode == 1 && !d_work)) return PT_ERR_NULL;
  if (n_t <= 0 || n_pv <= 0 || n_pb < 1 || n_pb > kGimMaxPb || n_ss < 1 || n_ldc < 1 || n_ldc > kGimMaxLdc || n_j < 0 ||
      n_j > kGimMaxNj || (t_stride_pv != 0 && t_stride_pv < n_t) || (mode == 1 && (n_in < 2 || n_out < 2)))
    return PT_ERR_SIZE;
  if (reinterpret_cast<uintptr_t>(d_coef) % 32 != 0) return PT_ERR_SIZE;
  GimArgs A{};
  A.coef = d_coef; A.n_ldc = n_ldc; A.n_j = n_j; A.times = d_times; A.n_t = n_t; A.t_stride_pv = t_stride_pv;
  A.params = d_params; A.n_pv = n_pv; A.n_pb = n_pb; A.n_ss = n_ss; A.t_exp = t_exp; A.flux = d_flux; A.status = d_status;
  A.work = d_work; A.n_in = n_in; A.n_out = n_out;
  cudaStream_t st = (cudaStream_t)stream;
  if (mode == 1) {
    const int64_t nn = n_pv * (int64_t)(n_in + n_out);
    if ((nn + 255) / 256 > 0x7fffffff) return PT_ERR_SIZE;
    gimenez_table_kernel<<<(unsigned)((nn + 255) / 256), 256, 0, st>>>(A);
    g_launches.fetch_add(1);
  }
  int64_t bpp = (n_t + 255) / 256;
  const int64_t cap = ((int64_t)sm_count() * 16 + n_pv - 1) / n_pv;
  if (bpp > cap) bpp = cap;
  if (bpp < 1) bpp = 1;
  if (n_pv * bpp > 0x7fffffff) return PT_ERR_SIZE;
  // the series reads the coefficient table (n_ldc+1)(n_j+1) x 64 bytes once per term: from shared memory when it fits
  const size_t coef_bytes = (size_t)(n_ldc + 1) * (n_j + 1) * kGimCoef * sizeof(double);
  const int in_smem = (mode == 0 && coef_bytes <= 40 * 1024) ? 1 : 0;
  if (mode == 0) gimenez_kernel<0><<<(unsigned)(n_pv * bpp), 256, in_smem ? coef_bytes : 0, st>>>(A, (int)bpp, in_smem);
  else gimenez_kernel<1><<<(unsigned)(n_pv * bpp), 256, 0, st>>>(A, (int)bpp, 0);
  g_launches.fetch_add(1);
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
}

int pt_gimenez_exact(const double* d_coef, int32_t n_ldc, int32_t n_j, const double* d_times, int64_t n_t, int64_t t_stride_pv,
                     const double* d_params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux,
                     int32_t* d_status, void* stream) {
  return gimenez_launch(0, d_coef, n_ldc, n_j, 0, 0, nullptr, d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss, t_exp,
                        d_flux, d_status, stream);
}

int pt_gimenez_interp(const double* d_coef, int32_t n_ldc, int32_t n_j, int32_t n_in, int32_t n_out, double* d_work,
                      const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                      int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux, int32_t* d_status, void* stream) {
  return gimenez_launch(1, d_coef, n_ldc, n_j, n_in, n_out, d_work, d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss,
                        t_exp, d_flux, d_status, stream);
}

// ---- pt_gimenez_interp for callers that must not allocate: the z-tables live in a fixed array of this library instead of
// caller memory.  In host code `g_gim_work` is only a handle: the device address comes from cudaGetSymbolAddress, once per
// device, with that device current.  Every call on a device shares the array (it keeps the last call's tables; a call
// overwrites every node it reads, so nothing has to be cleared); calls that overlap on the GPU race on it.
int64_t pt_gimenez_static_work_doubles(void) { return pt::kGimStaticWork; }

int pt_gimenez_interp_static(const double* d_coef, int32_t n_ldc, int32_t n_j, int32_t n_in, int32_t n_out,
                             const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                             int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux, int32_t* d_status, void* stream) {
  // sizes first: the static work area holds kGimStaticWork doubles
  if (n_pv <= 0 || n_ldc < 1 || n_ldc > kGimMaxLdc || n_in < 2 || n_out < 2) return PT_ERR_SIZE;
  if ((int64_t)n_in + n_out > pt::kGimStaticWork) return PT_ERR_SIZE;
  if (n_pv > pt::kGimStaticWork / ((int64_t)(n_ldc + 1) * ((int64_t)n_in + n_out))) return PT_ERR_SIZE;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return PT_ERR_CUDA;
  double* d_work = nullptr;
  {
    static std::mutex mu;
    static double* work_of[64];
    std::lock_guard<std::mutex> lock(mu);
    if (!work_of[dev]) {
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, pt::g_gim_work) != cudaSuccess || !p) { (void)cudaGetLastError(); return PT_ERR_CUDA; }
      work_of[dev] = (double*)p;
    }
    d_work = work_of[dev];
  }
  return gimenez_launch(1, d_coef, n_ldc, n_j, n_in, n_out, d_work, d_times, n_t, t_stride_pv, d_params, n_pv, n_pb, n_ss,
                        t_exp, d_flux, d_status, stream);
}

// ---- host-buffer forms: H2D, kernels, D2H on an internal stream, then wait.
// Scratch of the calling thread on one device: a stream and four grow-only device buffers (times, parameters, flux, status),
// kept between calls so that a steady-state call allocates nothing; freed when the thread ends.
struct HostScratch {
  cudaStream_t st = nullptr;
  void* buf[4] = {nullptr, nullptr, nullptr, nullptr};
  size_t cap[4] = {0, 0, 0, 0};
  ~HostScratch() {
    for (void* b : buf) if (b) cudaFree(b);
    if (st) cudaStreamDestroy(st);
  }
  bool reserve(int i, size_t bytes) {
    if (bytes <= cap[i]) return true;
    if (buf[i]) { cudaFree(buf[i]); buf[i] = nullptr; cap[i] = 0; }
    const size_t want = bytes + bytes / 4;
    if (cudaMalloc(&buf[i], want) != cudaSuccess) return false;
    cap[i] = want;
    return true;
  }
};

static int run_host(int mode, const pt_table* tb, const double* h_times, int64_t n_t, int64_t t_stride_pv,
                    const double* h_params, int64_t n_pv, int n_pb, int n_ss, double t_exp, int dtype, void* h_flux,
                    int32_t* h_status) {
  // every argument error is reported before anything is allocated or enqueued
  int rc = check_common(h_times, h_params, h_flux, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  if (dtype != PT_F64 && dtype != PT_F32 && dtype != PT_F32S) return PT_ERR_DTYPE;
  if (mode == 1 && !table_ok(tb)) return PT_ERR_TABLE;
  if (plan_tiles(n_pv, n_t, sm_count()).tile_len == 0) return PT_ERR_SIZE;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return PT_ERR_CUDA;
  static thread_local HostScratch scratch[64];      // one per device: the stream belongs to the device it was created on
  HostScratch& S = scratch[dev];
  if (!S.st && cudaStreamCreateWithFlags(&S.st, cudaStreamNonBlocking) != cudaSuccess) return PT_ERR_CUDA;
  const size_t nb_t = sizeof(double) * (size_t)(t_stride_pv == 0 ? n_t : (n_pv - 1) * t_stride_pv + n_t);
  const size_t nb_p = sizeof(double) * (size_t)n_pv * (6 + 3 * (size_t)n_pb);
  const size_t nb_f = (dtype == PT_F64 ? 8 : 4) * (size_t)n_pv * n_pb * n_t;
  if (!(S.reserve(0, nb_t) && S.reserve(1, nb_p) && S.reserve(2, nb_f) && S.reserve(3, 8))) {
    (void)cudaGetLastError();
    return PT_ERR_CUDA;
  }
  cudaStream_t st = S.st;
  double* d_t = (double*)S.buf[0];
  double* d_p = (double*)S.buf[1];
  void* d_f = S.buf[2];
  int32_t* d_s = (int32_t*)S.buf[3];
  cudaMemcpyAsync(d_t, h_times, nb_t, cudaMemcpyHostToDevice, st);
  cudaMemcpyAsync(d_p, h_params, nb_p, cudaMemcpyHostToDevice, st);
  cudaMemsetAsync(d_s, 0, 8, st);
  rc = launch_flux(mode, tb, d_t, n_t, t_stride_pv, d_p, n_pv, n_pb, n_ss, t_exp, dtype, d_f, d_s, st);
  if (rc == PT_OK) {
    cudaMemcpyAsync(h_flux, d_f, nb_f, cudaMemcpyDeviceToHost, st);
    if (h_status) cudaMemcpyAsync(h_status, d_s, 8, cudaMemcpyDeviceToHost, st);
  }
  if (cudaStreamSynchronize(st) != cudaSuccess && rc == PT_OK) rc = PT_ERR_CUDA;
  return rc;
}

int pt_ma_quad_exact_host(const double* h_times, int64_t n_t, int64_t t_stride_pv, const double* h_params, int64_t n_pv,
                          int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype, void* h_flux, int32_t* h_status) {
  return run_host(0, nullptr, h_times, n_t, t_stride_pv, h_params, n_pv, n_pb, n_ss, t_exp, dtype, h_flux, h_status);
}

int pt_ma_quad_interp_host(const pt_table* table, const double* h_times, int64_t n_t, int64_t t_stride_pv,
                           const double* h_params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp,
                           int32_t dtype, void* h_flux, int32_t* h_status) {
  return run_host(1, table, h_times, n_t, t_stride_pv, h_params, n_pv, n_pb, n_ss, t_exp, dtype, h_flux, h_status);
}

}  // extern "C"
