// pt_kernels.cu — sm_100a kernels and the C ABI of include/pt.h.
//
// The fused flux kernel (whole hot path in one persistent launch) lives in pt_flux.cuh; this file holds the orbit-only
// kernel, the table builder, the FP64 probe and the host side of the C ABI.
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/pt.h"
#include "pt_flux.cuh"

namespace pt {

static std::atomic<int64_t> g_launches{0};

// Scheduler slots of the flux kernel (tile counters + finished-warp counter each).  A launch takes the next slot in a ring;
// the kernel leaves its slot zeroed when it ends, so a slot is clean again long before the ring comes back to it (that
// would need kSchedSlots launches in flight at once).  This is the only state the library keeps on the device.
constexpr int kSchedSlots = 64;
constexpr int kSchedWords = 1024;   // [0] global ticket, [1] finished warps, [2 + pv] per-parameter-vector tickets
constexpr int kPvCacheMax = 512;    // parameter-vector records a slot can hold (pv_cache_kernel)
struct SchedSlot {
  unsigned long long w[kSchedWords];
  PvRec pv[kPvCacheMax];
};
__device__ SchedSlot g_sched[kSchedSlots];
static std::atomic<uint64_t> g_sched_seq{0};

static SchedSlot* sched_slot() {
  static std::atomic<SchedSlot*> base[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  SchedSlot* b = base[dev].load();
  if (!b) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_sched) != cudaSuccess) return nullptr;
    b = (SchedSlot*)p;
    base[dev].store(b);
  }
  return b + (g_sched_seq.fetch_add(1) % kSchedSlots);
}

// S1-S2 alone: signed projected separation of every subsample.
__global__ void __launch_bounds__(kThreads) orbit_kernel(const double* __restrict__ times, int64_t n_t,
                                                         int64_t t_stride_pv, const double* __restrict__ params,
                                                         int n_pb, int n_ss, double t_exp, double* __restrict__ z_out,
                                                         int blocks_per_pv) {
  __shared__ PvConst c;
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
  }
  __syncthreads();
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
      z = orbit_z_signed(c, fold_phase(ts, c.t0, c.P, c.invP, c.flags & PV_SLOWDIV));
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

// Fused likelihood, step 1: chi2 of the all-out-of-transit model, sum over (passband, exposure) of ((obs - 1) / sigma)².
// Block b reduces a contiguous range in a fixed order (strided per-thread sums, then a shared-memory tree) and writes one
// partial; the flux kernel adds the partials, again in a fixed order, to every parameter vector.  Also zeroes chi2[].
constexpr int kBaseBlocks = 128;
__global__ void __launch_bounds__(kThreads) chi2_base_kernel(const double* __restrict__ obs, const double* __restrict__ isig,
                                                             int64_t n, double* __restrict__ part, double* __restrict__ chi2,
                                                             int64_t n_pv) {
  __shared__ double s_sum[kThreads];
  asm volatile("griddepcontrol.launch_dependents;");   // the record kernel does not read this kernel's output
  const int64_t per = (n + gridDim.x - 1) / gridDim.x;
  const int64_t lo = (int64_t)blockIdx.x * per, hi = min(lo + per, n);
  double acc = 0.0;
  for (int64_t i = lo + threadIdx.x; i < hi; i += kThreads) {
    const double d = (__ldg(obs + i) - 1.0) * __ldg(isig + i);
    acc = fma(d, d, acc);
  }
  s_sum[threadIdx.x] = acc;
  __syncthreads();
  for (int o = kThreads / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[blockIdx.x] = s_sum[0];
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n_pv; i += (int64_t)gridDim.x * kThreads) chi2[i] = 0.0;
}

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

// ------------------------------------------------------------------------------------------------ host side
static int check_common(const void* times, const void* params, const void* out, int64_t n_t, int64_t t_stride_pv,
                        int64_t n_pv, int n_pb, int n_ss) {
  if (!times || !params || !out) return PT_ERR_NULL;
  if (n_t <= 0 || n_pv <= 0 || n_pb < 1 || n_ss < 1 || n_pb > kMaxPassbands) return PT_ERR_SIZE;
  if (t_stride_pv != 0 && t_stride_pv < n_t) return PT_ERR_SIZE;
  return PT_OK;
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
struct Plan {
  int tile_len;
  int64_t tiles_per_pv;
  int mode;
  int64_t blocks;
};
#ifndef PT_LPT_TILE
#define PT_LPT_TILE 256
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
  int64_t tpp = (n_t + tl - 1) / tl;
  const bool few = (n_pv <= kSchedWords - 2 - kBaseBlocks && tpp >= 2);   // the slot's tail holds the chi2 partials
  p.mode = few ? 1 : 0;
  if (few && n_pv <= kLptMax && n_pv * tpp >= 2 * warps) {   // worth ranking the rows only with several tiles per warp
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
constexpr int kDtypeChi2 = 2;   // internal: d_flux is chi2[n_pv], `like` holds the observations

static int launch_flux(int mode, const pt_table* tb, const double* d_times, int64_t n_t, int64_t t_stride_pv,
                       const double* d_params, int64_t n_pv, int n_pb, int n_ss, double t_exp, int dtype, void* d_flux,
                       int32_t* d_status, cudaStream_t st, const Chi2Args* like = nullptr, int pb_view = -1, int n_pb_row = 0) {
  int rc = check_common(d_times, d_params, d_flux, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  if (dtype != PT_F64 && dtype != PT_F32 && !(dtype == kDtypeChi2 && like)) return PT_ERR_DTYPE;
  FluxArgs A{};
  A.times = d_times; A.n_t = n_t; A.t_stride_pv = t_stride_pv; A.params = d_params; A.n_pv = n_pv;
  A.n_pb = n_pb; A.n_ss = n_ss; A.t_exp = t_exp; A.flux = d_flux; A.status = d_status;
  A.row_stride = 6 + 3 * (int64_t)n_pb; A.pb_first = 0; A.flux_pv_stride = (int64_t)n_pb * n_t; A.flux_off = 0;
  A.pbk = (pb_view == -2) ? 1 : 0;
  if (pb_view >= 0) {   // single-passband view of passband `pb_view` in rows of n_pb_row passbands
    A.row_stride = 6 + 3 * (int64_t)n_pb_row; A.pb_first = pb_view;
    A.flux_pv_stride = (int64_t)n_pb_row * n_t; A.flux_off = (int64_t)pb_view * n_t;
  }
  if (mode == 1) {
    if (!tb || !tb->d_data || tb->n_k < 2 || tb->n_z < 2 || (tb->n_fn != 3 && tb->n_fn != 4) || !(tb->dk > 0.0) ||
        !(tb->dz > 0.0) || (tb->dtype != PT_F64 && tb->dtype != PT_F32))
      return PT_ERR_TABLE;
    A.tb = tb->d_data; A.tb_dtype = tb->dtype; A.n_k = tb->n_k; A.n_z = tb->n_z; A.n_fn = tb->n_fn;
    A.k_min = tb->k_min; A.dk = tb->dk; A.dz = tb->dz;
  }
  const pt::Plan plan = plan_tiles(n_pv, n_t, sm_count());
  if (plan.tile_len == 0) return PT_ERR_SIZE;
  A.tile_len = plan.tile_len; A.tiles_per_pv = (int)plan.tiles_per_pv; A.n_tiles = n_pv * plan.tiles_per_pv;
  A.per_pv = plan.mode == 1; A.lpt = plan.mode == 2;
  int lg = 0;
  while (((int64_t)1 << lg) < (int64_t)n_ss) ++lg;
  A.fx_bits = 61 - lg;
  A.fx_scale = ldexp(1.0, A.fx_bits);
  A.fx_inv = 1.0 / (A.fx_scale * (double)n_ss);
  A.inv_nss = 1.0 / (double)n_ss;
  const dim3 grid((unsigned)plan.blocks);
  SchedSlot* slot = sched_slot();
  if (!slot) return PT_ERR_CUDA;
  A.sched = slot->w;
  // single passband, few parameter vectors, many tiles each: the per-vector records are computed once, by a small kernel
  // in front of the flux kernel (the setup is 15 % of the flux kernel's instructions on configs[1] when done per tile)
  if (n_pb == 1 && pb_view < 0 && n_pv <= kPvCacheMax && A.n_tiles >= 8 * n_pv) {
    const unsigned nb = (unsigned)((n_pv + kWarpsPerBlock - 1) / kWarpsPerBlock);
    // fused likelihood: the record kernel overlaps chi2_base_kernel (it waits for it only before it exits, so that the
    // flux kernel, which waits for the record kernel, also sees the baseline)
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t c2{};
    c2.gridDim = dim3(nb); c2.blockDim = dim3(kThreads); c2.dynamicSmemBytes = 0; c2.stream = st;
    c2.attrs = at; c2.numAttrs = (dtype == kDtypeChi2) ? 1 : 0;
    if (mode == 0) cudaLaunchKernelEx(&c2, pv_cache_kernel<0>, A, slot->pv);
    else cudaLaunchKernelEx(&c2, pv_cache_kernel<1>, A, slot->pv);
    A.pvcache = slot->pv;
    g_launches.fetch_add(1);
  }
  if (dtype == kDtypeChi2) {
    // step 1 of the fused likelihood: out-of-transit baseline into the tail of the scheduler slot, chi2[] zeroed
    double* part = reinterpret_cast<double*>(A.sched + kSchedWords - kBaseBlocks);
    const int64_t n_obs = (int64_t)n_pb * n_t;
    int nb = (int)((n_obs + 4095) / 4096);
    if (nb > kBaseBlocks) nb = kBaseBlocks;
    if (nb < 1) nb = 1;
    chi2_base_kernel<<<nb, kThreads, 0, st>>>(like->obs, like->isig, n_obs, part, (double*)d_flux, n_pv);
    g_launches.fetch_add(1);
    A.obs = like->obs; A.isig = like->isig; A.chi2 = (double*)d_flux; A.base_part = part; A.n_base_part = nb;
    A.flux = nullptr;
  }
  // 16-byte loads/stores need even row lengths/strides and 16-byte aligned bases
  const bool v2 = (n_t % 2 == 0) && (t_stride_pv % 2 == 0) && (reinterpret_cast<uintptr_t>(d_times) % 16 == 0) &&
                  (dtype == kDtypeChi2 || reinterpret_cast<uintptr_t>(d_flux) % 16 == 0);
  const bool p1 = (n_pb == 1), s1 = (n_ss == 1);
  // with the record cache the flux kernel is launched as a programmatic dependent of pv_cache_kernel: its launch and its
  // prologue (row ranking) overlap that kernel, and it waits (griddepcontrol.wait) before it reads the first record
  cudaLaunchAttribute pdl_attr[1];
  pdl_attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl_attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cfg.attrs = pdl_attr; cfg.numAttrs = A.pvcache ? 1 : 0;
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
  return cudaGetLastError() == cudaSuccess ? PT_OK : PT_ERR_CUDA;
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

int pt_orbit_z(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
               int32_t n_pb, int32_t n_ss, double t_exp, double* d_z, void* stream) {
  int rc = check_common(d_times, d_params, d_z, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  const int64_t n = n_t * n_ss;
  int64_t bpp = (n + (int64_t)kThreads * 8 - 1) / ((int64_t)kThreads * 8);
  const int64_t cap = (148 * 16 + n_pv - 1) / n_pv;
  if (bpp > cap) bpp = cap;
  if (bpp < 1) bpp = 1;
  if (n_pv * bpp > 0x7fffffff) return PT_ERR_SIZE;
  orbit_kernel<<<(unsigned)(n_pv * bpp), kThreads, 0, (cudaStream_t)stream>>>(d_times, n_t, t_stride_pv, d_params, n_pb,
                                                                              n_ss, t_exp, d_z, (int)bpp);
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

int pt_ma_table_build(double k_min, double k_max, int32_t n_k, double z_max, int32_t n_z, int32_t dtype, int32_t n_fn,
                      void* d_table, void* stream) {
  if (!d_table) return PT_ERR_NULL;
  if (n_k < 2 || n_z < 2 || (n_fn != 3 && n_fn != 4) || !(k_max > k_min) || !(k_min >= 0.0) || !(z_max > 0.0))
    return PT_ERR_SIZE;
  if (dtype != PT_F64 && dtype != PT_F32) return PT_ERR_DTYPE;
  const double dk = (k_max - k_min) / (double)(n_k - 1), dz = z_max / (double)(n_z - 1);
  const int64_t n = (int64_t)n_k * n_z;
  int64_t blocks = (n + kThreads - 1) / kThreads;
  if (blocks > 148 * 64) blocks = 148 * 64;
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

// ---- host-buffer forms: H2D, kernels, D2H on an internal stream, then wait.
static int run_host(int mode, const pt_table* tb, const double* h_times, int64_t n_t, int64_t t_stride_pv,
                    const double* h_params, int64_t n_pv, int n_pb, int n_ss, double t_exp, int dtype, void* h_flux,
                    int32_t* h_status) {
  int rc = check_common(h_times, h_params, h_flux, n_t, t_stride_pv, n_pv, n_pb, n_ss);
  if (rc) return rc;
  if (dtype != PT_F64 && dtype != PT_F32) return PT_ERR_DTYPE;
  static thread_local cudaStream_t st = nullptr;
  if (!st) {
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) return PT_ERR_CUDA;
    // keep the stream-ordered scratch in the pool between calls (the default hands it back at every synchronisation)
    int dev = 0;
    cudaMemPool_t pool;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      uint64_t keep = UINT64_MAX;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
  }
  const size_t nb_t = sizeof(double) * (size_t)(t_stride_pv == 0 ? n_t : (n_pv - 1) * t_stride_pv + n_t);
  const size_t nb_p = sizeof(double) * (size_t)n_pv * (6 + 3 * (size_t)n_pb);
  const size_t nb_f = (dtype == PT_F64 ? 8 : 4) * (size_t)n_pv * n_pb * n_t;
  double *d_t = nullptr, *d_p = nullptr;
  void* d_f = nullptr;
  int32_t* d_s = nullptr;
  bool ok = cudaMallocAsync(&d_t, nb_t, st) == cudaSuccess && cudaMallocAsync(&d_p, nb_p, st) == cudaSuccess &&
            cudaMallocAsync(&d_f, nb_f, st) == cudaSuccess && cudaMallocAsync(&d_s, 8, st) == cudaSuccess;
  if (ok) {
    cudaMemcpyAsync(d_t, h_times, nb_t, cudaMemcpyHostToDevice, st);
    cudaMemcpyAsync(d_p, h_params, nb_p, cudaMemcpyHostToDevice, st);
    cudaMemsetAsync(d_s, 0, 8, st);
    rc = launch_flux(mode, tb, d_t, n_t, t_stride_pv, d_p, n_pv, n_pb, n_ss, t_exp, dtype, d_f, d_s, st);
    if (rc == PT_OK) {
      cudaMemcpyAsync(h_flux, d_f, nb_f, cudaMemcpyDeviceToHost, st);
      if (h_status) cudaMemcpyAsync(h_status, d_s, 8, cudaMemcpyDeviceToHost, st);
    }
  } else {
    rc = PT_ERR_CUDA;
  }
  if (d_t) cudaFreeAsync(d_t, st);
  if (d_p) cudaFreeAsync(d_p, st);
  if (d_f) cudaFreeAsync(d_f, st);
  if (d_s) cudaFreeAsync(d_s, st);
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
