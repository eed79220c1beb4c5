/* pt.h — C ABI of the B200-native batched quadratic Mandel–Agol transit-model evaluator.
 *
 * The method is the one PyTransit (Parviainen 2015, arXiv 1504.07433) implements; "P:Ln" cites line n of the paper's
 * text, DESIGN.md §2 lists the readings taken where the paper is silent or garbled.
 *
 *   flux  f(k,z) = 1 - [(1-c) λe(k,z) + c λd(k,z) + b ηd(k,z)] / (1 - a/3 - b/6),  c = a + 2b          P:L136 (Eq. 13)
 *   (a,b) = (u1,u2): quadratic limb darkening  I(μ)/I(1) = 1 - a(1-μ) - b(1-μ)²                        P:L86  (Eq. 6)
 *   λe, λd, ηd: Mandel & Agol (2002) basis functions, independent of limb darkening
 *   "λd" is the continuous function λd + (2/3)Θ(k-z) (Eq. 13 prints no Θ term; R3)
 *
 * Conventions common to every entry point
 *   - Pointers named d_* are DEVICE pointers (e.g. torch tensor .data_ptr()); pointers named h_* are HOST pointers.
 *     The caller owns all of them.  The d_* entry points never allocate, free, copy to the host or synchronise: they
 *     validate their arguments, enqueue kernels on `stream` (a cudaStream_t passed as void*; NULL = default stream)
 *     and return.  They are re-entrant (any thread, any stream).  The only state the library keeps is a set of
 *     scheduler slots in device memory per device (work counters of the persistent kernels, and room for the records,
 *     row order and transit epochs of up to 4096 parameter vectors).  A launch takes a slot and leaves its counters
 *     zeroed; 16 slots are shared round-robin, each guarded by an event recorded behind the launch that holds it, and a
 *     launch that finds all of them in flight makes `stream` wait for the oldest (cudaStreamWaitEvent: ordering on the
 *     device, no host synchronisation), so two live launches never share one whatever the number of streams.  A launch
 *     made while `stream` is being captured into a CUDA graph takes one of 8 further slots for good and makes no CUDA
 *     call other than the kernel launches; when those are used up, capturing returns PT_ERR_CUDA.
 *   - Parameter rows (`d_params`, row-major [n_pv][6 + 3 n_pb] doubles):
 *         [ t0, P, a/R*, i, e, w,  k_0, u1_0, u2_0,  k_1, u1_1, u2_1, ... ]
 *     t0 = time of inferior conjunction, P = period (same unit as the times), a/R* = scaled semi-major axis,
 *     i = inclination and w = argument of periastron in RADIANS, e = eccentricity in [0,1), per passband j the
 *     radius ratio k_j = R_planet/R_star and the two limb-darkening coefficients.  n_pb = 1 is the 9-vector
 *     [t0,P,a/R*,i,e,w,k,u1,u2].  The orbit equations are not in the paper (P:L31 names the solvers): standard
 *     two-body projection, observer on +Z, transit at true anomaly π/2 - w (R5); e == 0 selects the circular
 *     routine, e > 0 the Newton–Kepler solver ("selects the most appropriate orbit calculation routine based on
 *     the eccentricity").
 *   - Times: `d_times` holds n_t doubles shared by all parameter vectors when t_stride_pv == 0, else row pv starts at
 *     d_times + pv * t_stride_pv (t_stride_pv >= n_t).
 *   - Supersampling: every exposure is the mean of n_ss model values at the midpoints of n_ss equal
 *     sub-intervals of [t - t_exp/2, t + t_exp/2]; n_ss == 1 ignores t_exp.
 *   - Multi-passband: the basis functions are evaluated once per sample at the mean radius ratio
 *     k̂ = (1/n_pb) Σ k_j and combined per passband; each passband's flux decrement is scaled by k_j²/k̂².
 *   - Planet behind the star, z >= 1 + k̂, or k̂ == 0  =>  flux = 1 exactly.
 *   - Return value: PT_OK, or a synchronous argument error (nothing is enqueued or written in that case).
 *     Data errors are asynchronous: a parameter row with a non-finite entry, P <= 0, a/R* <= 0, e outside [0,1), any
 *     k_j < 0 or 1 - u1_j/3 - u2_j/6 == 0 gets its whole output row set to NaN; if d_status != NULL,
 *     PT_ST_BAD_PARAM is OR-ed into d_status[0] and d_status[1] is incremented once per affected row.
 *     d_status (2 x int32) is only ever OR-ed/incremented: the caller zeroes it.
 */
#ifndef PT_H_
#define PT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { PT_OK = 0, PT_ERR_NULL = 1, PT_ERR_SIZE = 2, PT_ERR_DTYPE = 3, PT_ERR_TABLE = 4, PT_ERR_CUDA = 5 };
enum { PT_F64 = 0, PT_F32 = 1, PT_F32S = 2 };
/* Flux dtype.  PT_F64: fp64 arithmetic, double output.  PT_F32: the fp32 VARIANT of BASELINE.json (gate 2e-6 absolute;
 * SURVEY §8(c)-4 H5): float output and fp32 ARITHMETIC from the folded phase on — orbit, case split, λe, λd*, ηd, combine —
 * on the FP32 pipe; the subsample time and the phase fold stay fp64 (a time of ~1e3 d resolves 1e-4 d in fp32).  A
 * parameter vector for which fp32 cannot hold the gate — limb-darkening coefficients that would carry the measured
 * worst-case errors of the fp32 basis functions (λd*: 8e-7) beyond 1.75e-6 in flux, k > 0.7, a/R* > 50 or e > 0.85 —
 * is evaluated in fp64 and only stored as float (a per-vector decision).  fp32 arithmetic exists in pt_ma_quad_exact
 * with one passband; elsewhere (several passbands, pt_ma_quad_exact_pbk, pt_ma_quad_interp) PT_F32 means PT_F32S.
 * PT_F32S: fp64 arithmetic, float storage (half the output traffic).
 * Table dtype (pt_table.dtype, pt_ma_table_build): PT_F64 or PT_F32 = storage type of the nodes (computed in fp64). */
enum { PT_ST_BAD_PARAM = 1, PT_ST_K_OUT_OF_TABLE = 2 };   /* bits OR-ed into d_status[0] */

/* Interpolation table descriptor (host struct holding a device pointer).  Layout [n_k][n_z][n_fn], n_fn = 3
 * (λe, λd, ηd) or 4 (padded with 0); node (i,j) sits at k = k_min + i*dk, z = j*dz (R10). */
typedef struct pt_table {
  const void* d_data;
  int32_t dtype;      /* PT_F64 or PT_F32 storage; values are converted on load */
  int32_t n_k, n_z, n_fn;
  double k_min, dk, dz;
} pt_table;

/* Version / build information: returns the compute capability the kernels were built for (100 => sm_100a). */
int pt_build_arch(void);

/* S1-S2 of the hot path: projected separation of every subsample (P:L31 orbit utilities).
 *   d_z [n_pv][n_t][n_ss] doubles; the sign carries the side: +z planet in front of the star, -z behind it.
 *   Rows with bad parameters are NaN.  n_pb is only needed for the row length. */
int pt_orbit_z(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
               int32_t n_pb, int32_t n_ss, double t_exp, double* d_z, void* stream);

/* The other orbit routines the paper names ("circular and elliptic orbits (using either Newton's method, iteration,
 * or two series approximations) ... selects the most appropriate orbit calculation routine based on the eccentricity";
 * SURVEY §8(f) NEXT-3).  The paper prints no formulas; R19 fixes the reading:
 *   PT_SOLVER_EXACT   e == 0: circular routine, else Newton on Kepler's equation (what pt_orbit_z and every flux entry use)
 *   PT_SOLVER_NEWTON  the same
 *   PT_SOLVER_ITER    fixed-point iteration E <- M + e sin E from E = M, run until E moves by less than an ulp
 *   PT_SOLVER_PS3/5   true anomaly from the classical series of the equation of the centre f - M in powers of e, truncated
 *                     after e^3 / e^5; truncation error in f at most 1.5 e^4 / 2.2 e^6 rad, in z at most a (1+e)/(1-e)
 *                     times that
 *   PT_SOLVER_FAST    by eccentricity: e == 0 circular, e <= 0.006 order 3, e <= 0.03 order 5 (truncation error below
 *                     2e-9 rad in f), else Newton
 * Same arguments, layout and error behaviour as pt_orbit_z; an unknown solver is PT_ERR_SIZE. */
enum { PT_SOLVER_EXACT = 0, PT_SOLVER_NEWTON = 1, PT_SOLVER_ITER = 2, PT_SOLVER_PS3 = 3, PT_SOLVER_PS5 = 4, PT_SOLVER_FAST = 5 };
int pt_orbit_z_solver(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                      int32_t n_pb, int32_t n_ss, double t_exp, int32_t solver, double* d_z, void* stream);

/* S0-S7: exact quadratic Mandel–Agol flux (Eq. 13 with P:L143).
 *   dtype  PT_F64: d_flux is double.  PT_F32 / PT_F32S: d_flux is float (see the enum above).
 *   d_flux [n_pv][n_pb][n_t], time fastest.   d_status: NULL or 2 x int32 (see above). */
int pt_ma_quad_exact(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                     int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype, void* d_flux, int32_t* d_status,
                     void* stream);

/* Exact per-passband-k mode (P:L177-L179 describe the mean-k evaluation above as an approximation):
 * every passband is evaluated with its OWN radius ratio k_j, i.e. flux[pv][j][:] equals pt_ma_quad_exact called with
 * n_pb = 1 on the row [t0,P,a,i,e,w,k_j,u1_j,u2_j].  Same arguments and layout as pt_ma_quad_exact.  n_ss == 1: one fused
 * launch (the orbit once per sample, the basis functions once per passband).  n_ss > 1: one launch per passband on
 * `stream` (the single-passband kernel reads passband j of the wide rows in place; d_status[1] then counts affected
 * (row, passband) pairs). */
int pt_ma_quad_exact_pbk(const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                         int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype, void* d_flux, int32_t* d_status,
                         void* stream);

/* S8: build the (k,z) interpolation table ("precomputed into two-dimensional interpolation tables spanning
 * z = [0..1+k] and k ranges based on the prior set on k").
 *   node (i,j): k = k_min + i*dk, dk = (k_max-k_min)/(n_k-1);  z = j*dz, dz = z_max/(n_z-1)  (IEEE double, mul then add).
 *   Values are computed in fp64 and stored as `dtype`; d_table [n_k][n_z][n_fn], n_fn in {3,4}.
 *   Requires n_k >= 2, n_z >= 2, 0 <= k_min < k_max, z_max > 0. */
int pt_ma_table_build(double k_min, double k_max, int32_t n_k, double z_max, int32_t n_z, int32_t dtype, int32_t n_fn,
                      void* d_table, void* stream);

/* Node spacing of the table pt_ma_table_build builds for these arguments, exactly as the builder forms it in IEEE double:
 * *h_dk = (k_max-k_min)/(n_k-1), *h_dz = z_max/(n_z-1).  Host pointers; this is what belongs in pt_table.dk / .dz. */
int pt_table_spacing(double k_min, double k_max, int32_t n_k, double z_max, int32_t n_z, double* h_dk, double* h_dz);

/* S9 (+S0-S3, S6, S7): interpolated quadratic Mandel–Agol flux ("bilinear interpolation"):
 *   rk = (k̂-k_min)/dk, ik = min(floor(rk), n_k-2), fk = rk-ik; rz = z/dz, iz = min(floor(rz), n_z-2), fz = rz-iz;
 *   v = (1-fk)[(1-fz)T[ik][iz] + fz T[ik][iz+1]] + fk[(1-fz)T[ik+1][iz] + fz T[ik+1][iz+1]] for each function, then
 *   Eq. 13.  Samples with z >= 1+k̂ never touch the table.  `dtype` is the output type as above; the table's
 *   own storage type is in the descriptor.  A parameter vector whose k̂ lies outside [k_min, k_min+(n_k-1)dk] is
 *   evaluated by the exact device path and PT_ST_K_OUT_OF_TABLE is raised (paper silent; R13).
 *   PT_ERR_TABLE: descriptor inconsistent (NULL data, n_k/n_z < 2, n_fn not 3/4, dk/dz <= 0, unknown dtype). */
int pt_ma_quad_interp(const pt_table* table, const double* d_times, int64_t n_t, int64_t t_stride_pv,
                      const double* d_params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype,
                      void* d_flux, int32_t* d_status, void* stream);

/* Fused likelihood (the paper's "offload z and likelihood to the GPU" variant):
 *   chi2[pv] = sum over passbands j and exposures t of ((obs[j][t] - F_pv[j][t]) * isig[j][t])²
 * with F the flux of pt_ma_quad_exact (table == NULL) or pt_ma_quad_interp (table != NULL); no flux is written.
 *   d_obs, d_isig  [n_pb][n_t] doubles: observed flux and 1/sigma, ONE data set shared by all parameter vectors (the MCMC
 *                  case); d_times [n_t] is shared as well.
 *   d_chi2         [n_pv] doubles, overwritten.  A row with bad parameters gets NaN (+ PT_ST_BAD_PARAM).
 * The sum is formed as the all-out-of-transit value plus, per in-window exposure, the correction
 * (1-F) w² (2 (o-1) + (1-F)): exposures that cannot be in transit cost one window test and no memory traffic.
 * Corrections are added with floating-point atomics, so chi2 is reproducible to rounding (~1e-16 relative), not bitwise. */
int pt_ma_quad_chi2(const pt_table* table, const double* d_times, int64_t n_t, const double* d_params, int64_t n_pv,
                    int32_t n_pb, int32_t n_ss, double t_exp, const double* d_obs, const double* d_isig, double* d_chi2,
                    int32_t* d_status, void* stream);

/* Host-buffer convenience forms (the end-to-end path of P:L173/P:L198: copy inputs to the GPU, evaluate, copy the
 * flux back).  All pointers are HOST pointers (pinned memory makes the copies asynchronous); the call allocates
 * stream-ordered scratch on the current device, enqueues H2D copies, the same kernels as above and the D2H copy on an
 * internal stream, and returns after that stream has drained.  h_status: NULL or 2 x int32, overwritten.
 * pt_ma_quad_interp_host takes the table as a descriptor whose d_data is still a DEVICE pointer (tables are built once
 * and stay resident). */
int pt_ma_quad_exact_host(const double* h_times, int64_t n_t, int64_t t_stride_pv, const double* h_params, int64_t n_pv,
                          int32_t n_pb, int32_t n_ss, double t_exp, int32_t dtype, void* h_flux, int32_t* h_status);
int pt_ma_quad_interp_host(const pt_table* table, const double* h_times, int64_t n_t, int64_t t_stride_pv,
                           const double* h_params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp,
                           int32_t dtype, void* h_flux, int32_t* h_status);

/* The Giménez transit model (Eq. 1-12): general limb darkening
 *   I(μ)/I(1) = 1 - Σ_{n=1}^{N} u_n (1 - μ^n) (Eq. 4),   f = 1 - Σ_{n=0}^{N} C_n α_n(b,c), b = k/(1+k), c = z/(1+k) (Eq. 1, 2),
 *   α_n = b² (1-c²)^{ν+1} Σ_{j=0}^{n_j} A_{n,j} G_j(ν+2,ν+1;1-b)² G_j(ν+2,1;c²), ν = (n+2)/2 (Eq. 3, 10, 11), C_n from Eq. 7-8,
 * with the paper's two optimisations: the α_n are evaluated once per sample and combined per passband (Eq. 9), and the
 * coefficients A_{n,j} and those of the polynomial recurrence are precomputed into a table.  G_j(p,q;x) are
 * Kopal's Jacobi polynomials 2F1(-j, j+p; q; x) (R20: the paper does not define them).  n_j + 1 terms are summed
 * (j = 0..n_j); the truncation error falls slowly and oscillates (~1e-5 at n_j = 40, ~1e-6 at 100).
 *   Parameter rows [n_pv][7 + n_pb*n_ldc]: [t0, P, a/R*, i, e, w, k,  u_1..u_N (passband 0), u_1..u_N (passband 1), ...]
 *   (one radius ratio; the quadratic law (a, b) is u_1 = a + 2b, u_2 = -b).  Orbit, supersampling, flux layout
 *   [n_pv][n_pb][n_t] (double), d_status and bad rows (also 1 - Σ n u_n/(n+2) == 0) as for pt_ma_quad_exact.
 *   Limits: n_ldc <= 8, n_j <= 256, n_pb <= 64 (else PT_ERR_SIZE).
 * pt_gimenez_coef_size / pt_gimenez_coef_build: the coefficient table, (n_ldc+1)(n_j+1) x 8 doubles in memory the caller
 *   owns (32-byte aligned), built on the device.
 * pt_gimenez_exact: every in-transit subsample through the series.
 * pt_gimenez_interp: the paper's interpolation in z ("first evaluated for n points for z < 1 - k and m points
 *   for 1 - k < z < k + 1, and the light curve points are interpolated from these tabulated values"; R21): per
 *   parameter vector, every α_n on n_in nodes uniform on [0, 1-k] and n_out nodes uniform on [1-k, 1+k] (both ends
 *   included), linear interpolation inside the segment that holds z.  d_work: [n_pv][n_ldc+1][n_in+n_out] doubles owned by
 *   the caller, filled by the call (one launch) and readable afterwards.  k >= 1 (no inner segment): that row uses the series. */
int pt_gimenez_coef_size(int32_t n_ldc, int32_t n_j, int64_t* h_bytes);
int pt_gimenez_coef_build(int32_t n_ldc, int32_t n_j, double* d_coef, void* stream);
int pt_gimenez_exact(const double* d_coef, int32_t n_ldc, int32_t n_j, const double* d_times, int64_t n_t, int64_t t_stride_pv,
                     const double* d_params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux,
                     int32_t* d_status, void* stream);
int pt_gimenez_interp(const double* d_coef, int32_t n_ldc, int32_t n_j, int32_t n_in, int32_t n_out, double* d_work,
                      const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                      int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux, int32_t* d_status, void* stream);

/* pt_gimenez_interp for callers that cannot allocate device memory (CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): same operation, arguments, results and error codes as pt_gimenez_interp, but the z-tables (its d_work)
 * live in a fixed array inside the library — pt_gimenez_static_work_doubles() = 524288 doubles (4 MiB), held by every
 * device that loads the library until the process ends.  The call allocates nothing (no cudaMalloc / cudaFree, no
 * allocating library routine); d_coef, d_times, d_params, d_flux, d_status stay the caller's.
 *   Limit: n_pv * (n_ldc+1) * (n_in+n_out) <= pt_gimenez_static_work_doubles(), else PT_ERR_SIZE (nothing is enqueued).
 *   The array is shared by every call on the device and keeps the last call's tables; each call first overwrites every node
 *   it will read, so nothing needs clearing, and calls enqueued on ONE stream are safe back to back.  Calls that can overlap
 *   on the GPU (different streams, different host threads, concurrently replayed graphs) race on it: the caller serialises
 *   them.  The tables are not readable by the caller. */
int64_t pt_gimenez_static_work_doubles(void);
int pt_gimenez_interp_static(const double* d_coef, int32_t n_ldc, int32_t n_j, int32_t n_in, int32_t n_out,
                             const double* d_times, int64_t n_t, int64_t t_stride_pv, const double* d_params, int64_t n_pv,
                             int32_t n_pb, int32_t n_ss, double t_exp, double* d_flux, int32_t* d_status, void* stream);

/* Diagnostics for the roofline denominator (the FP64 vector-pipe peak is not in MEASURED_PEAKS.json):
 * every thread of `blocks` x 256 runs `iters` rounds of 8 independent DFMA chains and stores one double to
 * d_sink[blocks*256] so the work cannot be removed.  FP64 thread-instructions issued = blocks*256*iters*8. */
int pt_probe_dfma(int32_t blocks, int32_t iters, double* d_sink, void* stream);
/* The same for the FP32 pipe (roofline denominator of the fp32 variant): FFMA chains, d_sink: blocks*256 floats. */
int pt_probe_ffma(int32_t blocks, int32_t iters, float* d_sink, void* stream);

/* How the flux kernels would cut up a problem on a device with n_sm multiprocessors (pure host logic, no CUDA call; used
 * by the CPU tests).  h_out[0] = exposures per tile, [1] = tiles per parameter vector, [2] = scheduling mode (0 global
 * tile counter, 1 one counter per parameter vector, 2 global counter with rows in longest-processing-time-first order),
 * [3] = blocks of 256 threads in the persistent grid. */
int pt_plan(int64_t n_pv, int64_t n_t, int32_t n_sm, int64_t* h_out);

/* Number of kernel launches the library has enqueued so far in this process (bench.py's gpu_launches evidence). */
int64_t pt_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* PT_H_ */
