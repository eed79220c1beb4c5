"""bench.py — Mandel–Agol flux evaluations per second on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A step is one pass of the whole hot path (per-pv setup, supersample expansion, phase fold, orbit, case split, basis
functions, limb-darkening combine, supersample mean, store) over one batch of BASELINE.json configs[1] (Kepler
long-cadence-like: 64 parameter vectors x 60000 exposures x 10 supersamples, circular, fp64).  N > 1 (torchrun): every
rank evaluates its own seeded population of the same shape (weak scaling, no data-path collective).
Extra objects on the same line: `interp` (configs[3], table build + interpolated path, HBM roofline), `dense`
(every sample in transit, eccentric: the FP64-bound regime), `scaled` (configs[1] at 448 parameter vectors),
`roofline`, `cpu_baseline`, `e2e`, `clocks`.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Mandel-Agol flux evals/sec (fp64 exact)"
UNIT = "evals/s"
WORKLOAD = "BASELINE.json configs[1]: 64 pv x 60000 exposures x 10 supersamples, circular, 1 passband, fp64"

# Algorithmic FP64 thread-instructions per unit of work.
ALG_PER_EXPOSURE = 30.0       # phase fold + window test
ALG_PER_COMBINE = 5.0         # per (exposure, passband): 3 FMA + mul + sub
ALG_PER_TRANSIT_CIRC = 650.0  # in-transit subsample, circular orbit: z + case split + λe, λd, ηd
ALG_PER_TRANSIT_ECC = 900.0   # the same with the Newton–Kepler solve
FP64_LANES_PER_SM, FP32_LANES_PER_SM, N_SM = 64, 128, 148
# What the hardware executed, from the committed ncu captures of the same workloads (profiles/r2_ncu_*.md; one launch each):
#   fp64_inst  smsp__sass_thread_inst_executed_op_{dadd,dmul,dfma}_pred_on.sum (thread-instructions)
#   pipe_pct   sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active
#   dram       dram__bytes_read.sum + dram__bytes_write.sum (a kernel's output that is still in L2 when the capture ends
#              is not in its figure: configs[1] writes 30.7 MB < 126 MB L2)
CAPTURES = {
    "exact_config2": {"fp64_inst": 319160231.0, "pipe_pct": 48.5, "dram": 551680.0, "kernel": "epoch_kernel<0,32,1,0,double>", "ncu_us": 71.5},
    "scaled": {"fp64_inst": 1995302341.0, "pipe_pct": 58.9, "dram": 159538688.0, "kernel": "epoch_kernel<0,32,1,0,double>", "ncu_us": 329.6},
    "dense": {"fp64_inst": 4348782966.0, "pipe_pct": 64.2, "dram": 222173184.0, "kernel": "flux_kernel<0,2,1,1,double>", "ncu_us": 444.7},
    "dense_f32": {"fp64_inst": 311909426.0, "pipe_pct": 9.3, "dram": 173787136.0, "kernel": "direct_kernel<2,float,3>", "ncu_us": 268.4, "fp32_inst": 2231589904.0},
    "interp_f32": {"fp64_inst": 710701664.0, "pipe_pct": 7.7, "dram": 3294375512.0, "kernel": "epoch_kernel<1,512,1,1,double>", "ncu_us": 636.6},
    "interp_f64": {"fp64_inst": 710701664.0, "pipe_pct": 7.4, "dram": 3320690688.0, "kernel": "epoch_kernel<1,512,1,1,double>", "ncu_us": 658.5},
    "config3": {"fp64_inst": 64586338.0, "pipe_pct": 11.8, "dram": 1892352.0, "kernel": "flux_kernel<0,2,0,1,double>", "ncu_us": 51.7},
    "config5": {"fp64_inst": 4698671109.0, "pipe_pct": 64.3, "dram": 222058752.0, "kernel": "flux_kernel<0,2,1,1,double>", "ncu_us": 478.1},
}
CAPTURE_SOURCE = "profiles/r2_ncu_*.md (ncu --set full + sass op counters, one launch of the same workload)"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": float(p["hbm_gbs"]), "sm_max_mhz": float(p.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period, self.stop_flag = index, period, threading.Event()
        self.sm, self.reasons, self.max_sm = [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_sm = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
        while not self.stop_flag.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for n, bit in names.items():
                    if r & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_sm,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def _dist_setup(n_gpus: int):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def _max_over_ranks(x: float, world: int, device) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def _barrier(world: int):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def _time_steps(fn, steps: int, warmup: int, flush, world: int):
    """Per-step CUDA-event timing on the current stream; L2 is flushed between steps outside the event pairs.
    Returns total seconds over `steps` steps (this rank)."""
    import torch
    for _ in range(warmup):
        if flush is not None:
            flush()
        fn()
    _barrier(world)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        if flush is not None:
            flush()
        a.record()
        fn()
        b.record()
    _barrier(world)
    return sum(a.elapsed_time(b) for a, b in ev) * 1e-3


def _count_units(pt, w, d_times, d_params):
    """Units of work of one launch, counted with the product's own orbit stage (outside the timed region)."""
    import torch
    z = pt.pt_orbit_z(d_times, d_params, w.n_pb, w.n_ss, w.t_exp)
    khat = d_params[:, 6::3].mean(dim=1)
    in_tr = (z >= 0) & (z < (1.0 + khat)[:, None, None])
    n_in = int(in_tr.sum().item())
    del z, in_tr
    torch.cuda.empty_cache()
    return n_in


def _alu_roofline(alg_inst, t_s, peak_model, peak_meas, cap, n_in=None, pipe="fp64"):
    """Roofline object of an ALU-bound kernel: `frac` is the agreed algorithmic count (SURVEY §8(d) instructions per unit
    x units) over time over the model peak; `frac_executed` is what the hardware executed (thread-instructions of the
    committed ncu capture of this workload) over the live time over the same peak; `pipe_pct` the pipe-busy counter of
    that capture.  The algorithmic count is a static SASS count of library calls; the kernels do the same mathematics in
    fewer instructions, so `frac` can exceed the executed fraction — and 1: flagged then."""
    ach = alg_inst / t_s
    r = {"bound": "alu", "achieved": ach * 2 / 1e12, "peak": peak_model * 2 / 1e12, "unit": "TFLOP/s",
         "frac": ach / peak_model, "alg_%s_inst_per_launch" % pipe: alg_inst,
         "peak_source": "model: 148 SM x %d %s lanes x sm_max_mhz x 2 flop (DESIGN.md §6)" % (
             FP64_LANES_PER_SM if pipe == "fp64" else FP32_LANES_PER_SM, pipe.upper()),
         "%s_peak_measured_tflops" % pipe: peak_meas * 2 / 1e12, "frac_of_measured_peak": ach / peak_meas}
    if r["frac"] > 1.0 or r["frac_of_measured_peak"] > 1.0:
        r["frac_flag"] = ("algorithmic count exceeds what the pipe can execute: the kernel needs fewer instructions per unit "
                          "than SURVEY §8(d) counts; read frac_executed")
    ex = cap.get("%s_inst" % pipe) if cap else None
    if ex is not None:
        r["%s_inst_executed" % pipe] = ex
        r["frac_executed"] = ex / t_s / peak_model
        r["pipe_fp64_pct"] = cap.get("pipe_pct")
        r["executed_source"] = CAPTURE_SOURCE
    r["traffic"] = cap.get("dram") if cap else None
    r["kernel"] = cap.get("kernel") if cap else None
    if n_in is not None:
        r["in_transit_evals"] = n_in
    return r


def _hbm_roofline(bytes_alg, t_s, peaks, cap):
    return {"bound": "hbm", "achieved": bytes_alg / t_s / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
            "frac": bytes_alg / t_s / 1e9 / peaks["hbm_gbs"], "traffic": cap.get("dram") if cap else None,
            "kernel": cap.get("kernel") if cap else None, "peak_source": peaks["source"], "alg_bytes_per_launch": bytes_alg}


def run_ours(args):
    import torch

    import paper_1504_07433_b200 as pt
    from paper_1504_07433_b200 import build as cuda_build, inputs
    rank, world, local = _dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if rank == 0:
        cuda_build.build()
    _barrier(world)
    peaks = _peaks()
    fp64_model_peak = N_SM * FP64_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6   # FP64 thread-instructions / s
    fp32_model_peak = N_SM * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6

    def to_dev(x):
        return torch.from_numpy(np.ascontiguousarray(x)).to(dev)

    flush_buf = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)   # 256 MiB > 126 MB L2

    def flush():
        flush_buf.fill_(1.0)

    # ------------------------------------------------------------------ headline: configs[1], one population per rank
    w = inputs.config2(stream=rank)
    d_t, d_p = to_dev(w.times), to_dev(w.params)
    out = torch.empty((w.n_pv, w.n_pb, w.n_t), dtype=torch.float64, device=dev)
    n_in = _count_units(pt, w, d_t, d_p)

    def step():
        pt.pt_ma_quad_exact(d_t, d_p, w.n_pb, w.n_ss, w.t_exp, out=out)

    sampler = ClockSampler(local)
    sampler.start()
    l0 = pt.pt_launch_count()
    total_s = _time_steps(step, args.steps, args.warmup, flush, world)
    launches = (pt.pt_launch_count() - l0) * args.steps // (args.steps + args.warmup)   # kernels launched by the timed steps
    total_s = _max_over_ranks(total_s, world, dev)
    ms_per_step = total_s / args.steps * 1e3
    value = world * w.n_eval * args.steps / total_s
    kernel_s = total_s / args.steps
    alg_inst = (w.n_pv * w.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE * w.n_pb) + n_in * ALG_PER_TRANSIT_CIRC)

    # ------------------------------------------------------------------ FP64 / FP32 pipe peaks, measured
    sink = torch.empty(N_SM * 16 * 256, dtype=torch.float64, device=dev)
    sink32 = torch.empty(N_SM * 16 * 256, dtype=torch.float32, device=dev)
    iters = 20000
    t_probe = _time_steps(lambda: pt.pt_probe_dfma(N_SM * 16, iters, sink), 5, 2, None, 1) / 5
    fp64_meas_peak = N_SM * 16 * 256 * iters * 8 / t_probe
    t_probe32 = _time_steps(lambda: pt.pt_probe_ffma(N_SM * 16, iters, sink32), 5, 2, None, 1) / 5
    fp32_meas_peak = N_SM * 16 * 256 * iters * 8 / t_probe32
    roofline = _alu_roofline(alg_inst, kernel_s, fp64_model_peak, fp64_meas_peak, CAPTURES["exact_config2"], n_in)
    roofline["hbm_frac"] = w.n_pv * w.n_t * 8.0 / kernel_s / 1e9 / peaks["hbm_gbs"]
    roofline["traffic_source"] = CAPTURE_SOURCE

    # ------------------------------------------------------------------ e2e through the host-buffer C-ABI call
    h_t, h_p = torch.from_numpy(w.times).pin_memory(), torch.from_numpy(w.params).pin_memory()
    h_out = torch.empty((w.n_pv, w.n_pb, w.n_t), dtype=torch.float64).pin_memory()
    h_st = torch.zeros(2, dtype=torch.int32).pin_memory()
    e2e_steps = max(3, min(args.steps, 20))
    for _ in range(3):
        pt.pt_ma_quad_exact_host(h_t, h_p, h_out, w.n_pb, w.n_ss, w.t_exp, status=h_st)
    _barrier(world)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        pt.pt_ma_quad_exact_host(h_t, h_p, h_out, w.n_pb, w.n_ss, w.t_exp, status=h_st)
    _barrier(world)
    e2e_s = _max_over_ranks(time.perf_counter() - t0, world, dev)
    e2e = {"value": world * w.n_eval * e2e_steps / e2e_s, "unit": UNIT,
           "h2d_bytes_per_step": int(h_t.numel() * 8 + h_p.numel() * 8),
           "d2h_bytes_per_step": int(h_out.numel() * 8 + 8), "ms_per_step": e2e_s / e2e_steps * 1e3,
           "api": "pt_ma_quad_exact_host (pinned host buffers; H2D + kernel + D2H inside the call)"}
    sampler.stop_flag.set()
    sampler.join()
    clocks = sampler.result()

    extra = {}
    sections = set(args.sections.split(","))
    if rank == 0 and "scaled" in sections:
        # -------------------------------------------------------------- scaled configs[1] (448 pv, 2.7e8 evals)
        ws = inputs.config2(n_pv=448)
        st, sp = to_dev(ws.times), to_dev(ws.params)
        so = torch.empty((ws.n_pv, 1, ws.n_t), dtype=torch.float64, device=dev)
        n_in_s = _count_units(pt, ws, st, sp)
        t_s = _time_steps(lambda: pt.pt_ma_quad_exact(st, sp, 1, ws.n_ss, ws.t_exp, out=so), 10, 3, flush, 1) / 10
        alg_s = ws.n_pv * ws.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE) + n_in_s * ALG_PER_TRANSIT_CIRC
        extra["scaled"] = {"workload": "configs[1] population x7 (448 pv)", "value": ws.n_eval / t_s, "unit": UNIT,
                           "ms": t_s * 1e3, "in_transit_frac": n_in_s / ws.n_eval,
                           "roofline": _alu_roofline(alg_s, t_s, fp64_model_peak, fp64_meas_peak, CAPTURES["scaled"], n_in_s)}
        del st, sp, so
    if rank == 0 and "dense" in sections:
        # -------------------------------------------------------------- dense: every sample in transit, eccentric
        wd = inputs.dense_transit(n_pv=4096, n_t=4096)
        dt_, dp_ = to_dev(wd.times), to_dev(wd.params)
        do = torch.empty((wd.n_pv, 1, wd.n_t), dtype=torch.float64, device=dev)
        n_in_d = _count_units(pt, wd, dt_, dp_)
        t_d = _time_steps(lambda: pt.pt_ma_quad_exact(dt_, dp_, out=do), 10, 3, flush, 1) / 10
        alg_d = wd.n_pv * wd.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE) + n_in_d * ALG_PER_TRANSIT_ECC
        extra["dense"] = {"workload": "configs[4]-like population, 4096 pv x 4096 per-pv times, all within 0.75 T14, e~U(0,0.6)",
                          "value": wd.n_eval / t_d, "unit": UNIT, "ms": t_d * 1e3, "in_transit_frac": n_in_d / wd.n_eval,
                          "roofline": _alu_roofline(alg_d, t_d, fp64_model_peak, fp64_meas_peak, CAPTURES["dense"], n_in_d)}
        # the fp32 variant on the same workload: fp32 arithmetic from the folded phase on (PT_F32), and fp64 arithmetic with
        # float storage (PT_F32S)
        do32 = torch.empty((wd.n_pv, 1, wd.n_t), dtype=torch.float32, device=dev)
        t_d32 = _time_steps(lambda: pt.pt_ma_quad_exact(dt_, dp_, dtype=torch.float32, out=do32), 10, 3, flush, 1) / 10
        t_d32s = _time_steps(lambda: pt.pt_ma_quad_exact(dt_, dp_, dtype=torch.float32, out=do32, fp32_store_only=True),
                             10, 3, flush, 1) / 10
        r32 = _alu_roofline(alg_d, t_d32, fp32_model_peak, fp32_meas_peak, CAPTURES["dense_f32"], n_in_d, pipe="fp32")
        extra["dense"]["fp32_variant"] = {"value": wd.n_eval / t_d32, "unit": UNIT, "ms": t_d32 * 1e3, "dtype": "f32",
                                          "speedup_vs_fp64": t_d / t_d32, "roofline": r32,
                                          "note": "same algorithmic count as fp64 against the FP32 pipe; the phase fold stays fp64"}
        extra["dense"]["fp32_store_only"] = {"value": wd.n_eval / t_d32s, "unit": UNIT, "ms": t_d32s * 1e3}
        del dt_, dp_, do, do32
        # the opposite regime for the same two kernels: per-row axes that are sparse in transits (configs[1]'s population x 7,
        # every row on its own copy of the axis, n_ss = 1): the direct kernel must not lose to the general one there
        wsp = inputs.config2(n_pv=448)
        rng_sp = np.random.default_rng(5)
        st_ = to_dev(wsp.times[None, :] + rng_sp.uniform(0.0, 0.01, (wsp.n_pv, 1)))
        sp_ = to_dev(wsp.params)
        so64 = torch.empty((wsp.n_pv, 1, wsp.n_t), dtype=torch.float64, device=dev)
        so32 = torch.empty((wsp.n_pv, 1, wsp.n_t), dtype=torch.float32, device=dev)
        t_s64 = _time_steps(lambda: pt.pt_ma_quad_exact(st_, sp_, 1, 1, 0.0, out=so64), 10, 3, flush, 1) / 10
        t_s32 = _time_steps(lambda: pt.pt_ma_quad_exact(st_, sp_, 1, 1, 0.0, out=so32), 10, 3, flush, 1) / 10
        n_sp = wsp.n_pv * wsp.n_t
        extra["dense"]["sparse_rows"] = {"workload": "448 pv x 60000 per-pv times (configs[1] population, own axis per row), n_ss = 1",
                                         "fp64": {"value": n_sp / t_s64, "unit": UNIT, "ms": t_s64 * 1e3, "kernel": "flux_kernel (general)"},
                                         "fp32_variant": {"value": n_sp / t_s32, "unit": UNIT, "ms": t_s32 * 1e3, "kernel": "direct_kernel",
                                                          "speedup_vs_fp64": t_s64 / t_s32}}
        del st_, sp_, so64, so32
    if rank == 0 and "interp" in sections:
        # -------------------------------------------------------------- configs[3]: table build + interpolated path
        wi = inputs.config4()
        c = wi.table
        it_, ip_ = to_dev(wi.times), to_dev(wi.params)
        io = torch.empty((wi.n_pv, 1, wi.n_t), dtype=torch.float64, device=dev)
        res_i = {}
        for name, tdt in (("f32_table", torch.float32), ("f64_table", torch.float64)):
            t_build = _time_steps(lambda: pt.pt_ma_table_build(dtype=tdt, n_fn=4 if tdt == torch.float32 else 3, **c),
                                  3, 1, None, 1) / 3
            tb = pt.pt_ma_table_build(dtype=tdt, n_fn=4 if tdt == torch.float32 else 3, **c)
            t_i = _time_steps(lambda: pt.pt_ma_quad_interp(tb, it_, ip_, out=io), 10, 3, None, 1) / 10
            bytes_alg = wi.n_pv * wi.n_t * 8.0      # the flux write; shared times (0.8 MB) and the table live in L2
            res_i[name] = {"value": wi.n_eval / t_i, "unit": UNIT, "ms": t_i * 1e3, "table_build_ms": t_build * 1e3,
                           "roofline": _hbm_roofline(bytes_alg, t_i, peaks, CAPTURES["interp_f32" if name == "f32_table" else "interp_f64"])}
            del tb
        # fp32 flux halves the bytes
        tb = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, **c)
        io32 = torch.empty((wi.n_pv, 1, wi.n_t), dtype=torch.float32, device=dev)
        t_i32 = _time_steps(lambda: pt.pt_ma_quad_interp(tb, it_, ip_, out=io32), 10, 3, None, 1) / 10
        res_i["f32_table_f32_flux"] = {"value": wi.n_eval / t_i32, "unit": UNIT, "ms": t_i32 * 1e3,
                                       "roofline": _hbm_roofline(wi.n_pv * wi.n_t * 4.0, t_i32, peaks, None)}
        res_i["workload"] = "BASELINE.json configs[3]: 4096 pv x 100000 times, table 401 x 12501, fp64 flux (3.28 GB/launch > L2)"
        res_i["hbm_write_only_note"] = ("peak = MEASURED_PEAKS.json copy bandwidth (read+write); a pure fill of the same 3.28 GB "
                                        "(cudaMemsetAsync) takes 0.447 ms = 7.3 TB/s on this part (profiles/r2_summary.md)")
        extra["interp"] = res_i
        del it_, ip_, io, io32, tb
    if rank == 0 and "configs" in sections:
        # -------------------------------------------------------------- the other BASELINE configs, as specified
        res_o = {}
        w1 = inputs.config1()
        a1, b1 = to_dev(w1.times), to_dev(w1.params)
        o1 = torch.empty((1, 1, w1.n_t), dtype=torch.float64, device=dev)
        t1 = _time_steps(lambda: pt.pt_ma_quad_exact(a1, b1, out=o1), 20, 3, None, 1) / 20
        # the same call replayed from a CUDA graph (MCMC callers replay a fixed launch sequence)
        gs = torch.cuda.Stream()
        with torch.cuda.stream(gs):
            pt.pt_ma_quad_exact(a1, b1, out=o1)
            gs.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=gs):
                pt.pt_ma_quad_exact(a1, b1, out=o1)
        torch.cuda.synchronize()
        t1g = _time_steps(lambda: g.replay(), 20, 3, None, 1) / 20
        n_in1 = _count_units(pt, w1, a1, b1)
        res_o["config1"] = {"latency_us": t1 * 1e6, "latency_us_cuda_graph": t1g * 1e6, "value": w1.n_eval / t1, "unit": UNIT,
                            "note": "1000 evaluations: a latency, not a throughput (SURVEY §8(d)); launch-bound",
                            "roofline": _alu_roofline(w1.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE) + n_in1 * ALG_PER_TRANSIT_CIRC,
                                                      t1, fp64_model_peak, fp64_meas_peak, None, n_in1)}
        del g
        w3 = inputs.config3()
        a3, b3 = to_dev(w3.times), to_dev(w3.params)
        o3 = torch.empty((w3.n_pv, w3.n_pb, w3.n_t), dtype=torch.float64, device=dev)
        t3 = _time_steps(lambda: pt.pt_ma_quad_exact(a3, b3, w3.n_pb, out=o3), 10, 3, flush, 1) / 10
        t3k = _time_steps(lambda: pt.pt_ma_quad_exact_pbk(a3, b3, w3.n_pb, out=o3), 10, 3, flush, 1) / 10
        n_in3 = _count_units(pt, w3, a3, b3)
        alg3 = w3.n_pv * w3.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE * w3.n_pb) + n_in3 * ALG_PER_TRANSIT_CIRC
        res_o["config3"] = {"ms": t3 * 1e3, "z_evals_per_s": w3.n_pv * w3.n_t / t3, "fluxes_per_s": w3.n_pv * w3.n_pb * w3.n_t / t3,
                            "exact_per_passband_k_ms": t3k * 1e3,
                            "roofline": _alu_roofline(alg3, t3, fp64_model_peak, fp64_meas_peak, CAPTURES["config3"], n_in3),
                            "hbm_frac": w3.n_pv * w3.n_pb * w3.n_t * 8.0 / t3 / 1e9 / peaks["hbm_gbs"]}
        # config 5's boundary-targeted times are solved on an orbit routine handed to the generator: here the product's own
        w5 = inputs.config5(lambda t, p: pt.pt_orbit_z(to_dev(t), to_dev(p)).cpu().numpy()[:, :, 0])
        a5, b5 = to_dev(w5.times), to_dev(w5.params)
        o5 = torch.empty((w5.n_pv, 1, w5.n_t), dtype=torch.float64, device=dev)
        t5 = _time_steps(lambda: pt.pt_ma_quad_exact(a5, b5, out=o5), 10, 3, flush, 1) / 10
        n_in5 = _count_units(pt, w5, a5, b5)
        alg5 = w5.n_pv * w5.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE) + n_in5 * ALG_PER_TRANSIT_ECC
        res_o["config5"] = {"ms": t5 * 1e3, "value": w5.n_eval / t5, "unit": UNIT, "in_transit_frac": n_in5 / w5.n_eval,
                            "roofline": _alu_roofline(alg5, t5, fp64_model_peak, fp64_meas_peak, CAPTURES["config5"], n_in5)}
        # the orbit routines of P:L31 on config 5's population (S1-S2 alone)
        zo = torch.empty((w5.n_pv, w5.n_t, 1), dtype=torch.float64, device=dev)
        sol = {}
        for sv in ("exact", "iter", "ps3", "ps5", "fast"):
            tz = _time_steps(lambda: pt.pt_orbit_z_solver(a5, b5, sv, out=zo), 5, 2, flush, 1) / 5
            sol[sv] = {"z_evals_per_s": w5.n_eval / tz, "ms": tz * 1e3}
        sol["note"] = ("e ~ U(0, 0.6): 'fast' dispatches to Newton for almost every row here; ps3/ps5 are timed on this population "
                       "although their truncation error is only below 2e-9 rad for e <= 0.006 / 0.03 (DESIGN.md R19)")
        sol["hbm_frac_exact"] = w5.n_eval * 16.0 / (sol["exact"]["ms"] * 1e-3) / 1e9 / peaks["hbm_gbs"]
        res_o["config5"]["orbit_solvers"] = sol
        extra["configs"] = res_o
        del a1, b1, o1, a3, b3, o3, a5, b5, o5, zo
    if rank == 0 and "gimenez" in sections:
        # -------------------------------------------------------------- the Giménez model (S§8(f) NEXT-4): series and z-interpolation
        wg = inputs.dense_transit(n_pv=1024, n_t=4096)
        pg = np.concatenate([wg.params[:, :7], (wg.params[:, 7] + 2 * wg.params[:, 8])[:, None], -wg.params[:, 8][:, None]], axis=1)
        gt, gp = to_dev(wg.times), to_dev(pg)
        go = torch.empty((wg.n_pv, 1, wg.n_t), dtype=torch.float64, device=dev)
        res_g = {"workload": "1024 pv x 4096 per-pv times near transit (the `dense` population), quadratic law as N = 2, one passband"}
        for n_j in (20, 40):
            coef = pt.GimenezCoef(2, n_j)
            tg = _time_steps(lambda: pt.pt_gimenez_exact(coef, gt, gp, out=go), 5, 2, flush, 1) / 5
            res_g["series_nj%d" % n_j] = {"value": wg.n_eval / tg, "unit": UNIT, "ms": tg * 1e3}
        gw = torch.empty((wg.n_pv, 3, 256 + 256), dtype=torch.float64, device=dev)
        tgi = _time_steps(lambda: pt.pt_gimenez_interp(coef, 256, 256, gt, gp, out=go, work=gw), 5, 2, flush, 1) / 5
        res_g["interp_256_256_nj40"] = {"value": wg.n_eval / tgi, "unit": UNIT, "ms": tgi * 1e3}
        fm = pt.pt_ma_quad_exact(gt[:64].contiguous(), to_dev(wg.params[:64]))
        fgx = pt.pt_gimenez_exact(coef, gt[:64].contiguous(), gp[:64].contiguous())
        fgi, _ = pt.pt_gimenez_interp(coef, 256, 256, gt[:64].contiguous(), gp[:64].contiguous())
        res_g["max_abs_diff_series_nj40_vs_mandel_agol"] = float((fgx - fm).abs().max().item())
        res_g["max_abs_diff_interp_vs_series"] = float((fgi - fgx).abs().max().item())
        extra["gimenez"] = res_g
        del gt, gp, go, gw
    if rank == 0 and "chi2" in sections:
        # -------------------------------------------------------------- fused likelihood (S§8(f) NEXT-1): no flux is written
        res_c = {}
        rng = np.random.default_rng(1504)
        for name, wl, use_table in (("config2", inputs.config2(), False), ("config4_exact", inputs.config4(), False),
                                    ("config4_interp", inputs.config4(), True)):
            ct, cp = to_dev(wl.times), to_dev(wl.params)
            truth = pt.pt_ma_quad_exact(ct, cp[:1].contiguous(), 1, wl.n_ss, wl.t_exp)[0]
            obs = (truth + 2e-4 * torch.from_numpy(rng.standard_normal((1, wl.n_t))).to(dev)).contiguous()
            isig = torch.full_like(obs, 1.0 / 2e-4)
            tbl = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, **wl.table) if use_table else None
            co = torch.empty(wl.n_pv, dtype=torch.float64, device=dev)
            t_c = _time_steps(lambda: pt.pt_ma_quad_chi2(ct, cp, obs, isig, 1, wl.n_ss, wl.t_exp, table=tbl, out=co),
                              10, 3, flush, 1) / 10
            res_c[name] = {"value": wl.n_eval / t_c, "unit": UNIT, "ms": t_c * 1e3, "launches_per_call": 2}
            del ct, cp, obs, isig, co, tbl
        res_c["note"] = ("pt_ma_quad_chi2: chi2[pv] against one data set; exposures outside the transit windows cost nothing at all "
                         "(no flux is written), so the flux-store roofline does not apply")
        extra["chi2"] = res_c
    if rank == 0 and "cpu" in sections:
        # -------------------------------------------------------------- CPU leg: the oracle as it stands, timed on the host cores
        # per config, and (outside every timed GPU region) the GPU path's error against its __float128 instantiation
        from oracle import pt_oracle
        pt_oracle.build()
        cores = pt_oracle.num_threads()

        def cpu_time(fn, reps=3):
            best = float("inf")
            for _ in range(reps):
                t0_ = time.perf_counter()
                fn()
                best = min(best, time.perf_counter() - t0_)
            return best

        dt_cpu = cpu_time(lambda: pt_oracle.ma_quad_exact(w.times, w.params, w.n_pb, w.n_ss, w.t_exp, prec="f64"), 5)
        extra["cpu_baseline"] = {"value": w.n_eval / dt_cpu, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt_cpu,
                                 "sample": "all 64 pv of the same configs[1] batch (3.84e7 evals), oracle double instantiation (OpenMP), best of 5"}
        # thread sweep (the paper found fewer threads than cores optimal)
        sweep = {}
        for nt in sorted({max(1, cores // 2), max(1, (3 * cores) // 4), cores}):
            pt_oracle.set_num_threads(nt)
            sweep[str(nt)] = w.n_eval / cpu_time(lambda: pt_oracle.ma_quad_exact(w.times, w.params, w.n_pb, w.n_ss, w.t_exp, prec="f64"))
        pt_oracle.set_num_threads(cores)
        extra["cpu_baseline"]["threads_sweep_evals_per_s"] = sweep
        extra["cpu_baseline"]["best_threads"] = int(max(sweep, key=lambda k_: sweep[k_]))
        per_cfg, acc = {}, {}
        w1 = inputs.config1()
        per_cfg["config1"] = w1.n_eval / cpu_time(lambda: pt_oracle.ma_quad_exact(w1.times, w1.params, prec="f64"), 5)
        f1 = pt.pt_ma_quad_exact(to_dev(w1.times), to_dev(w1.params)).cpu().numpy()
        acc["config1"] = {"max_abs_err_vs_oracle": float(np.abs(f1 - pt_oracle.ma_quad_exact(w1.times, w1.params, prec="f128")).max()),
                          "sample": "all 1000 evaluations"}
        per_cfg["config2"] = extra["cpu_baseline"]["value"]
        f2 = out[:8].cpu().numpy()
        r2 = pt_oracle.ma_quad_exact(w.times, w.params[:8], w.n_pb, w.n_ss, w.t_exp, prec="f128")
        acc["config2"] = {"max_abs_err_vs_oracle": float(np.abs(f2 - r2).max()), "sample": "first 8 of 64 rows x 60000 exposures (the full 64 rows: tests/test_gpu_parity.py)"}
        f2f = pt.pt_ma_quad_exact(d_t, d_p[:8].contiguous(), 1, w.n_ss, w.t_exp, dtype=torch.float32).cpu().numpy()
        acc["config2_fp32_variant"] = {"max_abs_err_vs_oracle": float(np.abs(f2f.astype(np.float64) - r2).max()), "gate": 2e-6}
        w3 = inputs.config3()
        per_cfg["config3"] = w3.n_pv * w3.n_t / cpu_time(lambda: pt_oracle.ma_quad_exact(w3.times, w3.params, w3.n_pb, prec="f64"))
        f3 = pt.pt_ma_quad_exact(to_dev(w3.times), to_dev(w3.params[:32]), w3.n_pb).cpu().numpy()
        acc["config3"] = {"max_abs_err_vs_oracle": float(np.abs(f3 - pt_oracle.ma_quad_exact(w3.times, w3.params[:32], w3.n_pb, prec="f128")).max()),
                          "sample": "first 32 of 512 walkers x 20 passbands x 600 exposures"}
        w4 = inputs.config4(n_pv=256)
        c4 = w4.table
        tb_o = pt_oracle.ma_table_build(c4["k_min"], c4["k_max"], c4["n_k"], c4["z_max"], c4["n_z"], np.float64, 3, "f64")
        dk4, dz4 = pt_oracle.table_spacing(c4["k_min"], c4["k_max"], c4["n_k"], c4["z_max"], c4["n_z"])
        per_cfg["config4_interp"] = w4.n_eval / cpu_time(lambda: pt_oracle.ma_quad_interp(tb_o, c4["k_min"], dk4, dz4, w4.times, w4.params, prec="f64"), 2)
        per_cfg["config4_note"] = "interpolated path on the first 256 of 4096 parameter vectors (2.56e7 evals), the oracle's own fp64 table"
        tb_g = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, **c4)
        fi = pt.pt_ma_quad_interp(tb_g, to_dev(w4.times), to_dev(w4.params[:16])).cpu().numpy()
        ri = pt_oracle.ma_quad_interp(tb_g.data.cpu().numpy(), tb_g.k_min, tb_g.dk, tb_g.dz, w4.times, w4.params[:16], prec="f128")
        rx = pt_oracle.ma_quad_exact(w4.times, w4.params[:16], prec="f128")
        in_tr = rx < 1.0
        acc["config4_interp"] = {"max_abs_err_vs_oracle_interp_of_same_table": float(np.abs(fi - ri).max()),
                                 "interp_vs_exact_max": float(np.abs(fi - rx).max()),
                                 "interp_vs_exact_mean_in_transit": float(np.abs(fi - rx)[in_tr].mean()),
                                 "sample": "first 16 of 4096 rows x 100000 times, fp32 table 401 x 12501 (reported, not gated: P:L149)"}
        w5 = inputs.config5(lambda t, p: pt_oracle.orbit_z(t, p, prec="f64")[:, :, 0])
        per_cfg["config5"] = w5.n_eval / cpu_time(lambda: pt_oracle.ma_quad_exact(w5.times, w5.params, prec="f64"), 2)
        f5 = pt.pt_ma_quad_exact(to_dev(w5.times[:128]), to_dev(w5.params[:128])).cpu().numpy()
        acc["config5"] = {"max_abs_err_vs_oracle": float(np.abs(f5 - pt_oracle.ma_quad_exact(w5.times[:128], w5.params[:128], prec="f128")).max()),
                          "sample": "first 128 of 4096 rows x 4096 times (every population group: tests/test_gpu_parity.py)"}
        extra["cpu_baseline"]["per_config_evals_per_s"] = per_cfg
        extra["accuracy"] = acc

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "per_gpu": "one seeded population per rank, no collective",
                       "l2": "256 MiB buffer rewritten between timed steps (L2 flushed); per-step CUDA events"},
            "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e, "roofline": roofline,
        }
        line.update(extra)
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


WORKLOADS = ("config1", "config2", "config2x7", "config3", "config4_f32", "config4_f64", "config5", "dense", "dense_f32",
             "chi2_config2", "chi2_config4_interp")


def run_single(args):
    """`--workload NAME`: W + K launches of ONE named workload, per-launch CUDA-event times on stdout — the command the ncu
    captures under profiles/ are taken with (no oracle, no JSON line)."""
    import torch

    import paper_1504_07433_b200 as pt
    from paper_1504_07433_b200 import inputs
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)

    def to_dev(x):
        return torch.from_numpy(np.ascontiguousarray(x)).to(dev)

    name = args.workload
    if name in ("config1", "config2", "config2x7", "config3", "config5", "dense", "dense_f32"):
        w = {"config1": inputs.config1, "config2": inputs.config2, "config2x7": lambda: inputs.config2(n_pv=448),
             "config3": inputs.config3, "dense": inputs.dense_transit, "dense_f32": inputs.dense_transit,
             "config5": lambda: inputs.config5(lambda t, p: pt.pt_orbit_z(to_dev(t), to_dev(p)).cpu().numpy()[:, :, 0])}[name]()
        t, p = to_dev(w.times), to_dev(w.params)
        o = torch.empty((w.n_pv, w.n_pb, w.n_t), dtype=torch.float32 if name == "dense_f32" else torch.float64, device=dev)
        fn, n_eval = (lambda: pt.pt_ma_quad_exact(t, p, w.n_pb, w.n_ss, w.t_exp, out=o)), w.n_eval
    elif name in ("config4_f32", "config4_f64"):
        w = inputs.config4()
        t, p = to_dev(w.times), to_dev(w.params)
        f32 = name == "config4_f32"
        tb = pt.pt_ma_table_build(dtype=torch.float32 if f32 else torch.float64, n_fn=4 if f32 else 3, **w.table)
        o = torch.empty((w.n_pv, 1, w.n_t), dtype=torch.float64, device=dev)
        fn, n_eval = (lambda: pt.pt_ma_quad_interp(tb, t, p, out=o)), w.n_eval
    elif name in ("chi2_config2", "chi2_config4_interp"):
        w = inputs.config2() if name == "chi2_config2" else inputs.config4()
        t, p = to_dev(w.times), to_dev(w.params)
        truth = pt.pt_ma_quad_exact(t, p[:1].contiguous(), 1, w.n_ss, w.t_exp)[0]
        obs = (truth + 2e-4 * torch.randn_like(truth)).contiguous()
        isig = torch.full_like(obs, 5e3)
        tb = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, **w.table) if name == "chi2_config4_interp" else None
        co = torch.empty(w.n_pv, dtype=torch.float64, device=dev)
        fn, n_eval = (lambda: pt.pt_ma_quad_chi2(t, p, obs, isig, 1, w.n_ss, w.t_exp, table=tb, out=co)), w.n_eval
    else:
        raise SystemExit("unknown workload %r (one of %s)" % (name, ", ".join(WORKLOADS)))
    flush_buf = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)
    ts = []
    for i in range(args.warmup + args.steps):
        flush_buf.fill_(1.0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        if i >= args.warmup:
            ts.append(a.elapsed_time(b))
    print("%s: mean %.4f ms, min %.4f ms over %d launches after %d warm-up; %.4e evals/s" % (
        name, float(np.mean(ts)), float(np.min(ts)), len(ts), args.warmup, n_eval / (float(np.mean(ts)) * 1e-3)))


def run_reference(args):
    """The reference arm of this tier is the CPU oracle, as it stands, timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pt_oracle
    from paper_1504_07433_b200 import inputs
    pt_oracle.build()
    w = inputs.config2()
    n_pv = w.n_pv   # the whole configs[1] batch per step (0.1 s of CPU work on 16 cores): every core is busy
    p = w.params
    for _ in range(args.warmup):
        pt_oracle.ma_quad_exact(w.times, p, w.n_pb, w.n_ss, w.t_exp, prec="f64")
    t0 = time.perf_counter()
    for _ in range(args.steps):
        pt_oracle.ma_quad_exact(w.times, p, w.n_pb, w.n_ss, w.t_exp, prec="f64")
    dt = time.perf_counter() - t0
    n_eval = n_pv * w.n_t * w.n_ss
    value = n_eval * args.steps / dt
    sample = "all 64 parameter vectors of configs[1] per step (3.84e7 evals), oracle double instantiation (OpenMP over parameter vectors)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": pt_oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sections", default="scaled,dense,interp,configs,chi2,gimenez,cpu",
                    help="extra sections to run besides the headline: any of scaled,dense,interp,configs,chi2,gimenez,cpu (or 'none')")
    ap.add_argument("--workload", default=None, help="run only this workload (%s): the command of the ncu captures" % ", ".join(WORKLOADS))
    args = ap.parse_args()
    if args.workload:
        run_single(args)
        return
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
