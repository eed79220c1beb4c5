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
FP64_LANES_PER_SM, N_SM = 64, 148
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures (profiles/r1c_ncu_*.md);
# a kernel's output that is still in L2 when the capture ends is not in its figure (configs[1]: 30.7 MB of flux < 126 MB L2).
TRAFFIC_EXACT_CONFIG2 = 572.416e3 + 10.496e3
TRAFFIC_INTERP_F32 = 519.879936e6 + 3.233794e9
TRAFFIC_DENSE = 134.598656e6 + 88.509696e6


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

    alg_inst = (w.n_pv * w.n_t * (ALG_PER_EXPOSURE + ALG_PER_COMBINE * w.n_pb) + n_in * ALG_PER_TRANSIT_CIRC)
    kernel_s = total_s / args.steps
    ach = alg_inst / kernel_s

    # ------------------------------------------------------------------ FP64 pipe peak, measured
    sink = torch.empty(N_SM * 16 * 256, dtype=torch.float64, device=dev)
    iters = 20000
    t_probe = _time_steps(lambda: pt.pt_probe_dfma(N_SM * 16, iters, sink), 5, 2, None, 1) / 5
    fp64_meas_peak = N_SM * 16 * 256 * iters * 8 / t_probe

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
                           "fp64_frac_of_model_peak": alg_s / t_s / fp64_model_peak}
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
                          "fp64_frac_of_model_peak": alg_d / t_d / fp64_model_peak,
                          "fp64_frac_of_measured_peak": alg_d / t_d / fp64_meas_peak, "traffic": TRAFFIC_DENSE}
        # fp32-output variant on the same workload
        do32 = torch.empty((wd.n_pv, 1, wd.n_t), dtype=torch.float32, device=dev)
        t_d32 = _time_steps(lambda: pt.pt_ma_quad_exact(dt_, dp_, dtype=torch.float32, out=do32), 10, 3, flush, 1) / 10
        extra["dense"]["fp32_variant_value"] = wd.n_eval / t_d32
        del dt_, dp_, do, do32
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
                           "roofline": {"bound": "hbm", "achieved": bytes_alg / t_i / 1e9, "peak": peaks["hbm_gbs"],
                                        "unit": "GB/s", "frac": bytes_alg / t_i / 1e9 / peaks["hbm_gbs"],
                                        "traffic": TRAFFIC_INTERP_F32 if name == "f32_table" else None,
                                        "peak_source": peaks["source"]}}
            del tb
        res_i["workload"] = "BASELINE.json configs[3]: 4096 pv x 100000 times, table 401 x 12501, fp64 flux (3.28 GB/launch > L2)"
        extra["interp"] = res_i
        del it_, ip_, io
    if rank == 0 and "configs" in sections:
        # -------------------------------------------------------------- the other BASELINE configs, as specified
        res_o = {}
        w1 = inputs.config1()
        a1, b1 = to_dev(w1.times), to_dev(w1.params)
        o1 = torch.empty((1, 1, w1.n_t), dtype=torch.float64, device=dev)
        t1 = _time_steps(lambda: pt.pt_ma_quad_exact(a1, b1, out=o1), 20, 3, None, 1) / 20
        res_o["config1"] = {"latency_us": t1 * 1e6, "note": "1000 evaluations: a latency, not a throughput (SURVEY §8(d))"}
        w3 = inputs.config3()
        a3, b3 = to_dev(w3.times), to_dev(w3.params)
        o3 = torch.empty((w3.n_pv, w3.n_pb, w3.n_t), dtype=torch.float64, device=dev)
        t3 = _time_steps(lambda: pt.pt_ma_quad_exact(a3, b3, w3.n_pb, out=o3), 10, 3, flush, 1) / 10
        t3k = _time_steps(lambda: pt.pt_ma_quad_exact_pbk(a3, b3, w3.n_pb, out=o3), 10, 3, flush, 1) / 10
        res_o["config3"] = {"ms": t3 * 1e3, "z_evals_per_s": w3.n_pv * w3.n_t / t3, "fluxes_per_s": w3.n_pv * w3.n_pb * w3.n_t / t3,
                            "exact_per_passband_k_ms": t3k * 1e3}
        # config 5's boundary-targeted times are solved on an orbit routine handed to the generator: here the product's own
        w5 = inputs.config5(lambda t, p: pt.pt_orbit_z(to_dev(t), to_dev(p)).cpu().numpy()[:, :, 0])
        a5, b5 = to_dev(w5.times), to_dev(w5.params)
        o5 = torch.empty((w5.n_pv, 1, w5.n_t), dtype=torch.float64, device=dev)
        t5 = _time_steps(lambda: pt.pt_ma_quad_exact(a5, b5, out=o5), 10, 3, flush, 1) / 10
        res_o["config5"] = {"ms": t5 * 1e3, "value": w5.n_eval / t5, "unit": UNIT}
        extra["configs"] = res_o
        del a1, b1, o1, a3, b3, o3, a5, b5, o5
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
        res_c["note"] = ("pt_ma_quad_chi2: chi2[pv] against one data set; out-of-window exposures cost a window test and no "
                         "memory traffic (times are L2-resident), so the flux-store roofline does not apply")
        extra["chi2"] = res_c
    if rank == 0 and "cpu" in sections:
        # -------------------------------------------------------------- CPU baseline: the oracle as it stands
        from oracle import pt_oracle
        pt_oracle.build()
        n_cpu_pv = 64
        dt_cpu = float("inf")
        for _ in range(5):                                   # best of 5 wall-clock runs
            t0 = time.perf_counter()
            pt_oracle.ma_quad_exact(w.times, w.params[:n_cpu_pv], w.n_pb, w.n_ss, w.t_exp, prec="f64")
            dt_cpu = min(dt_cpu, time.perf_counter() - t0)
        extra["cpu_baseline"] = {"value": n_cpu_pv * w.n_t * w.n_ss / dt_cpu, "unit": UNIT, "cores": pt_oracle.num_threads(),
                                 "kind": "oracle", "seconds": dt_cpu,
                                 "sample": "all 64 pv of the same configs[1] batch (3.84e7 evals), oracle double instantiation (OpenMP), best of 5"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "per_gpu": "one seeded population per rank, no collective",
                       "l2": "256 MiB buffer rewritten between timed steps (L2 flushed); per-step CUDA events"},
            "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
            "roofline": {"bound": "alu", "achieved": ach * 2 / 1e12, "peak": fp64_model_peak * 2 / 1e12,
                         "unit": "TFLOP/s", "frac": ach / fp64_model_peak, "traffic": TRAFFIC_EXACT_CONFIG2,
                         "traffic_source": "profiles/r1c_ncu_exact_config2.md (bytes per launch)",
                         "kernel": "flux_kernel<0,2,1,0,double>", "in_transit_evals": n_in, "alg_fp64_inst_per_launch": alg_inst,
                         "peak_source": "model: 148 SM x 64 FP64 lanes x sm_max_mhz x 2 flop (DESIGN.md §6)",
                         "fp64_peak_measured_tflops": fp64_meas_peak * 2 / 1e12,
                         "frac_of_measured_dfma_peak": ach / fp64_meas_peak,
                         "hbm_frac": w.n_pv * w.n_t * 8.0 / kernel_s / 1e9 / peaks["hbm_gbs"]},
        }
        line.update(extra)
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def run_reference(args):
    """The reference arm of this tier is the CPU oracle, as it stands, timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pt_oracle
    from paper_1504_07433_b200 import inputs
    pt_oracle.build()
    w = inputs.config2()
    n_pv = 8   # bounded sample of the same workload per step
    p = w.params[:n_pv]
    for _ in range(args.warmup):
        pt_oracle.ma_quad_exact(w.times, p, w.n_pb, w.n_ss, w.t_exp, prec="f64")
    t0 = time.perf_counter()
    for _ in range(args.steps):
        pt_oracle.ma_quad_exact(w.times, p, w.n_pb, w.n_ss, w.t_exp, prec="f64")
    dt = time.perf_counter() - t0
    n_eval = n_pv * w.n_t * w.n_ss
    value = n_eval * args.steps / dt
    sample = "first 8 of the 64 parameter vectors of configs[1] per step (4.8e6 evals), oracle double instantiation"
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
    ap.add_argument("--sections", default="scaled,dense,interp,configs,chi2,cpu",
                    help="extra sections to run besides the headline: any of scaled,dense,interp,configs,chi2,cpu (or 'none')")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
