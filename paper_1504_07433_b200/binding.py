"""Thin Python binding of the C ABI in include/pt.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libpt_b200.so; PyTorch is used for device memory and streams.
There is no CPU fallback: importing works without a GPU (so that the symbol table can be checked), but loading fails
loudly if the shared library has not been built, and every compute call requires CUDA tensors.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpt_b200.so")

PT_OK, PT_ERR_NULL, PT_ERR_SIZE, PT_ERR_DTYPE, PT_ERR_TABLE, PT_ERR_CUDA = range(6)
PT_F64, PT_F32, PT_F32S = 0, 1, 2
PT_ST_BAD_PARAM, PT_ST_K_OUT_OF_TABLE = 1, 2
_ERR = {1: "PT_ERR_NULL", 2: "PT_ERR_SIZE", 3: "PT_ERR_DTYPE", 4: "PT_ERR_TABLE", 5: "PT_ERR_CUDA"}

EXPORTS = ("pt_build_arch", "pt_orbit_z", "pt_orbit_z_solver", "pt_ma_quad_exact", "pt_ma_table_build", "pt_table_spacing", "pt_ma_quad_interp", "pt_ma_quad_chi2", "pt_ma_quad_exact_pbk",
           "pt_ma_quad_exact_host", "pt_ma_quad_interp_host", "pt_plan", "pt_probe_dfma", "pt_probe_ffma",
           "pt_gimenez_coef_size", "pt_gimenez_coef_build", "pt_gimenez_exact", "pt_gimenez_interp", "pt_gimenez_interp_static",
           "pt_gimenez_static_work_doubles", "pt_launch_count")


class PtError(RuntimeError):
    pass


class pt_table(C.Structure):
    _fields_ = [("d_data", C.c_void_p), ("dtype", C.c_int32), ("n_k", C.c_int32), ("n_z", C.c_int32),
                ("n_fn", C.c_int32), ("k_min", C.c_double), ("dk", C.c_double), ("dz", C.c_double)]


_lib = None


def lib() -> C.CDLL:
    """Load libpt_b200.so (built in-tree by paper_1504_07433_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PtError("CUDA extension %s is missing: run `python -m paper_1504_07433_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        i32, i64, dbl, ptr = C.c_int32, C.c_int64, C.c_double, C.c_void_p
        common = [ptr, i64, i64, ptr, i64, i32, i32, dbl]
        L.pt_build_arch.restype = C.c_int
        L.pt_launch_count.restype = i64
        L.pt_orbit_z.argtypes = common + [ptr, ptr]
        L.pt_orbit_z_solver.argtypes = common + [i32, ptr, ptr]
        L.pt_ma_quad_exact.argtypes = common + [i32, ptr, ptr, ptr]
        L.pt_ma_quad_exact_pbk.argtypes = common + [i32, ptr, ptr, ptr]
        L.pt_ma_table_build.argtypes = [dbl, dbl, i32, dbl, i32, i32, i32, ptr, ptr]
        L.pt_table_spacing.argtypes = [dbl, dbl, i32, dbl, i32, C.POINTER(dbl), C.POINTER(dbl)]
        L.pt_ma_quad_interp.argtypes = [C.POINTER(pt_table)] + common + [i32, ptr, ptr, ptr]
        L.pt_ma_quad_chi2.argtypes = [C.POINTER(pt_table), ptr, i64, ptr, i64, i32, i32, dbl, ptr, ptr, ptr, ptr, ptr]
        L.pt_ma_quad_exact_host.argtypes = common + [i32, ptr, ptr]
        L.pt_ma_quad_interp_host.argtypes = [C.POINTER(pt_table)] + common + [i32, ptr, ptr]
        L.pt_probe_dfma.argtypes = [i32, i32, ptr, ptr]
        L.pt_gimenez_coef_size.argtypes = [i32, i32, C.POINTER(i64)]
        L.pt_gimenez_coef_build.argtypes = [i32, i32, ptr, ptr]
        L.pt_gimenez_exact.argtypes = [ptr, i32, i32, ptr, i64, i64, ptr, i64, i32, i32, dbl, ptr, ptr, ptr]
        L.pt_gimenez_interp.argtypes = [ptr, i32, i32, i32, i32, ptr, ptr, i64, i64, ptr, i64, i32, i32, dbl, ptr, ptr, ptr]
        L.pt_gimenez_interp_static.argtypes = [ptr, i32, i32, i32, i32, ptr, i64, i64, ptr, i64, i32, i32, dbl, ptr, ptr, ptr]
        L.pt_gimenez_static_work_doubles.argtypes = []
        L.pt_probe_ffma.argtypes = [i32, i32, ptr, ptr]
        L.pt_plan.argtypes = [i64, i64, i32, C.POINTER(C.c_int64)]
        for n in EXPORTS[1:-1]:
            getattr(L, n).restype = C.c_int
        L.pt_gimenez_static_work_doubles.restype = i64
        _lib = L
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != PT_OK:
        raise PtError("%s failed: %s" % (what, _ERR.get(rc, rc)))


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dtype_code(dtype: torch.dtype) -> int:
    if dtype == torch.float64:
        return PT_F64
    if dtype == torch.float32:
        return PT_F32
    raise PtError("flux/table dtype must be float64 or float32")


def _marshal(times: torch.Tensor, params: torch.Tensor, n_pb: int, device_required: bool = True):
    if params.dim() == 1:
        params = params[None, :]
    if times.dtype != torch.float64 or params.dtype != torch.float64:
        raise PtError("times and params must be float64")
    if not (times.is_contiguous() and params.is_contiguous()):
        raise PtError("times and params must be contiguous")
    if device_required and not (times.is_cuda and params.is_cuda):
        raise PtError("times and params must be CUDA tensors (there is no CPU path)")
    if not device_required and (times.is_cuda or params.is_cuda):
        raise PtError("the *_host entry points take host tensors")
    n_pv = params.shape[0]
    if params.shape[1] != 6 + 3 * n_pb:
        raise PtError("parameter rows must hold 6 + 3*n_pb doubles")
    if times.dim() == 1:
        n_t, stride = times.shape[0], 0
    elif times.dim() == 2 and times.shape[0] == n_pv:
        n_t, stride = times.shape[1], times.shape[1]
    else:
        raise PtError("times must be [n_t] or [n_pv][n_t]")
    return times, params, n_pv, n_t, stride


def pt_orbit_z(times: torch.Tensor, params: torch.Tensor, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0,
               out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Signed projected separation [n_pv][n_t][n_ss] (include/pt.h: pt_orbit_z)."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb)
    if out is None:
        out = torch.empty((n_pv, n_t, n_ss), dtype=torch.float64, device=times.device)
    _check(lib().pt_orbit_z(times.data_ptr(), n_t, stride, params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp),
                            out.data_ptr(), _stream()), "pt_orbit_z")
    return out


SOLVERS = {"exact": 0, "newton": 1, "iter": 2, "ps3": 3, "ps5": 4, "fast": 5}


def pt_orbit_z_solver(times: torch.Tensor, params: torch.Tensor, solver: str, n_pb: int = 1, n_ss: int = 1,
                      t_exp: float = 0.0, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Signed projected separation by one of the orbit routines of P:L31 (include/pt.h: pt_orbit_z_solver)."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb)
    if solver not in SOLVERS:
        raise PtError("solver must be one of %s" % sorted(SOLVERS))
    if out is None:
        out = torch.empty((n_pv, n_t, n_ss), dtype=torch.float64, device=times.device)
    _check(lib().pt_orbit_z_solver(times.data_ptr(), n_t, stride, params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp),
                                   SOLVERS[solver], out.data_ptr(), _stream()), "pt_orbit_z_solver")
    return out


def pt_ma_quad_exact(times: torch.Tensor, params: torch.Tensor, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0,
                     dtype: torch.dtype = torch.float64, out: Optional[torch.Tensor] = None,
                     status: Optional[torch.Tensor] = None, fp32_store_only: bool = False) -> torch.Tensor:
    """Exact quadratic Mandel–Agol flux [n_pv][n_pb][n_t] (include/pt.h: pt_ma_quad_exact).
    float32 output selects PT_F32 (fp32 arithmetic from the folded phase on), or PT_F32S with fp32_store_only."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb)
    if out is None:
        out = torch.empty((n_pv, n_pb, n_t), dtype=dtype, device=times.device)
    code = _dtype_code(out.dtype)
    if code == PT_F32 and fp32_store_only:
        code = PT_F32S
    _check(lib().pt_ma_quad_exact(times.data_ptr(), n_t, stride, params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp),
                                  code, out.data_ptr(),
                                  status.data_ptr() if status is not None else None, _stream()), "pt_ma_quad_exact")
    return out


def pt_ma_quad_exact_pbk(times: torch.Tensor, params: torch.Tensor, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0,
                         dtype: torch.dtype = torch.float64, out: Optional[torch.Tensor] = None,
                         status: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Exact flux with every passband at its own radius ratio (include/pt.h: pt_ma_quad_exact_pbk)."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb)
    if out is None:
        out = torch.empty((n_pv, n_pb, n_t), dtype=dtype, device=times.device)
    _check(lib().pt_ma_quad_exact_pbk(times.data_ptr(), n_t, stride, params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp),
                                      _dtype_code(out.dtype), out.data_ptr(),
                                      status.data_ptr() if status is not None else None, _stream()),
           "pt_ma_quad_exact_pbk")
    return out


class Table:
    """A device-resident (k,z) table plus its descriptor (include/pt.h: pt_table)."""

    def __init__(self, data: torch.Tensor, k_min: float, dk: float, dz: float):
        self.data, self.k_min, self.dk, self.dz = data, float(k_min), float(dk), float(dz)
        n_k, n_z, n_fn = data.shape
        self.desc = pt_table(data.data_ptr(), _dtype_code(data.dtype), n_k, n_z, n_fn, self.k_min, self.dk, self.dz)


def pt_ma_table_build(k_min: float, k_max: float, n_k: int, z_max: float, n_z: int,
                      dtype: torch.dtype = torch.float64, n_fn: int = 3, device="cuda") -> Table:
    """Build the interpolation table on the device (include/pt.h: pt_ma_table_build)."""
    data = torch.empty((n_k, n_z, n_fn), dtype=dtype, device=device)
    _check(lib().pt_ma_table_build(float(k_min), float(k_max), n_k, float(z_max), n_z, _dtype_code(dtype), n_fn,
                                   data.data_ptr(), _stream()), "pt_ma_table_build")
    dk, dz = C.c_double(), C.c_double()
    _check(lib().pt_table_spacing(float(k_min), float(k_max), n_k, float(z_max), n_z, C.byref(dk), C.byref(dz)),
           "pt_table_spacing")
    return Table(data, k_min, dk.value, dz.value)


def pt_ma_quad_interp(table: Table, times: torch.Tensor, params: torch.Tensor, n_pb: int = 1, n_ss: int = 1,
                      t_exp: float = 0.0, dtype: torch.dtype = torch.float64, out: Optional[torch.Tensor] = None,
                      status: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Interpolated quadratic Mandel–Agol flux [n_pv][n_pb][n_t] (include/pt.h: pt_ma_quad_interp)."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb)
    if out is None:
        out = torch.empty((n_pv, n_pb, n_t), dtype=dtype, device=times.device)
    _check(lib().pt_ma_quad_interp(C.byref(table.desc), times.data_ptr(), n_t, stride, params.data_ptr(), n_pv, n_pb,
                                   n_ss, float(t_exp), _dtype_code(out.dtype), out.data_ptr(),
                                   status.data_ptr() if status is not None else None, _stream()), "pt_ma_quad_interp")
    return out


def pt_ma_quad_chi2(times: torch.Tensor, params: torch.Tensor, obs: torch.Tensor, isig: torch.Tensor, n_pb: int = 1,
                    n_ss: int = 1, t_exp: float = 0.0, table: Optional[Table] = None, out: Optional[torch.Tensor] = None,
                    status: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Fused likelihood chi2[n_pv] against one data set obs/isig [n_pb][n_t] (include/pt.h: pt_ma_quad_chi2)."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb)
    if stride != 0:
        raise PtError("pt_ma_quad_chi2 takes one shared time axis [n_t]")
    for x in (obs, isig):
        if not (x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.numel() == n_pb * n_t):
            raise PtError("obs and isig must be contiguous CUDA float64 tensors of n_pb*n_t elements")
    if out is None:
        out = torch.empty(n_pv, dtype=torch.float64, device=times.device)
    _check(lib().pt_ma_quad_chi2(C.byref(table.desc) if table is not None else None, times.data_ptr(), n_t,
                                 params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp), obs.data_ptr(), isig.data_ptr(),
                                 out.data_ptr(), status.data_ptr() if status is not None else None, _stream()),
           "pt_ma_quad_chi2")
    return out


def pt_ma_quad_exact_host(times: torch.Tensor, params: torch.Tensor, out: torch.Tensor, n_pb: int = 1, n_ss: int = 1,
                          t_exp: float = 0.0, status: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Host buffers in, host buffer out; H2D + kernels + D2H inside the call (include/pt.h: pt_ma_quad_exact_host)."""
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb, device_required=False)
    _check(lib().pt_ma_quad_exact_host(times.data_ptr(), n_t, stride, params.data_ptr(), n_pv, n_pb, n_ss,
                                       float(t_exp), _dtype_code(out.dtype), out.data_ptr(),
                                       status.data_ptr() if status is not None else None), "pt_ma_quad_exact_host")
    return out


def pt_ma_quad_interp_host(table: Table, times: torch.Tensor, params: torch.Tensor, out: torch.Tensor, n_pb: int = 1,
                           n_ss: int = 1, t_exp: float = 0.0, status: Optional[torch.Tensor] = None) -> torch.Tensor:
    times, params, n_pv, n_t, stride = _marshal(times, params, n_pb, device_required=False)
    _check(lib().pt_ma_quad_interp_host(C.byref(table.desc), times.data_ptr(), n_t, stride, params.data_ptr(), n_pv,
                                        n_pb, n_ss, float(t_exp), _dtype_code(out.dtype), out.data_ptr(),
                                        status.data_ptr() if status is not None else None), "pt_ma_quad_interp_host")
    return out


class GimenezCoef:
    """The coefficient table of the Giménez model for (n_ldc, n_j), built on the device (include/pt.h: pt_gimenez_coef_build)."""

    def __init__(self, n_ldc: int, n_j: int, device=None):
        nbytes = C.c_int64(0)
        _check(lib().pt_gimenez_coef_size(n_ldc, n_j, C.byref(nbytes)), "pt_gimenez_coef_size")
        self.n_ldc, self.n_j = int(n_ldc), int(n_j)
        self.data = torch.empty(nbytes.value // 8, dtype=torch.float64, device=device or torch.device("cuda", torch.cuda.current_device()))
        _check(lib().pt_gimenez_coef_build(n_ldc, n_j, self.data.data_ptr(), _stream()), "pt_gimenez_coef_build")


def _marshal_gimenez(times, params, n_pb, n_ldc):
    if params.dim() == 1:
        params = params[None, :]
    if times.dtype != torch.float64 or params.dtype != torch.float64 or not (times.is_contiguous() and params.is_contiguous()):
        raise PtError("times and params must be contiguous float64")
    if not (times.is_cuda and params.is_cuda):
        raise PtError("times and params must be CUDA tensors (there is no CPU path)")
    n_pv = params.shape[0]
    if params.shape[1] != 7 + n_pb * n_ldc:
        raise PtError("Giménez parameter rows must hold 7 + n_pb*n_ldc doubles")
    if times.dim() == 1:
        n_t, stride = times.shape[0], 0
    elif times.dim() == 2 and times.shape[0] == n_pv:
        n_t, stride = times.shape[1], times.shape[1]
    else:
        raise PtError("times must be [n_t] or [n_pv][n_t]")
    return times, params, n_pv, n_t, stride


def pt_gimenez_exact(coef: GimenezCoef, times: torch.Tensor, params: torch.Tensor, n_pb: int = 1, n_ss: int = 1,
                     t_exp: float = 0.0, out: Optional[torch.Tensor] = None, status: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Giménez flux [n_pv][n_pb][n_t] by the series (include/pt.h: pt_gimenez_exact)."""
    times, params, n_pv, n_t, stride = _marshal_gimenez(times, params, n_pb, coef.n_ldc)
    if out is None:
        out = torch.empty((n_pv, n_pb, n_t), dtype=torch.float64, device=times.device)
    _check(lib().pt_gimenez_exact(coef.data.data_ptr(), coef.n_ldc, coef.n_j, times.data_ptr(), n_t, stride, params.data_ptr(),
                                  n_pv, n_pb, n_ss, float(t_exp), out.data_ptr(),
                                  status.data_ptr() if status is not None else None, _stream()), "pt_gimenez_exact")
    return out


def pt_gimenez_interp(coef: GimenezCoef, n_in: int, n_out: int, times: torch.Tensor, params: torch.Tensor, n_pb: int = 1,
                      n_ss: int = 1, t_exp: float = 0.0, out: Optional[torch.Tensor] = None,
                      work: Optional[torch.Tensor] = None, status: Optional[torch.Tensor] = None):
    """Giménez flux by interpolation in z (include/pt.h: pt_gimenez_interp); returns (flux, work) — work holds the tables
    [n_pv][n_ldc+1][n_in+n_out] the call filled."""
    times, params, n_pv, n_t, stride = _marshal_gimenez(times, params, n_pb, coef.n_ldc)
    if out is None:
        out = torch.empty((n_pv, n_pb, n_t), dtype=torch.float64, device=times.device)
    if work is None:
        work = torch.empty((n_pv, coef.n_ldc + 1, n_in + n_out), dtype=torch.float64, device=times.device)
    _check(lib().pt_gimenez_interp(coef.data.data_ptr(), coef.n_ldc, coef.n_j, n_in, n_out, work.data_ptr(), times.data_ptr(),
                                   n_t, stride, params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp), out.data_ptr(),
                                   status.data_ptr() if status is not None else None, _stream()), "pt_gimenez_interp")
    return out, work


def pt_gimenez_static_work_doubles() -> int:
    """Capacity, in doubles, of the library's fixed work area (include/pt.h: pt_gimenez_interp_static)."""
    return int(lib().pt_gimenez_static_work_doubles())


def pt_gimenez_interp_static(coef: GimenezCoef, n_in: int, n_out: int, times: torch.Tensor, params: torch.Tensor,
                             out: torch.Tensor, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0,
                             status: Optional[torch.Tensor] = None) -> torch.Tensor:
    """pt_gimenez_interp without any allocation (include/pt.h: pt_gimenez_interp_static): the z-tables live in the library's
    fixed work area and `out` [n_pv][n_pb][n_t] float64 must be given."""
    times, params, n_pv, n_t, stride = _marshal_gimenez(times, params, n_pb, coef.n_ldc)
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == n_pv * n_pb * n_t):
        raise PtError("out must be a contiguous CUDA float64 tensor of n_pv*n_pb*n_t elements")
    _check(lib().pt_gimenez_interp_static(coef.data.data_ptr(), coef.n_ldc, coef.n_j, n_in, n_out, times.data_ptr(), n_t, stride,
                                          params.data_ptr(), n_pv, n_pb, n_ss, float(t_exp), out.data_ptr(),
                                          status.data_ptr() if status is not None else None, _stream()),
           "pt_gimenez_interp_static")
    return out


def pt_probe_ffma(blocks: int, iters: int, sink: torch.Tensor) -> None:
    """FP32-pipe peak probe (include/pt.h: pt_probe_ffma); sink: CUDA float32 tensor of blocks*256 elements."""
    if not sink.is_cuda or sink.dtype != torch.float32 or sink.numel() < blocks * 256:
        raise PtError("sink must be a CUDA float32 tensor of at least blocks*256 elements")
    _check(lib().pt_probe_ffma(blocks, iters, sink.data_ptr(), _stream()), "pt_probe_ffma")


def pt_probe_dfma(blocks: int, iters: int, sink: torch.Tensor) -> None:
    """FP64-pipe peak probe (include/pt.h: pt_probe_dfma); sink: CUDA float64 tensor of blocks*256 elements."""
    if not sink.is_cuda or sink.dtype != torch.float64 or sink.numel() < blocks * 256:
        raise PtError("sink must be a CUDA float64 tensor of at least blocks*256 elements")
    _check(lib().pt_probe_dfma(blocks, iters, sink.data_ptr(), _stream()), "pt_probe_dfma")


def pt_plan(n_pv: int, n_t: int, n_sm: int = 148) -> dict:
    """Tiling and scheduling mode the flux kernels would use (include/pt.h: pt_plan); host logic only, works without a GPU."""
    out = (C.c_int64 * 4)()
    _check(lib().pt_plan(n_pv, n_t, n_sm, out), "pt_plan")
    return {"tile_len": int(out[0]), "tiles_per_pv": int(out[1]), "mode": int(out[2]), "blocks": int(out[3])}


def pt_launch_count() -> int:
    return int(lib().pt_launch_count())
