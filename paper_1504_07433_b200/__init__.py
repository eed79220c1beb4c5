"""B200-native batched quadratic Mandel–Agol transit model (the hot path of PyTransit, arXiv 1504.07433).

The product is the C-ABI CUDA library declared in include/pt.h; this package holds its sources (csrc/), the build
step (build.py), the thin ctypes binding (binding.py) and the seeded synthetic workloads (inputs.py).
"""
from .binding import (PT_F32, PT_F32S, PT_F64, SOLVERS, GimenezCoef, pt_gimenez_exact, pt_gimenez_interp, pt_gimenez_interp_static, pt_gimenez_static_work_doubles, pt_orbit_z_solver, PT_ST_BAD_PARAM, PT_ST_K_OUT_OF_TABLE, PtError, Table, pt_launch_count,  # noqa: F401
                      pt_ma_quad_chi2, pt_ma_quad_exact, pt_ma_quad_exact_pbk, pt_ma_quad_exact_host, pt_ma_quad_interp, pt_ma_quad_interp_host,
                      pt_ma_table_build, pt_orbit_z, pt_plan, pt_probe_dfma, pt_probe_ffma)
