"""ctypes loader for the CPU oracle (oracle/pt_oracle.cpp).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It never imports the CUDA package and the CUDA package never imports it.

`prec` selects the instantiation: "f64" (double, the timed CPU baseline) or "f128" (__float128, the parity arbiter;
results are rounded to double on return).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pt_oracle.cpp")
_LIB = os.path.join(_HERE, "libpt_oracle.so")
_lock = threading.Lock()
_lib = None

PREC = {"f64": 0, "f128": 1}


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no FMA contraction: the phase fold and subsample time are pinned IEEE ops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        cmd = ["g++", "-O2", "-std=gnu++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", tmp,
               "-lquadmath"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> C.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            _lib = C.CDLL(build())
            for name in ("pto_ma_basis", "pto_ellip", "pto_kepler", "pto_kepler_iter", "pto_true_anomaly_series", "pto_orbit_z", "pto_orbit_z_solver", "pto_gimenez_alpha", "pto_kopal_G", "pto_gimenez_exact", "pto_ma_quad_exact",
                         "pto_ma_table_build", "pto_ma_quad_interp", "pto_interp_basis", "pto_num_threads"):
                getattr(_lib, name).restype = C.c_int
            _lib.pto_set_num_threads.restype = None
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def num_threads() -> int:
    return int(lib().pto_num_threads())


def set_num_threads(n: int) -> None:
    lib().pto_set_num_threads(C.c_int(int(n)))


def ma_basis(k, z, prec: str = "f128"):
    """λe, λd*, ηd at matching arrays of radius ratio k and separation z."""
    k, z = np.broadcast_arrays(_f64(k), _f64(z))
    k, z = _f64(k), _f64(z)
    out = [np.empty(k.shape, np.float64) for _ in range(3)]
    rc = lib().pto_ma_basis(C.c_int(PREC[prec]), _p(k), _p(z), C.c_int64(k.size), *[_p(o) for o in out])
    assert rc == 0
    return tuple(out)


def ellip(m, n, prec: str = "f128"):
    """K(m), E(m), Π(n|m) — parameter form, minus-sign convention for n."""
    m, n = np.broadcast_arrays(_f64(m), _f64(n))
    m, n = _f64(m), _f64(n)
    out = [np.empty(m.shape, np.float64) for _ in range(3)]
    rc = lib().pto_ellip(C.c_int(PREC[prec]), _p(m), _p(n), C.c_int64(m.size), *[_p(o) for o in out])
    assert rc == 0
    return tuple(out)


def kepler(M, e, prec: str = "f128"):
    M, e = np.broadcast_arrays(_f64(M), _f64(e))
    M, e = _f64(M), _f64(e)
    E = np.empty(M.shape, np.float64)
    rc = lib().pto_kepler(C.c_int(PREC[prec]), _p(M), _p(e), C.c_int64(M.size), _p(E))
    assert rc == 0
    return E


def _shape_args(times, params, n_pb):
    times = _f64(times)
    params = _f64(params)
    if params.ndim == 1:
        params = params[None, :]
    n_pv = params.shape[0]
    assert params.shape[1] == 6 + 3 * n_pb, "parameter row must hold 6 + 3*n_pb doubles"
    if times.ndim == 1:
        n_t, stride = times.shape[0], 0
    else:
        assert times.shape[0] == n_pv
        n_t, stride = times.shape[1], times.shape[1]
    return times, params, n_pv, n_t, stride


def orbit_z(times, params, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0, prec: str = "f128"):
    """Signed projected separation [n_pv][n_t][n_ss]; negative = planet behind the star."""
    times, params, n_pv, n_t, stride = _shape_args(times, params, n_pb)
    z = np.empty((n_pv, n_t, n_ss), np.float64)
    rc = lib().pto_orbit_z(C.c_int(PREC[prec]), _p(times), C.c_int64(n_t), C.c_int64(stride), _p(params),
                           C.c_int64(n_pv), C.c_int32(n_pb), C.c_int32(n_ss), C.c_double(t_exp), _p(z))
    assert rc == 0, rc
    return z


SOLVERS = {"exact": 0, "newton": 1, "iter": 2, "ps3": 3, "ps5": 4, "fast": 5}


def orbit_z_solver(times, params, solver: str, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0, prec: str = "f128"):
    """Signed projected separation with one of the orbit routines of P:L31 (R19): 'exact'/'newton' (the Kepler
    solve), 'iter' (fixed-point iteration), 'ps3'/'ps5' (series of the equation of the centre), 'fast' (e-based dispatch)."""
    times, params, n_pv, n_t, stride = _shape_args(times, params, n_pb)
    out = np.empty((n_pv, n_t, n_ss), dtype=np.float64)
    rc = lib().pto_orbit_z_solver(C.c_int(PREC[prec]), C.c_int(SOLVERS[solver]), _p(times), C.c_int64(n_t), C.c_int64(stride),
                                  _p(params), C.c_int64(n_pv), C.c_int32(n_pb), C.c_int32(n_ss), C.c_double(t_exp), _p(out))
    if rc:
        raise RuntimeError("pto_orbit_z_solver failed: %d" % rc)
    return out


def kepler_iter(M, e, prec: str = "f128"):
    """E(M) by the fixed-point iteration E <- M + e sin E."""
    M, e = np.broadcast_arrays(_f64(M), _f64(e))
    M, e = np.ascontiguousarray(M), np.ascontiguousarray(e)
    out = np.empty_like(M)
    lib().pto_kepler_iter(C.c_int(PREC[prec]), _p(M), _p(e), C.c_int64(M.size), _p(out))
    return out


def true_anomaly_series(M, e, order: int, prec: str = "f128"):
    """True anomaly from the series of the equation of the centre truncated after e^order (order 3 or 5)."""
    M, e = np.broadcast_arrays(_f64(M), _f64(e))
    M, e = np.ascontiguousarray(M), np.ascontiguousarray(e)
    out = np.empty_like(M)
    rc = lib().pto_true_anomaly_series(C.c_int(PREC[prec]), C.c_int(order), _p(M), _p(e), C.c_int64(M.size), _p(out))
    if rc:
        raise RuntimeError("pto_true_anomaly_series failed: %d" % rc)
    return out


def ma_quad_exact(times, params, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0, prec: str = "f128"):
    """Relative flux [n_pv][n_pb][n_t] of the exact quadratic Mandel–Agol model."""
    times, params, n_pv, n_t, stride = _shape_args(times, params, n_pb)
    f = np.empty((n_pv, n_pb, n_t), np.float64)
    rc = lib().pto_ma_quad_exact(C.c_int(PREC[prec]), _p(times), C.c_int64(n_t), C.c_int64(stride), _p(params),
                                 C.c_int64(n_pv), C.c_int32(n_pb), C.c_int32(n_ss), C.c_double(t_exp), _p(f))
    assert rc == 0, rc
    return f


def table_spacing(k_min: float, k_max: float, n_k: int, z_max: float, n_z: int):
    """(dk, dz) exactly as the table builder forms them (IEEE double)."""
    return (np.float64(k_max) - np.float64(k_min)) / np.float64(n_k - 1), np.float64(z_max) / np.float64(n_z - 1)


def ma_table_build(k_min, k_max, n_k, z_max, n_z, dtype=np.float64, n_fn: int = 3, prec: str = "f128"):
    """(k,z) table [n_k][n_z][n_fn] of λe, λd*, ηd(, 0)."""
    dtype = np.dtype(dtype)
    code = {np.dtype(np.float64): 0, np.dtype(np.float32): 1}[dtype]
    tb = np.zeros((n_k, n_z, n_fn), dtype)
    rc = lib().pto_ma_table_build(C.c_int(PREC[prec]), C.c_double(k_min), C.c_double(k_max), C.c_int32(n_k),
                                  C.c_double(z_max), C.c_int32(n_z), C.c_int32(code), C.c_int32(n_fn), _p(tb))
    assert rc == 0, rc
    return tb


def ma_quad_interp(table, k_min, dk, dz, times, params, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0,
                   prec: str = "f128"):
    """Relative flux [n_pv][n_pb][n_t] by bilinear interpolation of `table`."""
    table = np.ascontiguousarray(table)
    code = {np.dtype(np.float64): 0, np.dtype(np.float32): 1}[table.dtype]
    n_k, n_z, n_fn = table.shape
    times, params, n_pv, n_t, stride = _shape_args(times, params, n_pb)
    f = np.empty((n_pv, n_pb, n_t), np.float64)
    rc = lib().pto_ma_quad_interp(C.c_int(PREC[prec]), _p(table), C.c_int32(code), C.c_int32(n_k), C.c_int32(n_z),
                                  C.c_int32(n_fn), C.c_double(k_min), C.c_double(dk), C.c_double(dz), _p(times),
                                  C.c_int64(n_t), C.c_int64(stride), _p(params), C.c_int64(n_pv), C.c_int32(n_pb),
                                  C.c_int32(n_ss), C.c_double(t_exp), _p(f))
    assert rc == 0, rc
    return f


def interp_basis(table, k_min, dk, dz, k, z, prec: str = "f128"):
    """The bilinear rule alone (S§8(c)-2 step 8): λe, λd*, ηd [n][3] looked up in `table` at (k, z)."""
    table = np.ascontiguousarray(table)
    code = {np.dtype(np.float64): 0, np.dtype(np.float32): 1}[table.dtype]
    n_k, n_z, n_fn = table.shape
    k, z = np.broadcast_arrays(_f64(k), _f64(z))
    k, z = _f64(k), _f64(z)
    out = np.empty((k.size, 3), np.float64)
    rc = lib().pto_interp_basis(C.c_int(PREC[prec]), _p(table), C.c_int32(code), C.c_int32(n_k), C.c_int32(n_z),
                                C.c_int32(n_fn), C.c_double(k_min), C.c_double(dk), C.c_double(dz), _p(k), _p(z),
                                C.c_int64(k.size), _p(out))
    assert rc == 0, rc
    return out.reshape(k.shape + (3,))


def chi2_of_flux(flux, obs, isig):
    """chi2[pv] = sum_{j,t} ((obs[j][t] - flux[pv][j][t]) * isig[j][t])^2 — the definition (the likelihood the
    paper proposes to evaluate on the GPU next to z), summed in extended precision over passbands and exposures."""
    flux = np.asarray(flux, dtype=np.longdouble)
    o = np.asarray(obs, dtype=np.longdouble).reshape(flux.shape[1:])
    w = np.asarray(isig, dtype=np.longdouble).reshape(flux.shape[1:])
    d = (o[None] - flux) * w[None]
    return np.asarray((d * d).sum(axis=(1, 2)), dtype=np.float64)


def ma_quad_chi2(times, params, obs, isig, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0, table=None,
                 prec: str = "f128"):
    """Fused-likelihood oracle: the exact (table is None) or interpolated flux of this module, then chi2_of_flux.
    table = (array, k_min, dk, dz)."""
    if table is None:
        f = ma_quad_exact(times, params, n_pb, n_ss, t_exp, prec)
    else:
        f = ma_quad_interp(table[0], table[1], table[2], table[3], times, params, n_pb, n_ss, t_exp, prec)
    return chi2_of_flux(f, obs, isig)


def ma_quad_exact_pbk(times, params, n_pb: int = 1, n_ss: int = 1, t_exp: float = 0.0, prec: str = "f128"):
    """Exact per-passband-k model (what the mean-k evaluation of P:L179 approximates): passband j is the
    single-passband model of the row [t0, P, a, i, e, w, k_j, u1_j, u2_j]."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    out = []
    for j in range(n_pb):
        row = np.concatenate([params[:, :6], params[:, 6 + 3 * j:9 + 3 * j]], axis=1)
        out.append(ma_quad_exact(times, row, 1, n_ss, t_exp, prec)[:, 0])
    return np.stack(out, axis=1)


# ---------------------------------------------------------------------------------------------------------------------
# Giménez model (R20)
def kopal_G(j: int, p: float, q: float, x, prec: str = "f128"):
    """Kopal's Jacobi polynomial G_j(p, q; x) = 2F1(-j, j+p; q; x) by its defining finite sum."""
    x = np.ascontiguousarray(_f64(x))
    out = np.empty_like(x)
    lib().pto_kopal_G(C.c_int(2 if prec == "defsum" else PREC[prec]), C.c_int(j), C.c_double(p), C.c_double(q), _p(x), C.c_int64(x.size), _p(out))
    return out


def gimenez_alpha(n: int, n_j: int, k, z, prec: str = "f128"):
    """α_n(k, z) of Eq. 3 with N_J = n_j terms beyond j = 0."""
    k, z = np.broadcast_arrays(_f64(k), _f64(z))
    k, z = np.ascontiguousarray(k), np.ascontiguousarray(z)
    out = np.empty_like(k)
    lib().pto_gimenez_alpha(C.c_int(PREC[prec]), C.c_int(n), C.c_int(n_j), _p(k), _p(z), C.c_int64(k.size), _p(out))
    return out


def gimenez_exact(times, params, n_pb: int = 1, n_ldc: int = 2, n_j: int = 40, n_ss: int = 1, t_exp: float = 0.0,
                  prec: str = "f128"):
    """Giménez flux [n_pv][n_pb][n_t]; rows [t0, P, a, i, e, w, k, u_1..u_N per passband]."""
    times, params = np.ascontiguousarray(_f64(times)), np.ascontiguousarray(_f64(params))
    if params.ndim == 1:
        params = params[None, :]
    n_pv = params.shape[0]
    assert params.shape[1] == 7 + n_pb * n_ldc
    if times.ndim == 1:
        n_t, stride = times.shape[0], 0
    else:
        assert times.shape[0] == n_pv
        n_t, stride = times.shape[1], times.shape[1]
    out = np.empty((n_pv, n_pb, n_t), dtype=np.float64)
    rc = lib().pto_gimenez_exact(C.c_int(PREC[prec]), _p(times), C.c_int64(n_t), C.c_int64(stride), _p(params), C.c_int64(n_pv),
                                 C.c_int32(n_pb), C.c_int32(n_ldc), C.c_int32(n_j), C.c_int32(n_ss), C.c_double(t_exp), _p(out))
    if rc:
        raise RuntimeError("pto_gimenez_exact failed: %d" % rc)
    return out


def gimenez_interp_alpha(tab_in, tab_out, k: float, z):
    """The z-interpolation of P:L165-L169 (R21) on given tables of one α_n: tab_in on n_in nodes uniform on
    [0, 1-k], tab_out on n_out nodes uniform on [1-k, 1+k]; linear interpolation inside the segment that holds z."""
    z = _f64(z)
    zi = np.linspace(0.0, 1.0 - k, len(tab_in))
    zo = np.linspace(1.0 - k, 1.0 + k, len(tab_out))
    return np.where(z < 1.0 - k, np.interp(z, zi, tab_in), np.interp(z, zo, tab_out))


def gimenez_interp_flux(tables, n_in: int, times, params, n_pb: int = 1, n_ldc: int = 2, n_ss: int = 1, t_exp: float = 0.0):
    """Flux of the interpolated Giménez model from GIVEN tables [n_pv][n_ldc+1][n_in+n_out] (R21): orbit of this
    oracle in quad, linear interpolation of every α_n in the segment that holds z, Eq. 7-9, supersample mean."""
    times, params = _f64(times), _f64(params)
    n_pv = params.shape[0]
    tt = np.broadcast_to(times, (n_pv, times.shape[-1])) if times.ndim == 1 else times
    n_t = tt.shape[1]
    orow = np.concatenate([params[:, :7], np.zeros((n_pv, 2))], axis=1)
    z = orbit_z(tt if times.ndim == 2 else times, orow, 1, n_ss, t_exp, prec="f128")          # [n_pv][n_t][n_ss]
    out = np.ones((n_pv, n_pb, n_t))
    for pv in range(n_pv):
        k = params[pv, 6]
        u = params[pv, 7:].reshape(n_pb, n_ldc)
        nn = np.arange(1, n_ldc + 1)
        den = 1.0 - (nn * u / (nn + 2.0)).sum(axis=1)
        Cc = np.concatenate([((1.0 - u.sum(axis=1)) / den)[:, None], u / den[:, None]], axis=1)      # [n_pb][n_ldc+1]
        zz = z[pv]
        intr = (zz >= 0) & (zz < 1.0 + k)
        an = np.zeros((n_ldc + 1,) + zz.shape)
        for n in range(n_ldc + 1):
            an[n] = np.where(intr, gimenez_interp_alpha(tables[pv, n, :n_in], tables[pv, n, n_in:], k, np.abs(zz)), 0.0)
        abar = an.mean(axis=2)                                                                         # [n_ldc+1][n_t]
        out[pv] = 1.0 - Cc @ abar
        out[pv][:, ~intr.any(axis=1)] = 1.0
    return out
