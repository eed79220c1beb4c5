"""Parity of the CUDA path (through the C ABI, via the thin binding) against the CPU oracle's __float128 instantiation
on the same seeded inputs.  Gates (BASELINE.json north_star): exact fp64 flux 1e-12 abs; fp32 variant 2e-6 abs;
interpolated path vs the oracle's interpolation of the SAME table 1e-12 abs."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_1504_07433_b200 import inputs  # noqa: E402

TOL64 = 1e-12
TOL32 = 2e-6


@pytest.fixture(scope="module")
def pt():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1504_07433_b200 as pkg
    from paper_1504_07433_b200 import binding
    assert binding.lib().pt_build_arch() == 100
    return pkg


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def gpu_exact(pt, w, dtype=torch.float64, status=None):
    f = pt.pt_ma_quad_exact(dev(w.times), dev(w.params), w.n_pb, w.n_ss, w.t_exp, dtype=dtype, status=status)
    torch.cuda.synchronize()
    return f.cpu().numpy()


def ora_exact(oracle, w, prec="f128"):
    return oracle.ma_quad_exact(w.times, w.params, w.n_pb, w.n_ss, w.t_exp, prec=prec)


def oz64(oracle):
    return lambda t, p: oracle.orbit_z(t, p, prec="f64")[:, :, 0]


# ------------------------------------------------------------------------------------------- exact path, configs 1-3, 5
def test_config1_full(pt, oracle, golden_config1):
    w = inputs.config1()
    f = gpu_exact(pt, w)
    assert f.shape == (1, 1, 1000)
    assert np.abs(f - ora_exact(oracle, w)).max() <= TOL64
    # and straight against the stored worked example (values from the integral definitions)
    w2 = inputs.Workload("g", golden_config1[:, 0].copy(), w.params)
    assert np.abs(gpu_exact(pt, w2)[0, 0] - golden_config1[:, 2]).max() <= TOL64
    z = pt.pt_orbit_z(dev(w2.times), dev(w2.params)).cpu().numpy()[0, :, 0]
    assert np.abs(z - golden_config1[:, 1]).max() <= 1e-13


@pytest.mark.parametrize("n_pv,n_t,n_ss", [(8, 5000, 10), (3, 1024, 10), (5, 1025, 3), (2, 2047, 1), (4, 700, 32),
                                           (3, 333, 33), (2, 100, 70), (6, 1, 10), (2, 4097, 7)])
def test_config2_reduced_supersampled(pt, oracle, n_pv, n_t, n_ss):
    w = inputs.config2(n_pv=n_pv, n_t=n_t)
    w.n_ss = n_ss
    f = gpu_exact(pt, w)
    r = ora_exact(oracle, w)
    assert np.abs(f - r).max() <= TOL64
    assert np.array_equal(f == 1.0, r == 1.0)   # out-of-transit samples are exactly 1 on both sides


def test_config3_full_multipassband(pt, oracle):
    w = inputs.config3()
    f = gpu_exact(pt, w)
    assert f.shape == (512, 20, 600)
    assert np.abs(f - ora_exact(oracle, w)).max() <= TOL64


@pytest.mark.parametrize("n_pb,n_t", [(1, 599), (3, 601), (20, 77), (64, 130)])
def test_config3_ragged(pt, oracle, n_pb, n_t):
    w = inputs.config3(n_pv=7, n_pb=n_pb, n_t=n_t)
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64


@pytest.mark.parametrize("order", ["sorted", "shuffled"])
def test_config5_reduced(pt, oracle, order):
    w = inputs.config5(oz64(oracle), n_pv=192, n_t=1100, order=order)
    f = gpu_exact(pt, w)
    r = ora_exact(oracle, w)
    err = np.abs(f - r)
    assert err.max() <= TOL64, (err.max(), np.unravel_index(np.argmax(err), err.shape))
    z = pt.pt_orbit_z(dev(w.times), dev(w.params)).cpu().numpy()
    zr = oracle.orbit_z(w.times, w.params, prec="f128")
    assert np.abs(z - zr).max() <= 2e-13 * 20
    assert np.array_equal(np.signbit(z), np.signbit(zr))


def test_high_eccentricity_and_long_baseline(pt, oracle):
    rng = np.random.default_rng(11)
    n = 64
    P = rng.uniform(1, 10, n)
    e = np.concatenate([rng.uniform(0.6, 0.95, n // 2), rng.uniform(0.95, 0.99, n // 2)])
    wv = rng.uniform(0, 2 * math.pi, n)
    a = rng.uniform(8, 30, n)
    b = rng.uniform(0, 0.9, n)
    inc = np.arccos(np.clip(b * (1 + e * np.sin(wv)) / (a * (1 - e * e)), -1, 1))
    params = np.stack([P * rng.uniform(0, 1, n), P, a, inc, e, wv, rng.uniform(0.02, 0.3, n), 0.4 + 0 * P, 0.2 + 0 * P], 1)
    times = np.sort(rng.uniform(0, 3000, 6000))   # whole orbits, ~3000 d baseline (phase fold at |x| ~ 1e3)
    w = inputs.Workload("ecc", times, params)
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64
    z = pt.pt_orbit_z(dev(times), dev(params)).cpu().numpy()
    zr = oracle.orbit_z(times, params, prec="f128")
    assert np.abs(z - zr).max() <= 1e-11


# ------------------------------------------------------------------------------------------- NEXT-3: the other orbit routines
@pytest.mark.parametrize("solver", ["newton", "iter", "ps3", "ps5", "fast"])
def test_orbit_solvers_parity(pt, oracle, solver):
    # Each routine of P:L31 against the SAME routine of the oracle in __float128 (R19).  Both sides evaluate the
    # same mathematical function (the root of Kepler's equation, or the same truncated series), so the tolerance is the
    # rounding of the fp64 evaluation: |Δz| <= a (1+e)/(1-e) x (a few ulp of the anomaly) — 1e-11 covers a <= 30, e <= 0.6;
    # the iteration stops when E moves by less than an ulp, i.e. within e/(1-e) ulp of its fixed point.
    rng = np.random.default_rng(41)
    n = 96
    P, a = rng.uniform(1, 10, n), rng.uniform(3, 30, n)
    emax = 0.6 if solver in ("newton", "iter", "fast") else 0.2
    e = rng.uniform(0, emax, n)
    e[:8] = [0.0, 1e-9, 0.004, 0.006, 0.0061, 0.03, 0.0301, 0.1]
    pe = np.stack([P * rng.uniform(0, 1, n), P, a, np.arccos(rng.uniform(0, 0.95, n) / a), e, rng.uniform(0, 2 * math.pi, n),
                   rng.uniform(0.02, 0.3, n), 0.3 + 0 * P, 0.2 + 0 * P], axis=1)
    pe[40, 1] = -1.0                                       # a bad row stays NaN whatever the routine
    t = np.sort(rng.uniform(0, 100, 1500))
    z = pt.pt_orbit_z_solver(dev(t), dev(pe), solver).cpu().numpy()
    zr = oracle.orbit_z_solver(t, pe, solver, prec="f128")
    assert np.array_equal(np.isnan(z), np.isnan(zr)) and np.all(np.isnan(z[40]))
    ok = ~np.isnan(zr)
    assert np.abs(z[ok] - zr[ok]).max() <= 1e-11
    # supersampled and per-row times through the same entry point
    tt = np.sort(rng.uniform(0, 50, (n, 64)), axis=1)
    z2 = pt.pt_orbit_z_solver(dev(tt), dev(pe), solver, 1, 3, 0.02).cpu().numpy()
    zr2 = oracle.orbit_z_solver(tt, pe, solver, 1, 3, 0.02, prec="f128")
    ok = ~np.isnan(zr2)
    assert np.abs(z2[ok] - zr2[ok]).max() <= 1e-11
    if solver in ("newton", "fast"):
        # exact routines: also the plain entry point; the dispatch picks the series only where its error is below 2e-9 rad
        zx = pt.pt_orbit_z(dev(t), dev(pe)).cpu().numpy()
        okx = ~np.isnan(zx)
        bound = (a * (1 + e) / (1 - e) * 2.1e-9)[:, None, None] + 1e-11
        assert np.all((np.abs(np.abs(z) - np.abs(zx)) <= bound)[okx])
        if solver == "newton":
            assert np.array_equal(z[okx], zx[okx])


def test_orbit_solver_argument_errors(pt):
    from paper_1504_07433_b200 import binding
    t = torch.zeros(8, dtype=torch.float64, device="cuda")
    p = torch.zeros((1, 9), dtype=torch.float64, device="cuda")
    o = torch.zeros(8, dtype=torch.float64, device="cuda")
    L = binding.lib()
    assert L.pt_orbit_z_solver(t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 1, 0.0, 6, o.data_ptr(), None) == binding.PT_ERR_SIZE
    assert L.pt_orbit_z_solver(t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 1, 0.0, -1, o.data_ptr(), None) == binding.PT_ERR_SIZE
    assert L.pt_orbit_z_solver(None, 8, 0, p.data_ptr(), 1, 1, 1, 0.0, 2, o.data_ptr(), None) == binding.PT_ERR_NULL


# ------------------------------------------------------------------------------------------- degenerate inputs
def test_edge_cases_k_and_geometry(pt, oracle):
    t = np.linspace(-0.3, 0.3, 1501)
    rows = []
    for k in (0.0, 1e-8, 0.5, 0.999, 1.0, 1.5, 3.0):
        for b in (0.0, 0.5, 1.0 + k, 1.0 + k + 1e-9):
            a = 6.0
            rows.append([0.0, 2.0, a, math.acos(min(1.0, b / a)), 0.0, 0.0, k, 0.3, 0.25])
    rows.append([0.0, 2.0, 1.2, math.pi / 2, 0.0, 0.0, 0.4, 0.3, 0.25])    # a < 1+k: always overlapping on the near side
    rows.append([0.0, 2.0, 6.0, 0.0, 0.0, 0.0, 0.1, 0.3, 0.25])            # face-on orbit, never transits
    rows.append([0.0, 2.0, 1.5, 1.2, 0.5, 0.3, 0.2, 0.3, 0.25])            # a(1-e) < 1+k
    rows.append([0.1, 2.0, 6.0, math.pi / 2, 0.0, 0.0, 0.1, 0.0, 0.0])     # uniform disk
    w = inputs.Workload("edge", t, np.array(rows))
    f, r = gpu_exact(pt, w), ora_exact(oracle, w)
    assert np.abs(f - r).max() <= TOL64
    # supersampled, exposure longer than the transit
    w.n_ss, w.t_exp = 5, 0.2
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64


def test_exact_equality_special_cases_via_orbit(pt, oracle):
    """b chosen so that z(t0) hits z = k, 1-k, 0 to within an ulp; plus the k = 1/2 neighbourhood."""
    rows = []
    a = 8.0
    for k in (0.1, 0.3, 0.5, 0.5 + 1e-9, 0.5 - 1e-9, 0.7):
        for zt in (k, abs(1 - k), 0.0, 1 + k, k * (1 + 1e-15), abs(1 - k) * (1 - 1e-15)):
            rows.append([0.0, 3.0, a, math.acos(zt / a), 0.0, 0.0, k, 0.5, 0.1])
    w = inputs.Workload("eq", np.array([0.0, 1e-9, -1e-9, 1e-6, 3.0, 1e-4]), np.array(rows))
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64


def test_bad_parameters_nan_rows_and_status(pt, oracle):
    w = inputs.config2(n_pv=9, n_t=2100)
    p = w.params
    p[1, 1] = -1.0; p[2, 4] = 1.0; p[3, 6] = -0.1; p[4, 2] = np.nan; p[6, 7] = 3.0; p[6, 8] = 0.0   # last: 1 - u1/3 = 0
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    f = gpu_exact(pt, w, status=st)
    r = ora_exact(oracle, w, "f64")
    assert np.array_equal(np.isnan(f), np.isnan(r))
    assert np.all(np.isnan(f[[1, 2, 3, 4, 6]])) and np.all(np.isfinite(f[[0, 5, 7, 8]]))
    assert st.cpu().tolist() == [pt.PT_ST_BAD_PARAM, 5]
    z = pt.pt_orbit_z(dev(w.times), dev(p)).cpu().numpy()
    assert np.all(np.isnan(z[[1, 2, 3, 4, 6]])) and np.all(np.isfinite(z[0]))


def test_argument_errors(pt):
    from paper_1504_07433_b200 import binding
    L = binding.lib()
    t = torch.zeros(8, dtype=torch.float64, device="cuda")
    p = torch.zeros((1, 9), dtype=torch.float64, device="cuda")
    o = torch.zeros(8, dtype=torch.float64, device="cuda")
    assert L.pt_ma_quad_exact(None, 8, 0, p.data_ptr(), 1, 1, 1, 0.0, 0, o.data_ptr(), None, None) == binding.PT_ERR_NULL
    assert L.pt_ma_quad_exact(t.data_ptr(), 0, 0, p.data_ptr(), 1, 1, 1, 0.0, 0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
    assert L.pt_ma_quad_exact(t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 0, 0.0, 0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
    assert L.pt_ma_quad_exact(t.data_ptr(), 8, 4, p.data_ptr(), 1, 1, 1, 0.0, 0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
    assert L.pt_ma_quad_exact(t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 1, 0.0, 7, o.data_ptr(), None, None) == binding.PT_ERR_DTYPE
    assert L.pt_ma_table_build(0.1, 0.05, 4, 1.2, 4, 0, 3, o.data_ptr(), None) == binding.PT_ERR_SIZE
    bad = binding.pt_table(None, 0, 4, 4, 3, 0.0, 0.1, 0.1)
    import ctypes as C
    assert L.pt_ma_quad_interp(C.byref(bad), t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 1, 0.0, 0, o.data_ptr(), None, None) == binding.PT_ERR_TABLE
    with pytest.raises(binding.PtError):
        pt.pt_ma_quad_exact(t.cpu(), p.cpu())


def test_unaligned_output_and_odd_row_length(pt, oracle):
    w = inputs.config2(n_pv=3, n_t=1501)
    w.n_ss = 2
    buf = torch.empty(3 * 1501 + 1, dtype=torch.float64, device="cuda")
    out = buf[1:].view(3, 1, 1501)    # 8-byte aligned only
    pt.pt_ma_quad_exact(dev(w.times), dev(w.params), 1, 2, w.t_exp, out=out)
    assert np.abs(out.cpu().numpy() - ora_exact(oracle, w)).max() <= TOL64


# ------------------------------------------------------------------------------------------- fp32 variant
@pytest.mark.parametrize("cfg", ["c2", "c3", "c5"])
def test_fp32_variant(pt, oracle, cfg):
    w = {"c2": lambda: inputs.config2(n_pv=8, n_t=3000), "c3": lambda: inputs.config3(n_pv=32),
         "c5": lambda: inputs.config5(oz64(oracle), n_pv=96, n_t=600)}[cfg]()
    f = gpu_exact(pt, w, dtype=torch.float32)
    assert f.dtype == np.float32
    assert np.abs(f.astype(np.float64) - ora_exact(oracle, w)).max() <= TOL32


def test_fp32_store_only_mode_is_fp64_arithmetic(pt, oracle):
    # PT_F32S: fp64 arithmetic, float storage: equals the fp64 flux rounded to float
    w = inputs.config5(oz64(oracle), n_pv=64, n_t=512)
    f64 = gpu_exact(pt, w)
    f = pt.pt_ma_quad_exact(dev(w.times), dev(w.params), dtype=torch.float32, fp32_store_only=True)
    torch.cuda.synchronize()
    assert np.array_equal(f.cpu().numpy(), f64.astype(np.float32))


@pytest.mark.parametrize("u", [(0.4, 0.2), (0.0, 0.0), (0.9, -0.1), (0.0, 1.0)])
def test_fp32_arith_h5_grid(pt, oracle, u):
    # the region where fp32 λd* is worst — small k, close to the inner contact — on an explicit grid:
    # k in {0.01, 0.05, 0.1, 0.4}, |z - (1-k)| in {1e-6, 1e-4, 1e-2}, plus z = k, z -> 0 and the outer contact.
    # Circular orbit seen edge-on (i = π/2): z(t) = a |sin(2π t / P)|, so a wanted z is the time P/(2π) asin(z/a).
    # (0, 1) is an extreme law whose coefficients send the row to fp64 arithmetic (f32_ok): it must hold the gate too.
    a, P = 10.0, 3.0
    rows, times = [], []
    for k in (0.01, 0.05, 0.1, 0.4):
        zs = [1e-7, 0.5 * k, k, k * (1 + 1e-5), 0.5, 1.0 + k - 1e-4, 1.0 + k - 1e-2]
        for d in (1e-6, 1e-4, 1e-2):
            zs += [1.0 - k - d, 1.0 - k + d]
        zs.append(1.0 - k)
        zs = np.array(zs)
        times.append(P / (2 * np.pi) * np.arcsin(zs / a))
        rows.append([0.0, P, a, 0.5 * np.pi, 0.0, 0.0, k, u[0], u[1]])
    params = np.array(rows)
    t = np.array(times)
    f = pt.pt_ma_quad_exact(dev(t), dev(params), dtype=torch.float32)
    torch.cuda.synchronize()
    ref = oracle.ma_quad_exact(t, params, prec="f128")
    err = np.abs(f.cpu().numpy().astype(np.float64) - ref)
    assert err.max() <= TOL32, (err.max(), np.unravel_index(err.argmax(), err.shape))


def test_fp32_arith_dense_eccentric_and_shared_axis(pt, oracle):
    # the two kernels that have the fp32 path: per-row times (eccentric, n_ss = 1) and the shared ascending axis (epoch
    # kernel, supersampled), both at sizes that span many tiles
    w = inputs.dense_transit(n_pv=256, n_t=1024)
    f = gpu_exact(pt, w, dtype=torch.float32)
    err = np.abs(f.astype(np.float64) - ora_exact(oracle, w, "f64")).max()
    assert err <= TOL32, err
    w = inputs.config2(n_pv=48, n_t=6000)
    f = gpu_exact(pt, w, dtype=torch.float32)
    err = np.abs(f.astype(np.float64) - ora_exact(oracle, w, "f64")).max()
    assert err <= TOL32, err
    assert (f == 1.0).mean() > 0.9                       # out of transit: exactly 1


@pytest.mark.parametrize("n_pv,n_t,kind", [(300, 100, "dense"), (64, 3000, "dense"), (40, 3001, "dense"), (7, 40000, "sparse"),
                                           (33, 2049, "sparse"), (3, 1, "dense")])
def test_direct_kernel_shapes(pt, oracle, n_pv, n_t, kind):
    """The direct kernel (fp32 variant, per-row times, n_ss = 1): one tile per row (records per tile) and several (records from
    prep_kernel), odd row lengths (no 16-byte loads), rows dense and sparse in transits (full and ragged list rounds, passes
    that leave a remainder), a bad row and a row the rule keeps in fp64 arithmetic — every element written, gate 2e-6."""
    if kind == "dense":
        w = inputs.dense_transit(n_pv=n_pv, n_t=n_t)
        times, params = w.times, w.params
    else:
        w = inputs.config2(n_pv=n_pv, n_t=n_t)
        rng = np.random.default_rng(n_t)
        times = np.ascontiguousarray(w.times[None, :] + rng.uniform(0.0, 0.01, (n_pv, 1)))
        params = w.params.copy()
    params = params.copy()
    if n_pv > 2:
        params[1, 1] = -1.0                  # bad row: NaN
        params[2, 6] = 0.75                  # k > 0.7: the rule keeps this row in fp64 arithmetic (f32_ok)
    out = torch.full((n_pv, 1, n_t), float("nan"), dtype=torch.float32, device="cuda")
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    pt.pt_ma_quad_exact(dev(times), dev(params), 1, 1, 0.0, out=out, status=st)
    torch.cuda.synchronize()
    f = out.cpu().numpy().astype(np.float64)
    r = oracle.ma_quad_exact(times, params, 1, 1, 0.0, prec="f64")
    assert np.array_equal(np.isnan(f), np.isnan(r))
    ok = ~np.isnan(r)
    assert np.abs(f[ok] - r[ok]).max() <= TOL32
    if n_pv > 2:
        assert np.all(np.isnan(f[1])) and st.cpu().tolist() == [pt.PT_ST_BAD_PARAM, 1]


# ------------------------------------------------------------------------------------------- table + interpolated path
def _table_cfg(small=True):
    return dict(k_min=0.05, k_max=0.25, n_k=41, z_max=1.25, n_z=1251) if small else inputs.config4(1, 1).table


@pytest.mark.parametrize("dtype,n_fn", [(torch.float64, 3), (torch.float32, 4), (torch.float64, 4), (torch.float32, 3)])
def test_table_build_parity(pt, oracle, dtype, n_fn):
    c = _table_cfg()
    tb = pt.pt_ma_table_build(dtype=dtype, n_fn=n_fn, **c)
    torch.cuda.synchronize()
    ref = oracle.ma_table_build(c["k_min"], c["k_max"], c["n_k"], c["z_max"], c["n_z"],
                                np.float64 if dtype == torch.float64 else np.float32, n_fn, "f128")
    got = tb.data.cpu().numpy()
    tol = 1e-14 if dtype == torch.float64 else 6e-8
    assert np.abs(got.astype(np.float64) - ref.astype(np.float64)).max() <= tol
    dk, dz = oracle.table_spacing(c["k_min"], c["k_max"], c["n_k"], c["z_max"], c["n_z"])
    assert tb.dk == dk and tb.dz == dz


@pytest.mark.parametrize("tdtype,n_fn", [(torch.float64, 3), (torch.float32, 4)])
def test_interp_vs_oracle_interp_of_same_table(pt, oracle, tdtype, n_fn):
    c = _table_cfg()
    tb = pt.pt_ma_table_build(dtype=tdtype, n_fn=n_fn, **c)
    w = inputs.config4(n_pv=24, n_t=5003)
    w.params[3, 6] = 0.3     # off the table: exact fallback + status bit
    w.params[5, 6] = 0.25    # last node
    w.params[6, 6] = 0.05    # first node
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    f = pt.pt_ma_quad_interp(tb, dev(w.times), dev(w.params), status=st).cpu().numpy()
    host_tb = tb.data.cpu().numpy()      # the SAME table, downloaded
    r = oracle.ma_quad_interp(host_tb, tb.k_min, tb.dk, tb.dz, w.times, w.params, prec="f128")
    assert np.abs(f - r).max() <= TOL64
    assert st.cpu().tolist() == [pt.PT_ST_K_OUT_OF_TABLE, 1]
    # reported, not gated: error against the exact model
    fe = ora_exact(oracle, w)
    err = np.abs(f - fe)
    print("interp vs exact: max %.3e mean(in transit) %.3e" % (err.max(), err[fe < 1].mean()))
    assert err.max() < 5e-5
    # supersampled + multi-passband through the table
    w3 = inputs.config3(n_pv=5, n_pb=4, n_t=300)
    w3.n_ss, w3.t_exp = 3, 0.002
    f3 = pt.pt_ma_quad_interp(tb, dev(w3.times), dev(w3.params), 4, 3, w3.t_exp).cpu().numpy()
    r3 = oracle.ma_quad_interp(host_tb, tb.k_min, tb.dk, tb.dz, w3.times, w3.params, 4, 3, w3.t_exp, prec="f128")
    assert np.abs(f3 - r3).max() <= TOL64


# ------------------------------------------------------------------------------------------- host-buffer entry points
def test_host_entry_points(pt, oracle):
    w = inputs.config2(n_pv=4, n_t=3000)
    t, p = torch.from_numpy(w.times).pin_memory(), torch.from_numpy(w.params).pin_memory()
    out = torch.empty((4, 1, 3000), dtype=torch.float64).pin_memory()
    st = torch.zeros(2, dtype=torch.int32)
    pt.pt_ma_quad_exact_host(t, p, out, 1, w.n_ss, w.t_exp, status=st)
    assert np.abs(out.numpy() - ora_exact(oracle, w)).max() <= TOL64 and st.tolist() == [0, 0]
    tb = pt.pt_ma_table_build(**_table_cfg())
    w.n_ss = 1
    pt.pt_ma_quad_interp_host(tb, t, p, out, 1, 1, 0.0)
    r = oracle.ma_quad_interp(tb.data.cpu().numpy(), tb.k_min, tb.dk, tb.dz, w.times, w.params, prec="f128")
    assert np.abs(out.numpy() - r).max() <= TOL64


# ------------------------------------------------------------------------------------------- full sizes, sampled
def test_config2_full_size_all_rows(pt, oracle):
    """BASELINE configs[1] exactly as bench.py launches it (LPT tile order, record cache, dependent launch, range mode):
    every one of the 64 rows against the quad oracle."""
    w = inputs.config2()
    f = gpu_exact(pt, w)
    assert f.shape == (64, 1, 60000)
    r = ora_exact(oracle, w)
    assert np.abs(f - r).max() <= TOL64
    assert np.array_equal(f == 1.0, r == 1.0)
    # properties that hold at any size: bounded, exactly 1 away from transit (checked through the product's own z)
    assert f.max() == 1.0 and f.min() > 0.9
    z = pt.pt_orbit_z(dev(w.times), dev(w.params), 1, w.n_ss, w.t_exp).cpu().numpy()
    k = w.params[:, 6][:, None]
    out = np.all((z < 0) | (z >= 1 + k[:, :, None]), axis=2)
    assert np.all(f[:, 0][out] == 1.0) and np.all(f[:, 0][~out] < 1.0)


def test_config4_full_size_sampled(pt, oracle):
    """BASELINE configs[3] at full size; 256 rows drawn by seed (plus the first and last) against the oracle's interpolation
    of the SAME downloaded table; every other row through size-independent properties."""
    w = inputs.config4()
    c = w.table
    rows = np.unique(np.concatenate([[0, 4095], np.random.default_rng(404).choice(4096, 256, replace=False)]))
    ws = inputs.Workload("s", w.times, w.params[rows])
    fe = ora_exact(oracle, ws)
    res = {}
    for tdtype, n_fn in ((torch.float32, 4), (torch.float64, 3)):
        tb = pt.pt_ma_table_build(dtype=tdtype, n_fn=n_fn, **c)
        f = pt.pt_ma_quad_interp(tb, dev(w.times), dev(w.params))
        torch.cuda.synchronize()
        host_rows = f[torch.from_numpy(rows).cuda()].cpu().numpy()
        host_tb = tb.data.cpu().numpy()
        r = oracle.ma_quad_interp(host_tb, tb.k_min, tb.dk, tb.dz, ws.times, ws.params, prec="f128")
        assert np.abs(host_rows - r).max() <= TOL64
        assert np.array_equal(host_rows == 1.0, r == 1.0)
        err = np.abs(host_rows - fe)
        res[str(tdtype)] = (err.max(), err[fe < 1].mean())
        assert err.max() < 2e-6          # reported, not gated (S§8(d) expects ~2.5e-7 max): a loose sanity bound
        assert float(f.max()) == 1.0 and float(f.min()) > 0.9
        # all rows: exactly 1 where the product's own orbit stage says "no overlap", below 1 elsewhere
        for lo in range(0, 4096, 512):
            z = pt.pt_orbit_z(dev(w.times), dev(w.params[lo:lo + 512]))[:, :, 0]
            k = dev(w.params[lo:lo + 512, 6])[:, None]
            out = (z < 0) | (z >= 1 + k)
            blk = f[lo:lo + 512, 0]
            assert bool((blk[out] == 1.0).all()) and bool((blk[~out] < 1.0).all())
            del z, out, blk
        del f, tb
    print("config4 interp vs exact (max, mean in transit):", res)


def test_config5_full_size_sampled(pt, oracle):
    """BASELINE configs[4] at full size: 256 rows by seed, at least 32 from each of the four population groups."""
    w = inputs.config5(oz64(oracle))
    assert w.n_eval == 2 ** 24
    f = gpu_exact(pt, w)
    rng = np.random.default_rng(505)
    grp = w.meta["groups"]
    rows = np.unique(np.concatenate([rng.choice(np.flatnonzero(grp == g), 64, replace=False) for g in range(4)]))
    assert len(rows) == 256
    ws = inputs.Workload("s", w.times[rows], w.params[rows])
    r = ora_exact(oracle, ws)
    err = np.abs(f[rows] - r)
    assert err.max() <= TOL64, err.max()
    # Kipping's (q1,q2) keep the intensity profile non-negative, so the true flux lies in (0, 1]
    assert f.max() <= 1.0 and f.min() > 0.0


# ------------------------------------------------------------------------------------------- pipeline mechanics
def test_bitwise_reproducible_across_launches(pt):
    """Tiles are dealt to warps dynamically, so the split of an exposure's subsamples over basis rounds differs from
    launch to launch; the fixed-point supersample sum makes the flux independent of it."""
    w = inputs.config2(n_pv=16, n_t=20000)
    t, p = dev(w.times), dev(w.params)
    ref = pt.pt_ma_quad_exact(t, p, 1, w.n_ss, w.t_exp).clone()
    for n_ss in (w.n_ss, 7, 33):
        ref = pt.pt_ma_quad_exact(t, p, 1, n_ss, w.t_exp).clone()
        for _ in range(5):
            again = pt.pt_ma_quad_exact(t, p, 1, n_ss, w.t_exp)
            assert torch.equal(ref.view(torch.int64), again.view(torch.int64))


@pytest.mark.parametrize("n_pv,n_t,n_ss,n_pb", [(3000, 7, 4, 1), (3000, 5, 1, 1), (700, 33, 1, 3), (300, 61, 5, 2), (257, 1, 1, 1)])
def test_many_short_rows(pt, oracle, n_pv, n_t, n_ss, n_pb):
    """More parameter vectors than warps, rows far shorter than a tile: every tile is ragged and queues cross tiles."""
    w = inputs.config3(n_pv=n_pv, n_pb=n_pb, n_t=n_t)
    w.n_ss, w.t_exp = n_ss, 0.004
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64


def test_long_exposure_many_subsamples(pt, oracle):
    """n_ss > 32: an exposure is expanded in several sub-rounds with basis rounds in between; exposures that are only
    partly in transit and exposures whose subsamples all miss the star sit next to each other."""
    w = inputs.config2(n_pv=6, n_t=1500)
    for n_ss, t_exp in ((97, 0.08), (64, 0.02), (200, 0.3)):
        w.n_ss, w.t_exp = n_ss, t_exp
        f, r = gpu_exact(pt, w), ora_exact(oracle, w)
        assert np.abs(f - r).max() <= TOL64
        assert np.array_equal(f == 1.0, r == 1.0)


def test_scheduler_slots_are_reused_cleanly(pt, oracle):
    """More launches than the library has scheduler slots: each launch must leave its slot zeroed."""
    w = inputs.config2(n_pv=2, n_t=700)
    t, p = dev(w.times), dev(w.params)
    out = torch.empty((2, 1, 700), dtype=torch.float64, device="cuda")
    for _ in range(4096 + 300):
        pt.pt_ma_quad_exact(t, p, 1, w.n_ss, w.t_exp, out=out)
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy() - ora_exact(oracle, w)).max() <= TOL64


def test_concurrent_streams(pt, oracle):
    """Launches on two streams overlap on the device; each has its own scheduler slot."""
    wa, wb = inputs.config2(n_pv=24, n_t=30000), inputs.config5(oz64(oracle), n_pv=256, n_t=1024)
    ta, pa, tb_, pb = dev(wa.times), dev(wa.params), dev(wb.times), dev(wb.params)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    outs = []
    for _ in range(4):
        with torch.cuda.stream(sa):
            fa = pt.pt_ma_quad_exact(ta, pa, 1, wa.n_ss, wa.t_exp)
        with torch.cuda.stream(sb):
            fb = pt.pt_ma_quad_exact(tb_, pb)
        outs.append((fa, fb))
    torch.cuda.synchronize()
    ra, rb = ora_exact(oracle, wa), ora_exact(oracle, wb)
    for fa, fb in outs:
        assert np.abs(fa.cpu().numpy() - ra).max() <= TOL64
        assert np.abs(fb.cpu().numpy() - rb).max() <= TOL64


# ------------------------------------------------------------------------------------------- fused likelihood (NEXT-1)
def _data_for(oracle, w, truth_row=0, sigma=2e-4, seed=3):
    """Synthetic observations: the oracle's flux of one parameter vector plus seeded Gaussian noise."""
    wt = inputs.Workload("truth", w.times, w.params[truth_row:truth_row + 1], w.n_pb, w.n_ss, w.t_exp)
    f = ora_exact(oracle, wt, "f64")[0]
    rng = np.random.default_rng(seed)
    obs = f + sigma * rng.standard_normal(f.shape)
    isig = np.full(f.shape, 1.0 / sigma) * rng.uniform(0.5, 2.0, f.shape)
    return obs, isig


@pytest.mark.parametrize("cfg", ["c2", "c2_ss1", "c3", "short", "ecc"])
def test_chi2_exact_parity(pt, oracle, cfg):
    if cfg == "c2":
        w = inputs.config2(n_pv=24, n_t=9000)
    elif cfg == "c2_ss1":
        w = inputs.config2(n_pv=24, n_t=9001); w.n_ss = 1
    elif cfg == "c3":
        w = inputs.config3(n_pv=64, n_pb=5, n_t=601)
    elif cfg == "short":
        w = inputs.config3(n_pv=1500, n_pb=2, n_t=40); w.n_ss, w.t_exp = 3, 0.003
    else:
        wd = inputs.dense_transit(n_pv=1, n_t=2000)
        rng = np.random.default_rng(9)
        p = np.repeat(wd.params, 200, 0)
        p[:, 6] *= rng.uniform(0.9, 1.1, 200); p[:, 0] += rng.normal(0, 2e-3, 200); p[:, 4] = rng.uniform(0.0, 0.5, 200)
        w = inputs.Workload("ecc", wd.times[0].copy(), p)
    obs, isig = _data_for(oracle, w)
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    c = pt.pt_ma_quad_chi2(dev(w.times), dev(w.params), dev(obs), dev(isig), w.n_pb, w.n_ss, w.t_exp, status=st)
    r = oracle.ma_quad_chi2(w.times, w.params, obs, isig, w.n_pb, w.n_ss, w.t_exp)
    assert st.cpu().tolist() == [0, 0]
    # flux parity is 1e-12 abs; a residual of r sigma turns that into 2 r 1e-12/sigma per term: relative 1e-10 is ample
    assert np.abs(c.cpu().numpy() - r).max() <= 1e-10 * np.abs(r).max(), (np.abs(c.cpu().numpy() - r).max(), np.abs(r).max())
    # and it is the same number as the library's own flux pushed through the definition
    f = gpu_exact(pt, w)
    assert np.allclose(c.cpu().numpy(), oracle.chi2_of_flux(f, obs, isig), rtol=1e-11)


def test_chi2_interp_and_bad_rows(pt, oracle):
    c4 = dict(k_min=0.05, k_max=0.25, n_k=41, z_max=1.25, n_z=1251)
    tb = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, **c4)
    w = inputs.config4(n_pv=40, n_t=6000)
    w.params[3, 6] = 0.31          # off the table: exact fallback
    w.params[7, 1] = -2.0          # bad period: NaN
    obs, isig = _data_for(oracle, w)
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    c = pt.pt_ma_quad_chi2(dev(w.times), dev(w.params), dev(obs), dev(isig), table=tb, status=st).cpu().numpy()
    r = oracle.ma_quad_chi2(w.times, w.params, obs, isig, table=(tb.data.cpu().numpy(), tb.k_min, tb.dk, tb.dz))
    assert np.isnan(c[7]) and np.isnan(r[7])
    ok = np.arange(40) != 7
    assert np.abs(c[ok] - r[ok]).max() <= 1e-10 * np.abs(r[ok]).max()
    assert st.cpu().tolist() == [pt.PT_ST_BAD_PARAM | pt.PT_ST_K_OUT_OF_TABLE, 2]


# ------------------------------------------------------------------------------------------- range mode (ascending shared axis)
def _axis_population(n_pv, seed):
    rng = np.random.default_rng(seed)
    P = rng.uniform(0.8, 9.0, n_pv)
    a = rng.uniform(4, 15, n_pv)
    b = rng.uniform(0, 1.1, n_pv)
    e = np.where(np.arange(n_pv) % 3 == 0, rng.uniform(0.05, 0.6, n_pv), 0.0)
    wv = rng.uniform(0, 2 * np.pi, n_pv)
    inc = np.arccos(np.clip(b * (1 + e * np.sin(wv)) / (a * (1 - e * e)), -1, 1))
    q1, q2 = rng.uniform(0, 1, n_pv), rng.uniform(0, 1, n_pv)
    u1, u2 = inputs.kipping_to_quadratic(q1, q2)
    return np.stack([P * rng.uniform(0, 1, n_pv), P, a, inc, e, wv, rng.uniform(0.02, 0.3, n_pv), u1, u2], 1)


@pytest.mark.parametrize("axis", ["uniform", "irregular", "duplicates", "shuffled", "nan_inside", "inf_at_end", "odd_length",
                                  "many_epochs", "bjd"])
@pytest.mark.parametrize("n_ss", [1, 4])
def test_range_mode_axis_variants(pt, oracle, axis, n_ss):
    """One shared time axis, large enough for the axis check: ascending axes take range mode (in-window index ranges by
    search, the rest pure fills), anything else must fall back to the per-exposure window test — same flux either way."""
    rng = np.random.default_rng(77)
    n_pv, n_t = 12, 30000
    params = _axis_population(n_pv, 78)
    t = 3.0 + np.arange(n_t) * 0.0204
    if axis == "irregular":
        t = np.sort(np.concatenate([rng.uniform(0, 90, 12000), rng.uniform(200, 201, 9000), rng.uniform(350, 900, 9000)]))
    elif axis == "duplicates":
        t = np.sort(np.repeat(3.0 + np.arange(n_t // 4) * 0.08, 4))
    elif axis == "shuffled":
        t = rng.permutation(t)
    elif axis == "nan_inside":
        t[12345] = np.nan
    elif axis == "inf_at_end":
        t[-1] = np.inf
    elif axis == "odd_length":
        t = t[:-1]
    elif axis == "many_epochs":
        params[:, 1] = rng.uniform(0.011, 0.03, n_pv)      # periods near the cadence: an epoch per exposure or two
        params[:, 0] = params[:, 1] * rng.uniform(0, 1, n_pv)
        params[:, 2] = rng.uniform(1.5, 3.0, n_pv)
    elif axis == "bjd":
        t = t + 2455000.0
        params[:, 0] += 2455000.0
    w = inputs.Workload(axis, np.ascontiguousarray(t), params, 1, n_ss, 0.0204)
    f, r = gpu_exact(pt, w), ora_exact(oracle, w)
    assert np.abs(f - r).max() <= TOL64
    assert np.array_equal(f == 1.0, r == 1.0)
    if n_ss == 1:
        # the interpolated path and the fused likelihood ride on the same streaming code
        tb = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, k_min=0.01, k_max=0.31, n_k=61, z_max=1.31, n_z=1311)
        fi = pt.pt_ma_quad_interp(tb, dev(w.times), dev(w.params)).cpu().numpy()
        ri = oracle.ma_quad_interp(tb.data.cpu().numpy(), tb.k_min, tb.dk, tb.dz, w.times, w.params, prec="f128")
        assert np.abs(fi - ri).max() <= TOL64
    if axis in ("uniform", "shuffled", "irregular"):
        obs, isig = _data_for(oracle, w)
        c = pt.pt_ma_quad_chi2(dev(w.times), dev(w.params), dev(obs), dev(isig), 1, n_ss, w.t_exp).cpu().numpy()
        rc = oracle.chi2_of_flux(r, obs, isig)
        assert np.abs(c - rc).max() <= 1e-10 * np.abs(rc).max()


@pytest.mark.parametrize("n_pv,n_t,n_ss", [(64, 4097, 10), (17, 2500, 1), (40, 6001, 3), (40, 6000, 40), (300, 2048, 1)])
def test_epoch_kernel_writes_every_element(pt, oracle, n_pv, n_t, n_ss):
    """The epoch kernel (one passband, shared ascending axis) partitions every row into gaps (pure fills) and transit
    windows (evaluated) found by search: an output buffer pre-filled with NaN must come back without one, for the exact
    and the interpolated model, fp64 and fp32 flux, even and odd row lengths, rows that never transit, rows cut into
    chunks (short periods, planet always overlapping) and bad rows."""
    w = inputs.config2(n_pv=n_pv, n_t=n_t)
    w.n_ss = n_ss
    p = w.params
    p[0, 1] = 0.05; p[1, 1] = 0.11; p[2, 2] = 1.05; p[3, 3] = 0.3; p[5, 6] = 0.0; p[6, 1] = 5000.0; p[7, 0] = 1e6
    p[4, 1] = -1.0                                           # bad row: NaN on both sides
    t, dp = dev(w.times), dev(p)
    r = ora_exact(oracle, w)
    for dtype, tol in ((torch.float64, TOL64), (torch.float32, TOL32)):
        out = torch.full((n_pv, 1, n_t), float("nan"), dtype=dtype, device="cuda")
        pt.pt_ma_quad_exact(t, dp, 1, w.n_ss, w.t_exp, out=out)
        f = out.cpu().numpy().astype(np.float64)
        assert np.array_equal(np.isnan(f), np.isnan(r)) and np.all(np.isnan(f[4]))
        ok = ~np.isnan(r)
        assert np.abs(f[ok] - r[ok]).max() <= tol
    tb = pt.pt_ma_table_build(dtype=torch.float32, n_fn=4, k_min=0.05, k_max=0.25, n_k=41, z_max=1.25, n_z=1251)
    out = torch.full((n_pv, 1, n_t), float("nan"), dtype=torch.float64, device="cuda")
    pt.pt_ma_quad_interp(tb, t, dp, 1, w.n_ss, w.t_exp, out=out)
    ri = oracle.ma_quad_interp(tb.data.cpu().numpy(), tb.k_min, tb.dk, tb.dz, w.times, p, 1, w.n_ss, w.t_exp, prec="f128")
    f = out.cpu().numpy()
    assert np.array_equal(np.isnan(f), np.isnan(ri))
    ok = ~np.isnan(ri)
    assert np.abs(f[ok] - ri[ok]).max() <= TOL64


def test_range_mode_multipassband_and_fp32(pt, oracle):
    rng = np.random.default_rng(5)
    n_pv, n_pb, n_t = 40, 3, 6000
    base = _axis_population(n_pv, 6)
    tail = np.concatenate([np.stack([base[:, 6] * rng.uniform(0.95, 1.05, n_pv), base[:, 7], base[:, 8]], 1) for _ in range(n_pb)], 1)
    params = np.concatenate([base[:, :6], tail], 1)
    t = 1.0 + np.arange(n_t) * 0.01
    w = inputs.Workload("mp", t, params, n_pb, 2, 0.01)
    r = ora_exact(oracle, w)
    assert np.abs(gpu_exact(pt, w) - r).max() <= TOL64
    assert np.abs(gpu_exact(pt, w, dtype=torch.float32) - r).max() <= TOL32


# ------------------------------------------------------------------------------------------- launch chain and slots
def test_inputs_written_by_device_kernels_right_before_the_call(pt, oracle):
    """the first kernel of a call must be ordered behind whatever the caller enqueued before it on the stream —
    here the parameters and the zeroed status word are produced by device kernels immediately in front of the call."""
    w = inputs.config2(n_pv=48, n_t=20000)
    obs, isig = _data_for(oracle, w)
    src = dev(w.params)
    garbage = torch.full_like(src, float("nan"))
    t, o, s = dev(w.times), dev(obs), dev(isig)
    r = oracle.ma_quad_chi2(w.times, w.params, obs, isig, 1, w.n_ss, w.t_exp)
    rf = ora_exact(oracle, w)
    for _ in range(5):
        p = garbage.clone()
        st = torch.full((2,), 7, dtype=torch.int32, device="cuda")
        big = torch.randn(1 << 24, device="cuda").cumsum(0)        # a long kernel in front, so that an early start would show
        p.copy_(src * 1.0)                                         # parameters written by device kernels ...
        st.zero_()                                                 # ... and the status word zeroed by one
        c = pt.pt_ma_quad_chi2(t, p, o, s, 1, w.n_ss, w.t_exp, status=st)
        p2 = garbage.clone()
        p2.copy_(src + 0.0)
        f = pt.pt_ma_quad_exact(t, p2, 1, w.n_ss, w.t_exp, status=st)
        torch.cuda.synchronize()
        assert st.cpu().tolist() == [0, 0]
        assert np.abs(c.cpu().numpy() - r).max() <= 1e-10 * np.abs(r).max()
        assert np.abs(f.cpu().numpy() - rf).max() <= TOL64
        del big


def test_more_launches_in_flight_than_scheduler_slots(pt, oracle):
    """24 streams x 3 launches each, all enqueued before any has finished: the library must never hand a live scheduler
    slot to a second launch (it makes the late launches wait on the device instead)."""
    w = inputs.config2(n_pv=16, n_t=16000)
    t, p = dev(w.times), dev(w.params)
    r = ora_exact(oracle, w)
    streams = [torch.cuda.Stream() for _ in range(24)]
    torch.cuda.synchronize()
    outs = []
    for rep in range(3):
        for s in streams:
            with torch.cuda.stream(s):
                outs.append(pt.pt_ma_quad_exact(t, p, 1, w.n_ss, w.t_exp))
    torch.cuda.synchronize()
    for f in outs:
        assert np.abs(f.cpu().numpy() - r).max() <= TOL64


def test_cuda_graph_capture_and_replay(pt, oracle):
    """An MCMC loop captures the model call once and replays it with new parameters in the same buffers."""
    w = inputs.config2(n_pv=32, n_t=12000)
    t, p = dev(w.times), dev(w.params)
    out = torch.empty((w.n_pv, 1, w.n_t), dtype=torch.float64, device="cuda")
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    pt.pt_ma_quad_exact(t, p, 1, w.n_ss, w.t_exp, out=out, status=st)      # warm-up outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        pt.pt_ma_quad_exact(t, p, 1, w.n_ss, w.t_exp, out=out, status=st)
    for seed in (1, 2, 3):
        w2 = inputs.config2(n_pv=32, n_t=12000, stream=seed)
        p.copy_(dev(w2.params))
        out.fill_(-1.0)
        g.replay()
        g.replay()                                                         # back-to-back replays of one graph
        torch.cuda.synchronize()
        ref = oracle.ma_quad_exact(w.times, w2.params, 1, w.n_ss, w.t_exp, prec="f128")
        assert np.abs(out.cpu().numpy() - ref).max() <= TOL64
    # ordinary launches keep working next to the graph's bound slot
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64


# ------------------------------------------------------------------------------------------- exact per-passband k (NEXT-2)
@pytest.mark.parametrize("n_pv,n_pb,n_t,n_ss", [(64, 20, 600, 1), (9, 3, 2501, 4), (200, 2, 33, 1), (5, 40, 700, 1)])
def test_per_passband_k_mode(pt, oracle, n_pv, n_pb, n_t, n_ss):
    w = inputs.config3(n_pv=n_pv, n_pb=n_pb, n_t=n_t)
    w.params[:, 6::3] *= np.linspace(0.7, 1.4, n_pb)[None, :]       # a wide spread of radius ratios
    w.n_ss, w.t_exp = n_ss, 0.003
    f = pt.pt_ma_quad_exact_pbk(dev(w.times), dev(w.params), n_pb, n_ss, w.t_exp).cpu().numpy()
    r = oracle.ma_quad_exact_pbk(w.times, w.params, n_pb, n_ss, w.t_exp)
    assert np.abs(f - r).max() <= TOL64
    f32 = pt.pt_ma_quad_exact_pbk(dev(w.times), dev(w.params), n_pb, n_ss, w.t_exp, dtype=torch.float32).cpu().numpy()
    assert np.abs(f32 - r).max() <= TOL32


# ------------------------------------------------------------------------------------------- window-test robustness
def test_large_epochs_unsorted_times_and_padded_rows(pt, oracle):
    """The cheap window test folds with t*(1/P) + c0; its error bound must hold for BJD-sized epochs (|t0/P| ~ 2e6),
    negative times, unsorted and repeated times, NaN/inf times (flux 1), and rows padded beyond n_t."""
    rng = np.random.default_rng(21)
    n_pv, n_t = 12, 5000
    P = rng.uniform(0.7, 9.0, n_pv)
    a = rng.uniform(4, 15, n_pv)
    b = rng.uniform(0, 0.9, n_pv)
    e = np.where(np.arange(n_pv) % 2 == 0, 0.0, rng.uniform(0.05, 0.5, n_pv))
    wv = rng.uniform(0, 2 * np.pi, n_pv)
    inc = np.arccos(np.clip(b * (1 + e * np.sin(wv)) / (a * (1 - e * e)), -1, 1))
    t0 = 2455000.0 + P * rng.uniform(0, 1, n_pv)
    params = np.stack([t0, P, a, inc, e, wv, rng.uniform(0.03, 0.25, n_pv), 0.4 + 0 * P, 0.25 + 0 * P], 1)
    times = 2455000.0 + rng.uniform(-400.0, 400.0, n_t)          # unsorted, ~800 d around the epochs
    times[::97] = times[1::97][: len(times[::97])]                # repeated values
    times[5], times[6], times[7] = np.nan, np.inf, -np.inf
    for n_ss, t_exp in ((1, 0.0), (6, 0.02)):
        w = inputs.Workload("bjd", times, params, 1, n_ss, t_exp)
        f, r = gpu_exact(pt, w), ora_exact(oracle, w)
        assert np.abs(f - r).max() <= TOL64
        assert np.array_equal(f == 1.0, r == 1.0)
    # the same through negative epochs and per-pv time rows with a padded stride
    tt = np.full((n_pv, n_t + 37), 123.0)
    for i in range(n_pv):
        tt[i, :n_t] = -3.0e5 + np.sort(rng.uniform(-50, 50, n_t))
    params[:, 0] = -3.0e5 + P * rng.uniform(0, 1, n_pv)
    dt, dp = dev(tt), dev(params)
    out = torch.empty((n_pv, 1, n_t), dtype=torch.float64, device="cuda")
    from paper_1504_07433_b200 import binding
    rc = binding.lib().pt_ma_quad_exact(dt.data_ptr(), n_t, n_t + 37, dp.data_ptr(), n_pv, 1, 3, 0.01, 0, out.data_ptr(), None,
                                        torch.cuda.current_stream().cuda_stream)
    assert rc == 0
    torch.cuda.synchronize()
    ref = oracle.ma_quad_exact(np.ascontiguousarray(tt[:, :n_t]), params, 1, 3, 0.01, prec="f128")
    assert np.abs(out.cpu().numpy() - ref).max() <= TOL64


def test_max_passbands_and_many_subsamples(pt, oracle):
    """n_pb at the library's limit (1024: combine coefficients beyond the per-warp cache come from the row) and a
    four-digit supersample count."""
    w = inputs.config3(n_pv=3, n_pb=1024, n_t=64)
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64
    w = inputs.config2(n_pv=2, n_t=300)
    w.n_ss, w.t_exp = 1500, 0.05
    assert np.abs(gpu_exact(pt, w) - ora_exact(oracle, w)).max() <= TOL64


# ------------------------------------------------------------------------------------------- NEXT-4: the Giménez model
def _gimenez_population(n_pv, n_pb, n_ldc, seed):
    rng = np.random.default_rng(seed)
    P, a = rng.uniform(1, 10, n_pv), rng.uniform(4, 20, n_pv)
    e = np.where(rng.uniform(size=n_pv) < 0.5, 0.0, rng.uniform(0, 0.5, n_pv))
    wv = rng.uniform(0, 2 * math.pi, n_pv)
    inc = np.arccos(np.clip(rng.uniform(0, 0.9, n_pv) * (1 + e * np.sin(wv)) / (a * (1 - e * e)), -1, 1))
    k = rng.uniform(0.02, 0.3, n_pv)
    u = rng.uniform(-0.1, 0.5, (n_pv, n_pb * n_ldc)) / n_ldc
    return np.concatenate([np.stack([P * rng.uniform(0, 1, n_pv), P, a, inc, e, wv, k], 1), u], 1)


@pytest.mark.parametrize("n_pb,n_ldc,n_j,n_ss", [(1, 2, 40, 1), (3, 2, 25, 1), (2, 4, 30, 3), (1, 1, 60, 1), (2, 8, 10, 1)])
def test_gimenez_exact_parity(pt, oracle, n_pb, n_ldc, n_j, n_ss):
    """The series of Eq. 3 with the same N_J on both sides: the kernel runs the polynomials up by the three-term recurrence in
    fp64 from a precomputed table, the oracle sums each polynomial explicitly in __float128.  Tolerance 1e-11 absolute: the
    recurrences are stable inside [-1, 1] (error growth ~ j ulp), N_J <= 60 terms of size <= 1e-2 each."""
    n_pv, n_t = 12, 120
    params = _gimenez_population(n_pv, n_pb, n_ldc, 50 + n_ldc)
    rng = np.random.default_rng(7)
    t14 = params[:, 1] / (math.pi * params[:, 2])
    t = params[:, 0][:, None] + params[:, 1][:, None] * rng.integers(0, 5, (n_pv, 1)) + rng.uniform(-1.5, 1.5, (n_pv, n_t)) * t14[:, None]
    params[5, 1] = -1.0
    coef = pt.GimenezCoef(n_ldc, n_j)
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    f = pt.pt_gimenez_exact(coef, dev(t), dev(params), n_pb, n_ss, 0.01, status=st).cpu().numpy()
    r = oracle.gimenez_exact(t, params, n_pb, n_ldc, n_j, n_ss, 0.01, prec="f128")
    assert np.array_equal(np.isnan(f), np.isnan(r)) and np.all(np.isnan(f[5])) and st.cpu().tolist() == [pt.PT_ST_BAD_PARAM, 1]
    ok = ~np.isnan(r)
    assert np.abs(f[ok] - r[ok]).max() <= 1e-11
    assert np.array_equal(f[ok] == 1.0, r[ok] == 1.0) and (r[ok] < 1.0).mean() > 0.3


def test_gimenez_quadratic_law_against_mandel_agol(pt, oracle):
    # N = 2, u_1 = a + 2b, u_2 = -b: the Giménez kernel against the Mandel-Agol kernel and oracle (truncation error, falling with N_J)
    w = inputs.config2(n_pv=6, n_t=4000)
    pm = w.params
    pg = np.concatenate([pm[:, :7], (pm[:, 7] + 2 * pm[:, 8])[:, None], -pm[:, 8][:, None]], axis=1)
    fm = gpu_exact(pt, inputs.Workload("m", w.times, pm))[:, 0]
    errs = []
    for n_j in (10, 40, 160):
        fg = pt.pt_gimenez_exact(pt.GimenezCoef(2, n_j), dev(w.times), dev(pg)).cpu().numpy()[:, 0]
        errs.append(np.abs(fg - fm).max())
        assert np.array_equal(fg == 1.0, fm == 1.0)
    assert errs[0] > 3 * errs[1] > 9 * errs[2] and errs[1] <= 5e-5 and errs[2] <= 6e-6, errs


def test_gimenez_interp_parity(pt, oracle):
    """the tables the call leaves in d_work against the oracle's α_n at the nodes, and the flux against the
    oracle's interpolation of THE SAME tables (1e-12); the error against the series is reported, not gated."""
    n_pv, n_pb, n_ldc, n_j, n_in, n_out, n_t = 6, 2, 2, 30, 40, 60, 400
    params = _gimenez_population(n_pv, n_pb, n_ldc, 91)
    rng = np.random.default_rng(8)
    t14 = params[:, 1] / (math.pi * params[:, 2])
    t = params[:, 0][:, None] + rng.uniform(-1.2, 1.2, (n_pv, n_t)) * t14[:, None]
    coef = pt.GimenezCoef(n_ldc, n_j)
    for n_ss in (1, 3):
        f, work = pt.pt_gimenez_interp(coef, n_in, n_out, dev(t), dev(params), n_pb, n_ss, 0.004)
        f, tab = f.cpu().numpy(), work.cpu().numpy()
        r = oracle.gimenez_interp_flux(tab, n_in, t, params, n_pb, n_ldc, n_ss, 0.004)
        assert np.abs(f - r).max() <= 1e-12
    for pv in (0, 3):
        k = params[pv, 6]
        zn = np.concatenate([np.linspace(0, 1 - k, n_in), np.linspace(1 - k, 1 + k, n_out)])
        for n in range(n_ldc + 1):
            ref = oracle.gimenez_alpha(n, n_j, k, zn, "f128")
            ref[-1] = 0.0
            assert np.abs(tab[pv, n] - ref).max() <= 1e-12
    fx = pt.pt_gimenez_exact(coef, dev(t), dev(params), n_pb, 3, 0.004).cpu().numpy()
    print("gimenez interp vs series: max %.2e mean %.2e" % (np.abs(f - fx).max(), np.abs(f - fx).mean()))
    assert np.abs(f - fx).max() <= 1e-3


def test_gimenez_argument_errors(pt):
    from paper_1504_07433_b200 import binding
    L = binding.lib()
    import ctypes as C
    nb = C.c_int64(0)
    assert L.pt_gimenez_coef_size(2, 40, C.byref(nb)) == 0 and nb.value == 3 * 41 * 8 * 8
    assert L.pt_gimenez_coef_size(9, 40, C.byref(nb)) == binding.PT_ERR_SIZE
    assert L.pt_gimenez_coef_size(2, 257, C.byref(nb)) == binding.PT_ERR_SIZE
    coef = pt.GimenezCoef(2, 10)
    t = torch.zeros(8, dtype=torch.float64, device="cuda")
    p = torch.zeros((1, 9), dtype=torch.float64, device="cuda")
    o = torch.zeros(8, dtype=torch.float64, device="cuda")
    assert L.pt_gimenez_exact(None, 2, 10, t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 1, 0.0, o.data_ptr(), None, None) == binding.PT_ERR_NULL
    assert L.pt_gimenez_exact(coef.data.data_ptr(), 2, 10, t.data_ptr(), 8, 0, p.data_ptr(), 1, 65, 1, 0.0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
    assert L.pt_gimenez_interp(coef.data.data_ptr(), 2, 10, 1, 5, o.data_ptr(), t.data_ptr(), 8, 0, p.data_ptr(), 1, 1, 1, 0.0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
