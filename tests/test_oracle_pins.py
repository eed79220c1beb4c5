"""Pins for the CPU oracle: every function of oracle/pt_oracle.cpp is checked against something other than itself
(SURVEY §8(c)-5 P1-P12): the integral definitions by quadrature, mpmath's elliptic integrals, closed forms,
symmetries, brute force, the paper's printed interpolation error.  CPU only."""
import math

import numpy as np
import pytest

from oracle import ma_definition as mdef
from paper_1504_07433_b200 import inputs

DEG = math.pi / 180.0


def quad_flux(le, ld, ed, u1, u2):
    """Eq. 13 retyped independently of the oracle."""
    c = u1 + 2 * u2
    return 1.0 - ((1 - c) * le + c * ld + u2 * ed) / (1 - u1 / 3 - u2 / 6)


# ------------------------------------------------------------------ elliptic integrals (Carlson) vs mpmath
def test_carlson_elliptic_vs_mpmath(oracle):
    import mpmath as mp
    mp.mp.dps = 30
    rng = np.random.default_rng(1)
    m = np.concatenate([rng.uniform(0, 1, 40), 1 - 10.0 ** rng.uniform(-12, -1, 20), [0.0, 0.5, 1e-12]])
    n = -np.concatenate([10.0 ** rng.uniform(-3, 12, 40), rng.uniform(0, 1, 20), [0.0, 1.0, 1e6]])
    for prec, tol in (("f128", 4e-16), ("f64", 2e-13)):
        K, E, Pi = oracle.ellip(m, n, prec)
        for i in range(len(m)):
            k_ref, e_ref, p_ref = mp.ellipk(m[i]), mp.ellipe(m[i]), mp.ellippi(n[i], m[i])
            assert abs(K[i] - k_ref) <= tol * max(1, abs(k_ref)), (prec, m[i])
            assert abs(E[i] - e_ref) <= tol * max(1, abs(e_ref)), (prec, m[i])
            assert abs(Pi[i] - p_ref) <= tol * max(1, abs(p_ref)), (prec, n[i], m[i])


# ------------------------------------------------------------------ basis functions vs their definitions
def test_basis_vs_integral_definition_golden(oracle, golden_basis):
    """P5/P12: closed forms == 30-digit quadrature of the Eq. 6 + Eq. 13 integrals, all regions and boundaries."""
    k, z = golden_basis[:, 0], golden_basis[:, 1]
    got = np.stack(oracle.ma_basis(k, z, "f128"), axis=1)
    err = np.abs(got - golden_basis[:, 2:5])
    assert err.max() <= 1e-15, (err.max(), golden_basis[np.argmax(err.max(axis=1))])


def test_basis_double_instantiation_away_from_boundaries(oracle, golden_basis):
    """The double instantiation (timed CPU baseline) is the same text; textbook forms lose digits only near boundaries."""
    k, z = golden_basis[:, 0], golden_basis[:, 1]
    dist = np.min(np.abs(np.stack([z - k, z - (1 - k), z - (1 + k), k - 0.5 + 0 * z])), axis=0)
    far = (dist > 1e-3) | (dist == 0)
    got = np.stack(oracle.ma_basis(k, z, "f64"), axis=1)
    assert np.abs(got - golden_basis[:, 2:5])[far].max() <= 2e-13
    assert np.abs(got - golden_basis[:, 2:5]).max() <= 1e-6   # documented loss of the textbook forms in double


def test_basis_vs_2d_gauss_legendre_random(oracle):
    """north_star pin: 2-D quadrature of the intensity profile over the occulted area (gate 1e-7; reaches ~1e-13)."""
    rng = np.random.default_rng(7)
    k = np.concatenate([rng.uniform(0.01, 0.7, 40), rng.uniform(1.0, 2.0, 5)])
    z = rng.uniform(0, 1, 45) * (1 + k)
    got = np.stack(oracle.ma_basis(k, z, "f128"), axis=1)
    ref = np.array([mdef.basis_gl2d(float(a), float(b), n_r=300) for a, b in zip(k, z)])
    assert np.abs(got - ref).max() <= 1e-11


def test_basis_and_flux_vs_pixel_brute_force(oracle):
    """Brute force on tiny inputs: pixel sums of Eq. 6 *as printed* over the occulted area (catches wrong weights)."""
    pts = [(0.1, 0.3), (0.1, 0.95), (0.3, 0.2), (0.3, 0.85), (0.6, 0.5), (0.2, 1.1), (1.3, 0.9)]
    for k, z in pts:
        le, ld, ed = (float(v[0]) for v in oracle.ma_basis([k], [z], "f128"))
        ple, pld, ped = mdef.basis_pixels(k, z, 3000)
        assert abs(le - ple) < 2e-5 and abs(ld - pld) < 2e-5 and abs(ed - ped) < 2e-5, (k, z)
        for u1, u2 in ((0.4, 0.2), (0.7, -0.1), (0.0, 0.0)):
            params = np.array([[0.0, 1.0, z, math.pi / 2, 0.0, 0.0, k, u1, u2]])  # a = z, i = 90°, t = t0  =>  z(t0) = a cos i ~ 0
            # drive z through the orbit instead: b = z via cos i = z/a
            a = 10.0
            params = np.array([[0.0, 1.0, a, math.acos(z / a), 0.0, 0.0, k, u1, u2]])
            f = oracle.ma_quad_exact(np.array([0.0]), params, prec="f128")[0, 0, 0]
            assert abs(f - mdef.flux_pixels(k, z, u1, u2, 3000)) < 6e-5, (k, z, u1, u2)
            assert abs(f - quad_flux(le, ld, ed, u1, u2)) < 1e-13


def test_p1_no_overlap_is_exactly_one(oracle):
    k = np.array([0.1, 0.1, 0.5, 1.5, 0.0, 0.0])
    z = np.array([1.1, 5.0, 1.5, 2.5, 0.3, 0.0])
    for prec in ("f64", "f128"):
        le, ld, ed = oracle.ma_basis(k, z, prec)
        assert np.all(le == 0) and np.all(ld == 0) and np.all(ed == 0)
    w = inputs.config1()
    f = oracle.ma_quad_exact(w.times, w.params, prec="f128")[0, 0]
    z = np.abs(oracle.orbit_z(w.times, w.params, prec="f128")[0, :, 0])
    assert np.all(f[z >= 1.1] == 1.0) and np.all(f[z < 1.1 - 1e-9] < 1.0)


def lens_area(r, R, d):
    """Textbook area of intersection of two circles of radii r, R at centre distance d (partial overlap)."""
    return (r * r * math.acos((d * d + r * r - R * R) / (2 * d * r)) + R * R * math.acos((d * d + R * R - r * r) / (2 * d * R))
            - 0.5 * math.sqrt((-d + r + R) * (d + r - R) * (d - r + R) * (d + r + R)))


def test_p2_uniform_disk_is_lens_area(oracle):
    rng = np.random.default_rng(3)
    k = rng.uniform(0.02, 1.5, 200)
    z = np.abs(1 - k) + rng.uniform(0.001, 0.999, 200) * (1 + k - np.abs(1 - k))
    le, _, _ = oracle.ma_basis(k, z, "f128")
    ref = np.array([lens_area(a, 1.0, b) / math.pi for a, b in zip(k, z)])
    assert np.abs(le - ref).max() <= 1e-14
    # through the flux: u1 = u2 = 0  =>  F = 1 - λe  (uniform model)
    a = 10.0
    params = np.stack([0 * k, 1 + 0 * k, a + 0 * k, np.arccos(z / a), 0 * k, 0 * k, k, 0 * k, 0 * k], axis=1)
    f = oracle.ma_quad_exact(np.array([0.0]), params, prec="f128")[:, 0, 0]
    assert np.abs(f - np.clip(1 - ref, 0, None)).max() <= 1e-14


def test_p3_planet_fully_inside(oracle):
    rng = np.random.default_rng(4)
    k = rng.uniform(0.01, 0.9, 200)
    z = rng.uniform(0, 1, 200) * (1 - k)
    le, ld, ed = oracle.ma_basis(k, z, "f128")
    assert np.abs(le - k * k).max() <= 1e-16
    assert np.abs(ed - k * k * (k * k + 2 * z * z) / 2).max() <= 1e-16
    # z = 0: λd = (2/3)(1 - (1-k²)^(3/2))
    le0, ld0, ed0 = oracle.ma_basis(k, 0 * k, "f128")
    assert np.abs(ld0 - 2 / 3 * (1 - (1 - k * k) ** 1.5)).max() <= 2e-16
    # SURVEY §8(c)-5 P3 worked value, k = 0.1, u = (0.4, 0.2), z = 0
    f = quad_flux(*[float(v[0]) for v in oracle.ma_basis([0.1], [0.0], "f128")], 0.4, 0.2)
    assert abs(f - 0.9880120401507544) <= 1e-15
    # the generic inside formula tends to the z = 0 closed form
    le1, ld1, ed1 = oracle.ma_basis(k, 1e-9 + 0 * k, "f128")
    assert np.abs(ld1 - ld0).max() <= 1e-12


def test_p8_special_values(oracle):
    le, ld, ed = oracle.ma_basis([0.75, 0.5, 1.5, 3.0, 1.0], [0.25, 0.5, 0.5, 1.0, 0.0], "f128")
    assert abs(ld[0] - 4 / 9) <= 1e-16 and abs(le[0] - 0.5625) <= 1e-16
    assert abs(ld[1] - (1 / 3 - 4 / (9 * math.pi))) <= 1e-16 and abs(ed[1] - 3 / 32) <= 1e-16 and abs(le[1] - 0.25) <= 1e-16
    for i in (2, 3, 4):  # star covered: flux 0 for any limb darkening
        assert (le[i], ld[i], ed[i]) == (1.0, 2 / 3, 0.5)
        assert abs(quad_flux(le[i], ld[i], ed[i], 0.4, 0.2)) <= 3e-16


def test_p7_continuity_across_case_boundaries(oracle):
    """Each exact-equality formula equals the limit of the generic one."""
    for k in (0.05, 0.1, 0.3, 0.45, 0.5, 0.6, 0.9):
        for z0 in (k, 1 - k, 1 + k, 0.0):
            if z0 < 0:
                continue
            for d in (1e-9, -1e-9):
                z1 = z0 + d
                if z1 < 0:
                    continue
                a = np.array(oracle.ma_basis([k], [z0], "f128")).ravel()
                b = np.array(oracle.ma_basis([k], [z1], "f128")).ravel()
                assert np.abs(a - b).max() <= 1e-7, (k, z0, d, a, b)
    # k -> 1/2 at z = k
    a = np.array(oracle.ma_basis([0.5], [0.5], "f128")).ravel()
    for d in (1e-9, -1e-9):
        b = np.array(oracle.ma_basis([0.5 + d], [0.5 + d], "f128")).ravel()
        assert np.abs(a - b).max() <= 1e-7


def test_p6_linearity_in_limb_darkening(oracle):
    w = inputs.config3(n_pv=4, n_pb=5, n_t=60)
    f = oracle.ma_quad_exact(w.times, w.params, n_pb=5, prec="f128")
    z = oracle.orbit_z(w.times, w.params, n_pb=5, prec="f128")[:, :, 0]
    for pv in range(4):
        ks = w.params[pv, 6::3]
        khat = ks.mean()
        le, ld, ed = oracle.ma_basis(np.full(60, khat), np.abs(z[pv]), "f128")
        for j in range(5):
            u1, u2 = w.params[pv, 7 + 3 * j], w.params[pv, 8 + 3 * j]
            ref = 1 - (ks[j] / khat) ** 2 * (1 - quad_flux(le, ld, ed, u1, u2))   # P:L179 correction on the decrement
            assert np.abs(f[pv, j] - ref).max() <= 1e-15


# ------------------------------------------------------------------ worked example, symmetry
def test_config1_worked_example(oracle, golden_config1):
    """P12: BASELINE.json configs[0] against flux values obtained from the definitions (tests/golden/make_golden.py)."""
    w = inputs.config1()
    t = golden_config1[:, 0]
    z = oracle.orbit_z(t, w.params, prec="f128")[0, :, 0]
    f = oracle.ma_quad_exact(t, w.params, prec="f128")[0, 0]
    assert np.abs(z - golden_config1[:, 1]).max() <= 2e-15
    assert np.abs(f - golden_config1[:, 2]).max() <= 1e-15
    fd = oracle.ma_quad_exact(t, w.params, prec="f64")[0, 0]
    assert np.abs(fd - golden_config1[:, 2]).max() <= 1e-13
    # SURVEY §8(c)-5 prints z(0) = 0.279195973620008 and F(0) = 0.98820877925565
    assert abs(z[0] - 0.279195973620008) < 1e-15 and abs(f[0] - 0.98820877925565) < 1e-14


def test_p4_symmetry_and_periodicity(oracle):
    w = inputs.config1()
    dt = np.arange(0, 600) * 2.0 ** -12   # representable offsets
    fp = oracle.ma_quad_exact(dt, w.params, prec="f128")[0, 0]
    fm = oracle.ma_quad_exact(-dt, w.params, prec="f128")[0, 0]
    assert np.array_equal(fp, fm)
    f2 = oracle.ma_quad_exact(dt + 3.0 * 7, w.params, prec="f128")[0, 0]
    assert np.abs(f2 - fp).max() <= 1e-13
    # eccentric: periodic, not symmetric
    pe = np.array([[0.3, 2.75, 9.0, 87 * DEG, 0.4, 1.0, 0.12, 0.3, 0.3]])
    t = 0.3 + np.linspace(-0.1, 0.1, 101)
    fa = oracle.ma_quad_exact(t, pe, prec="f128")[0, 0]
    fb = oracle.ma_quad_exact(t + 2.75 * 4, pe, prec="f128")[0, 0]
    assert np.abs(fa - fb).max() <= 1e-12 and np.abs(fa - fa[::-1]).max() > 1e-6


# ------------------------------------------------------------------ orbit
def test_p10_kepler_residual_and_limits(oracle):
    rng = np.random.default_rng(5)
    M = rng.uniform(-math.pi, math.pi, 2000)
    e = rng.uniform(0, 0.95, 2000)
    for prec in ("f64", "f128"):
        E = oracle.kepler(M, e, prec)
        assert np.abs(E - e * np.sin(E) - M).max() <= 1e-15 * 4
    assert np.array_equal(oracle.kepler(M, 0 * e, "f128"), M)


def test_orbit_identities(oracle):
    rng = np.random.default_rng(6)
    n = 300
    P, a = rng.uniform(1, 10, n), rng.uniform(3, 20, n)
    t0 = P * rng.uniform(0, 1, n)
    inc = np.arccos(rng.uniform(0, 0.9, n) / a)
    e, wv = rng.uniform(0.01, 0.8, n), rng.uniform(0, 2 * math.pi, n)
    pe = np.stack([t0, P, a, inc, e, wv, 0.1 + 0 * P, 0 * P, 0 * P], axis=1)
    # z(t0) = a cos i (1-e²)/(1+e sin w), planet in front
    z0 = oracle.orbit_z(t0[:, None], pe, prec="f128")[:, 0, 0]
    assert np.abs(z0 - a * np.cos(inc) * (1 - e * e) / (1 + e * np.sin(wv))).max() <= 2e-14
    # half a period later (in mean anomaly) the planet is behind the star for a circular orbit
    pc = pe.copy(); pc[:, 4] = 0
    zb = oracle.orbit_z((t0 + P / 2)[:, None], pc, prec="f128")[:, 0, 0]
    assert np.all(zb < 0)
    # e -> 0: the eccentric branch tends to the circular formula for any w
    ps = pe.copy(); ps[:, 4] = 1e-13
    t = t0[:, None] + P[:, None] * np.linspace(-0.5, 0.5, 41)[None, :]
    zc = oracle.orbit_z(t, pc, prec="f128")[:, :, 0]
    zs = oracle.orbit_z(t, ps, prec="f128")[:, :, 0]
    assert np.abs(np.abs(zc) - np.abs(zs)).max() <= 1e-10
    # circular formula retyped: z = a sqrt(sin² + cos²i cos²)
    ph = (t - t0[:, None]) / P[:, None]; ph = ph - np.rint(ph)
    ref = a[:, None] * np.sqrt(np.sin(2 * np.pi * ph) ** 2 + (np.cos(inc)[:, None] * np.cos(2 * np.pi * ph)) ** 2)
    assert np.abs(np.abs(zc) - ref).max() <= 1e-13
    # independent check of the eccentric geometry through the true anomaly: r sqrt(1 - sin²(w+f) sin² i)
    import mpmath as mp
    mp.mp.dps = 30
    for j in range(0, n, 29):
        for tt in t[j, ::7]:
            x = (tt - t0[j]) / P[j]; p1 = x - np.rint(x)
            Mtr_f = mp.pi / 2 - mp.mpf(wv[j])
            Etr = 2 * mp.atan(mp.sqrt((1 - mp.mpf(e[j])) / (1 + mp.mpf(e[j]))) * mp.tan(Mtr_f / 2))
            Mtr = Etr - mp.mpf(e[j]) * mp.sin(Etr)
            Mm = 2 * mp.pi * mp.mpf(float(p1)) + Mtr
            E = mp.findroot(lambda x_: x_ - mp.mpf(e[j]) * mp.sin(x_) - Mm, Mm)
            f = 2 * mp.atan(mp.sqrt((1 + mp.mpf(e[j])) / (1 - mp.mpf(e[j]))) * mp.tan(E / 2))
            r = mp.mpf(a[j]) * (1 - mp.mpf(e[j]) * mp.cos(E))
            zz = r * mp.sqrt(1 - (mp.sin(mp.mpf(wv[j]) + f) * mp.sin(mp.mpf(inc[j]))) ** 2)
            got = oracle.orbit_z(np.array([tt]), pe[j:j + 1], prec="f128")[0, 0, 0]
            assert abs(abs(got) - zz) <= 1e-13, (j, tt)
            assert (got > 0) == (mp.sin(mp.mpf(wv[j]) + f) > 0)


def _true_anomaly_exact(oracle, M, e):
    E = oracle.kepler(M, e, "f128")
    return 2.0 * np.arctan2(np.sqrt(1 + e) * np.sin(E / 2), np.sqrt(1 - e) * np.cos(E / 2))


def test_next3_fixed_point_iteration_reaches_the_kepler_root(oracle):
    # S§8(f) NEXT-3, "iteration": E <- M + e sin E.  Pinned against the bisection solve (a different method) and
    # against Kepler's equation itself.
    rng = np.random.default_rng(31)
    M = rng.uniform(-math.pi, math.pi, 500)
    e = rng.uniform(0, 0.9, 500)
    for prec, tol in (("f64", 4e-15), ("f128", 1e-15)):
        E = oracle.kepler_iter(M, e, prec)
        assert np.abs(E - e * np.sin(E) - M).max() <= 4 * tol / (1 - 0.9)       # residual / (1 - e cos E) = error in E
        assert np.abs(E - oracle.kepler(M, e, "f128")).max() <= 4e-14
    assert np.array_equal(oracle.kepler_iter(M, 0 * e, "f128"), M)               # e -> 0 limit: E = M


def test_next3_series_coefficients_are_the_fourier_coefficients_of_the_equation_of_the_centre(oracle):
    # The two series are truncations of f - M = sum_k c_k(e) sin kM.  The coefficients are pinned against the
    # mathematics, not against their own formula: c_k(e) = (2/π) ∫_0^π (f - M) sin kM dM of the EXACT true anomaly
    # (bisection Kepler solve), by the trapezoidal rule on a periodic integrand (spectrally accurate).  A wrong
    # coefficient (13/12 -> 13/16, a dropped e^5 term, a wrong sign) fails at the e^6 / e^4 level of the remainder.
    n = 4096
    M = (np.arange(n) + 0.5) * (2 * math.pi / n) - math.pi
    for e in (0.02, 0.05, 0.1):
        ev = np.full(n, e)
        d_exact = _true_anomaly_exact(oracle, M, ev) - M
        ck = [(2.0 / n) * np.sum(d_exact * np.sin(k * M)) for k in range(1, 7)]
        for order, rem in ((3, 3.0 * e ** 4), (5, 4.0 * e ** 6)):
            d_series = oracle.true_anomaly_series(M, ev, order, "f128") - M
            sk = [(2.0 / n) * np.sum(d_series * np.sin(k * M)) for k in range(1, 7)]
            # harmonics the truncation keeps agree up to the first neglected power of e; the ones it drops are absent
            for k in range(1, 7):
                assert abs(sk[k - 1] - ck[k - 1]) <= rem + 1e-14, (e, order, k, sk[k - 1], ck[k - 1])
                if k > order:
                    assert abs(sk[k - 1]) <= 1e-14


def test_next3_series_error_versus_eccentricity_curve(oracle):
    # error-vs-e curve of the two series against the exact true anomaly: order 3 falls like e^4, order 5 like e^6, and the
    # constants are those of the first neglected terms; this is what the e-based dispatch of DESIGN.md R19 rests on
    M = np.linspace(-math.pi, math.pi, 2001)
    es = np.array([0.003, 0.006, 0.012, 0.03, 0.06, 0.12])
    err = {3: [], 5: []}
    for e in es:
        ev = np.full(M.size, e)
        fx = _true_anomaly_exact(oracle, M, ev)
        for order in (3, 5):
            err[order].append(np.abs(oracle.true_anomaly_series(M, ev, order, "f128") - fx).max())
    e3, e5 = np.array(err[3]), np.array(err[5])
    s3 = np.polyfit(np.log(es), np.log(e3), 1)[0]
    s5 = np.polyfit(np.log(es[2:]), np.log(e5[2:]), 1)[0]          # below e ~ 0.01 the e^6 error sinks under double rounding
    assert 3.9 <= s3 <= 4.2 and 5.8 <= s5 <= 6.3, (s3, s5)
    assert np.all(e3 <= 1.5 * es ** 4 * 1.1) and np.all(e3 >= 1.0 * es ** 4)      # max_M |(-11/24) sin 2M + (103/96) sin 4M| = 1.40
    assert np.all(e5[2:] <= 2.2 * es[2:] ** 6 * 1.2)
    # the dispatch thresholds: below them the truncation error is under 2e-9 rad
    assert e3[es <= 0.006].max() <= 2e-9 and e5[es <= 0.03].max() <= 2e-9
    # e -> 0: every routine tends to the circular orbit
    rng = np.random.default_rng(32)
    p = np.array([[0.3, 2.5, 9.0, 1.5, 1e-12, 0.7, 0.1, 0.3, 0.2]])
    pc = p.copy(); pc[0, 4] = 0.0
    t = rng.uniform(0, 10, 200)
    zc = oracle.orbit_z(t, pc, prec="f128")
    for sv in ("iter", "ps3", "ps5", "fast", "newton"):
        assert np.abs(np.abs(oracle.orbit_z_solver(t, p, sv, prec="f128")) - np.abs(zc)).max() <= 1e-9


def test_next3_orbit_z_by_each_routine(oracle):
    # z through each routine against the exact orbit: the iteration to rounding, the series within a·|Δf|·(1+e)/(1-e)
    # (|∂(position)/∂f| <= r_max/a), and the dispatch picks the routine R19 states
    rng = np.random.default_rng(33)
    n = 40
    P, a = rng.uniform(1, 10, n), rng.uniform(3, 20, n)
    e = np.concatenate([[0.0, 0.004, 0.006, 0.02, 0.03, 0.031], rng.uniform(0, 0.5, n - 6)])
    pe = np.stack([P * rng.uniform(0, 1, n), P, a, np.arccos(rng.uniform(0, 0.9, n) / a), e, rng.uniform(0, 6.28, n),
                   0.1 + 0 * P, 0 * P, 0 * P], axis=1)
    t = np.sort(rng.uniform(0, 30, 400))
    zx = oracle.orbit_z(t, pe, prec="f128")
    assert np.abs(oracle.orbit_z_solver(t, pe, "iter", prec="f128") - zx).max() <= 1e-11
    assert np.array_equal(oracle.orbit_z_solver(t, pe, "newton", prec="f128"), zx)
    for sv, c, pw in (("ps3", 1.5, 4), ("ps5", 2.2, 6)):
        dz = np.abs(np.abs(oracle.orbit_z_solver(t, pe, sv, prec="f128")) - np.abs(zx)).max(axis=(1, 2))
        bound = a * (1 + e) / (1 - e) * c * 1.3 * e ** pw + 1e-12
        assert np.all(dz <= bound), (sv, (dz / bound).max())
    zf = oracle.orbit_z_solver(t, pe, "fast", prec="f128")
    for j in range(n):
        sv = "exact" if e[j] == 0 else ("ps3" if e[j] <= 0.006 else ("ps5" if e[j] <= 0.03 else "newton"))
        assert np.array_equal(zf[j], oracle.orbit_z_solver(t, pe[j:j + 1], sv, prec="f128")[0]), (j, e[j])


# ------------------------------------------------------------------ supersampling, passbands
def test_supersampling_is_mean_of_midpoint_subsamples(oracle):
    w = inputs.config2(n_pv=3, n_t=400)
    n_ss, t_exp = 7, w.t_exp
    f = oracle.ma_quad_exact(w.times, w.params, n_ss=n_ss, t_exp=t_exp, prec="f128")
    sub = np.stack([w.times + t_exp * ((s + 0.5) / n_ss - 0.5) for s in range(n_ss)])   # P:L163, midpoints
    fs = np.stack([oracle.ma_quad_exact(sub[s], w.params, prec="f128") for s in range(n_ss)])
    assert np.abs(f - fs.mean(axis=0)).max() <= 1e-15
    f1 = oracle.ma_quad_exact(w.times, w.params, n_ss=1, t_exp=t_exp, prec="f128")
    f0 = oracle.ma_quad_exact(w.times, w.params, n_ss=1, t_exp=0.0, prec="f128")
    assert np.array_equal(f1, f0)
    # converges to the exposure integral: n_ss = 200 vs n_ss = 400
    fa = oracle.ma_quad_exact(w.times[:60], w.params, n_ss=200, t_exp=t_exp, prec="f64")
    fb = oracle.ma_quad_exact(w.times[:60], w.params, n_ss=400, t_exp=t_exp, prec="f64")
    assert np.abs(fa - fb).max() <= 1e-6


def test_k_correction_passbands(oracle):
    """evaluate at mean k, scale each passband's decrement by k_i²/k̂²; equal k reduces to single-passband calls."""
    w = inputs.config3(n_pv=6, n_pb=4, n_t=80)
    p = w.params.copy()
    p[:, 6::3] = p[:, 6:7]   # all passbands share k
    f = oracle.ma_quad_exact(w.times, p, n_pb=4, prec="f128")
    for j in range(4):
        pj = np.concatenate([p[:, :6], p[:, 6 + 3 * j:9 + 3 * j]], axis=1)
        fj = oracle.ma_quad_exact(w.times, pj, n_pb=1, prec="f128")[:, 0]
        assert np.abs(f[:, j] - fj).max() <= 1e-15


def test_bad_parameters_give_nan_rows(oracle):
    w = inputs.config2(n_pv=6, n_t=50)
    p = w.params.copy()
    p[1, 1] = -1.0; p[2, 4] = 1.0; p[3, 6] = -0.1; p[4, 2] = np.nan
    f = oracle.ma_quad_exact(w.times, p, n_ss=2, t_exp=0.01, prec="f64")
    assert np.all(np.isnan(f[1:5])) and np.all(np.isfinite(f[0])) and np.all(np.isfinite(f[5]))


# ------------------------------------------------------------------ interpolated model
def test_table_nodes_are_the_basis_functions(oracle):
    k_min, k_max, n_k, z_max, n_z = 0.05, 0.25, 21, 1.25, 126
    tb = oracle.ma_table_build(k_min, k_max, n_k, z_max, n_z, np.float64, 3, "f128")
    dk, dz = oracle.table_spacing(k_min, k_max, n_k, z_max, n_z)
    kk = k_min + np.arange(n_k) * dk
    zz = np.arange(n_z) * dz
    K, Z = np.meshgrid(kk, zz, indexing="ij")
    ref = np.stack(oracle.ma_basis(K.ravel(), Z.ravel(), "f128"), axis=1).reshape(n_k, n_z, 3)
    assert np.array_equal(tb, ref)
    tb32 = oracle.ma_table_build(k_min, k_max, n_k, z_max, n_z, np.float32, 4, "f128")
    assert np.array_equal(tb32[:, :, :3], ref.astype(np.float32)) and np.all(tb32[:, :, 3] == 0)


def test_bilinear_rule_reproduces_an_affine_table(oracle):
    """Feed the interpolator a table that is affine in (k,z): bilinear interpolation must return it exactly."""
    k_min, dk, n_k, dz, n_z = 0.05, 0.01, 16, 0.01, 131
    kk = k_min + np.arange(n_k) * dk
    zz = np.arange(n_z) * dz
    co = np.array([[0.01, 0.2, 0.03], [0.002, 0.1, -0.01], [0.0, 0.05, 0.02]])   # f = c0 + c1 k + c2 z
    tb = co[None, None, :, 0] + co[None, None, :, 1] * kk[:, None, None] + co[None, None, :, 2] * zz[None, :, None]
    w = inputs.config2(n_pv=12, n_t=3000)
    f = oracle.ma_quad_interp(tb, k_min, dk, dz, w.times, w.params, prec="f128")
    z = oracle.orbit_z(w.times, w.params, prec="f128")[:, :, 0]
    for pv in range(12):
        k, u1, u2 = w.params[pv, 6:9]
        b = [co[f_, 0] + co[f_, 1] * k + co[f_, 2] * z[pv] for f_ in range(3)]
        ref = np.where((z[pv] >= 0) & (z[pv] < 1 + k), quad_flux(b[0], b[1], b[2], u1, u2), 1.0)
        assert np.abs(f[pv, 0] - ref).max() <= 1e-14



def test_bilinear_cell_choice_on_a_non_affine_table(oracle):
    """Cell choice and clamps of the bilinear rule (S§8(c)-2 step 8) on a table that is NOT affine, so a
    wrong cell (ceil/round instead of floor, a shifted clamp, swapped k/z weights) changes the value: expected values are
    numpy.interp along z in each of the two bracketing k-rows, blended linearly in k."""
    k_min, dk, n_k, dz, n_z = 0.05, 0.0125, 17, 0.03125, 41          # dk, dz exactly representable: nodes are exact
    kk = k_min + np.arange(n_k) * dk
    zz = np.arange(n_z) * dz
    K, Z = np.meshgrid(kk, zz, indexing="ij")
    tb = np.stack([Z * Z + 0.1 * K, np.sin(3.0 * Z) + K * K, K * np.exp(Z)], axis=2)
    z_max = zz[-1]
    rng = np.random.default_rng(5)
    kq = np.concatenate([rng.uniform(k_min, kk[-1], 400), kk[[0, 3, 16]], [kk[3] + 0.25 * dk, kk[15] + 0.999 * dk]])
    zq = np.concatenate([rng.uniform(0.0, z_max, 380), zz[[0, 1, 7, 39, 40]], zz[7] + dz * np.array([1e-9, 0.5, 1 - 1e-9]),
                         z_max - dz * np.array([0.75, 0.5, 1e-12]), [z_max + 0.01, z_max + 0.3, 0.0],  # last cell; beyond z_max
                         rng.uniform(0.0, z_max, 11)])
    assert kq.size == zq.size
    got = oracle.interp_basis(tb, k_min, dk, dz, kq, zq, prec="f128")
    ik = np.minimum(np.floor((kq - k_min) / dk).astype(int), n_k - 2)
    fk = (kq - k_min) / dk - ik
    for f in range(3):
        lo = np.array([np.interp(min(z, z_max), zz, tb[i, :, f]) for i, z in zip(ik, zq)])
        hi = np.array([np.interp(min(z, z_max), zz, tb[i + 1, :, f]) for i, z in zip(ik, zq)])
        inside = zq <= z_max
        ref = (1 - fk) * lo + fk * hi
        assert np.abs(got[inside, f] - ref[inside]).max() <= 1e-14
    # beyond z_max the clamp keeps the LAST cell and extrapolates along its segment (iz = n_z-2, fz > 1)
    out = zq > z_max
    for f in range(3):
        seg = lambda i, z: tb[i, -2, f] + (z - zz[-2]) / dz * (tb[i, -1, f] - tb[i, -2, f])
        ref = np.array([(1 - w) * seg(i, z) + w * seg(i + 1, z) for i, w, z in zip(ik[out], fk[out], zq[out])])
        assert np.abs(got[out, f] - ref).max() <= 1e-13
    # exactly on a node the node value comes back (k on a node and z on a node)
    g = oracle.interp_basis(tb, k_min, dk, dz, np.repeat(kk[[0, 5, 16]], 3), np.tile(zz[[0, 9, 40]], 3))
    assert np.abs(g - tb[np.repeat([0, 5, 16], 3), np.tile([0, 9, 40], 3)]).max() <= 1e-15
    # an fp32-stored table is converted on load, the arithmetic stays in the working precision
    g32 = oracle.interp_basis(tb.astype(np.float32), k_min, dk, dz, kq[:50], zq[:50])
    g64 = oracle.interp_basis(tb.astype(np.float32).astype(np.float64), k_min, dk, dz, kq[:50], zq[:50])
    assert np.array_equal(g32, g64)


def test_p11_paper_interpolation_error_figures(oracle):
    """default table n_k=128, n_z=256, Δk=0.02: max error ~4 ppm, mean over the transit ~0.05 ppm;
    P:L216: the maximum sits at the end of ingress / start of egress.  Order-of-magnitude check (the paper does not
    say where its grid sits)."""
    k0, n_k, n_z = 0.09, 128, 256
    tb = oracle.ma_table_build(k0, k0 + 0.02, n_k, 1.0 + k0 + 0.02, n_z, np.float64, 3, "f64")
    dk, dz = oracle.table_spacing(k0, k0 + 0.02, n_k, 1.0 + k0 + 0.02, n_z)
    a, k = 8.0, 0.1
    params = np.array([[0.0, 3.0, a, 88 * DEG, 0, 0, k, 0.4, 0.2]])
    t = np.linspace(-0.07, 0.07, 20001)
    fi = oracle.ma_quad_interp(tb, k0, dk, dz, t, params, prec="f64")[0, 0]
    fe = oracle.ma_quad_exact(t, params, prec="f64")[0, 0]
    z = np.abs(oracle.orbit_z(t, params, prec="f64")[0, :, 0])
    err = np.abs(fi - fe)
    in_tr = z < 1 + k
    assert 0.5e-6 < err.max() < 40e-6
    assert 0.005e-6 < err[in_tr].mean() < 2e-6
    assert abs(z[np.argmax(err)] - (1 - k)) < 3 * dz or abs(z[np.argmax(err)] - (1 + k)) < 3 * dz
    # coarser table in k only: a smaller effect than the z-resolution (n_k = 8 -> ~8 ppm)
    tb8 = oracle.ma_table_build(k0, k0 + 0.02, 8, 1.0 + k0 + 0.02, n_z, np.float64, 3, "f64")
    dk8, _ = oracle.table_spacing(k0, k0 + 0.02, 8, 1.0 + k0 + 0.02, n_z)
    f8 = oracle.ma_quad_interp(tb8, k0, dk8, dz, t, params, prec="f64")[0, 0]
    assert np.abs(f8 - fe).max() < 80e-6


def test_interp_k_outside_table_falls_back_to_exact(oracle):
    tb = oracle.ma_table_build(0.05, 0.1, 11, 1.1, 111, np.float64, 3, "f64")
    dk, dz = oracle.table_spacing(0.05, 0.1, 11, 1.1, 111)
    params = np.array([[0.0, 3.0, 8.0, 88 * DEG, 0, 0, 0.15, 0.4, 0.2]])
    t = np.linspace(-0.1, 0.1, 201)
    fi = oracle.ma_quad_interp(tb, 0.05, dk, dz, t, params, prec="f64")
    fe = oracle.ma_quad_exact(t, params, prec="f64")
    assert np.array_equal(fi, fe)


def test_f64_vs_f128_flux_on_bulk_workloads(oracle):
    """P9 (restricted): the double instantiation agrees with the quad arbiter to 1e-12 away from case boundaries."""
    w = inputs.config2(n_pv=8, n_t=2000)
    a = oracle.ma_quad_exact(w.times, w.params, n_ss=3, t_exp=w.t_exp, prec="f64")
    b = oracle.ma_quad_exact(w.times, w.params, n_ss=3, t_exp=w.t_exp, prec="f128")
    assert np.abs(a - b).max() <= 1e-11


# ------------------------------------------------------------------------------------------- likelihood (S§8(f) NEXT-1)
def test_chi2_definition_pins(oracle):
    """chi2_of_flux against facts that do not involve it: zero residuals, one known residual, scaling with 1/sigma,
    additivity over passbands, and the expectation n for unit-variance noise."""
    w = inputs.config3(n_pv=3, n_pb=2, n_t=200)
    f = oracle.ma_quad_exact(w.times, w.params, 2, 1, 0.0, prec="f64")
    ones = np.ones((2, 200))
    assert np.all(oracle.chi2_of_flux(f, f[1], 7.0 * ones)[1] == 0.0)
    obs = f[0].copy()
    obs[1, 17] += 3e-4                                        # one residual of 3 sigma at sigma = 1e-4
    c = oracle.chi2_of_flux(f[:1], obs, 1e4 * ones)
    assert abs(c[0] - 9.0) < 1e-9
    assert np.allclose(oracle.chi2_of_flux(f, obs, 2e4 * ones), 4.0 * oracle.chi2_of_flux(f, obs, 1e4 * ones), rtol=1e-14)
    both = oracle.chi2_of_flux(f, obs, 1e4 * ones)
    each = sum(oracle.chi2_of_flux(f[:, j:j + 1], obs[j:j + 1], 1e4 * ones[j:j + 1]) for j in range(2))
    assert np.allclose(both, each, rtol=1e-14)
    rng = np.random.default_rng(5)
    sig = 2e-4
    noisy = f[2] + sig * rng.standard_normal(f[2].shape)
    c = oracle.chi2_of_flux(f[2:3], noisy, ones / sig)[0]
    assert abs(c - 400.0) < 5 * np.sqrt(2 * 400.0)              # chi-square with 400 degrees of freedom
    # the decomposition the kernel uses is an identity: ((o-F)w)^2 = ((o-1)w)^2 + (1-F) w^2 (2(o-1) + (1-F))
    o, F, ww = noisy, f[2], ones / sig
    lhs = ((o - F) * ww) ** 2
    rhs = ((o - 1) * ww) ** 2 + (1 - F) * ww ** 2 * (2 * (o - 1) + (1 - F))
    assert np.abs(lhs - rhs).max() <= 1e-9 * max(1.0, np.abs(lhs).max())


def test_per_passband_k_mode_pins(oracle):
    """Exact per-passband-k oracle: equal k in every passband reduces to the mean-k model; with config-3's spread the two
    differ by the few 1e-4 SURVEY §8(f) quotes; a uniform-disk passband inside the limb is exactly 1 - k_j²."""
    w = inputs.config3(n_pv=4, n_pb=3, n_t=120)
    p = w.params.copy()
    a = oracle.ma_quad_exact_pbk(w.times, p, 3, prec="f64")
    b = oracle.ma_quad_exact(w.times, p, 3, prec="f64")
    d = np.abs(a - b).max()
    assert 1e-6 < d < 2e-3
    p[:, 9] = p[:, 6]; p[:, 12] = p[:, 6]
    assert np.abs(oracle.ma_quad_exact_pbk(w.times, p, 3, prec="f64") - oracle.ma_quad_exact(w.times, p, 3, prec="f64")).max() < 1e-14
    q = np.array([[0.0, 3.0, 8.0, np.pi / 2, 0.0, 0.0, 0.1, 0.0, 0.0, 0.2, 0.0, 0.0]])
    f = oracle.ma_quad_exact_pbk(np.array([0.0]), q, 2, prec="f64")
    assert abs(f[0, 0, 0] - (1 - 0.01)) < 1e-15 and abs(f[0, 1, 0] - (1 - 0.04)) < 1e-15


# ------------------------------------------------------------------ NEXT-4: the Giménez model
def test_next4_kopal_polynomials(oracle):
    # G_j(p,q;x) = 2F1(-j, j+p; q; x) (R20): the oracle's two-binomial evaluation against mpmath's hypergeometric
    # function and, where that sum is still benign, against the defining sum itself
    import mpmath as mp
    mp.mp.dps = 40
    for j, p, q, x in [(0, 3.0, 2.0, 0.4), (1, 3.5, 2.5, 0.3), (5, 3.5, 2.5, 0.3), (17, 4.0, 1.0, 0.55), (40, 3.5, 2.5, 0.909),
                       (60, 3.0, 1.0, 0.7), (60, 3.5, 1.0, 0.02), (80, 3.0, 2.0, 0.97)]:
        ref = mp.hyp2f1(-j, j + p, q, x)
        got = oracle.kopal_G(j, p, q, [x], "f128")[0]
        assert abs(got - ref) <= 1e-13 * max(1.0, abs(ref)), (j, p, q, x)
        if j <= 17:
            assert abs(oracle.kopal_G(j, p, q, [x], "defsum")[0] - ref) <= 1e-13
    assert oracle.kopal_G(1, 3.5, 2.5, [0.3], "f128")[0] == pytest.approx(1 - 4.5 * 0.3 / 2.5, abs=1e-15)   # 1 - (1+p) x / q


def test_next4_series_converges_to_the_definition(oracle):
    # Eq. 3 as printed, with Kopal's polynomials, against α_n = (1/π) ∫_occ μ^n dA (the definition that follows from Eq. 4, 7, 8)
    # by 30-digit quadrature: the error falls as N_J grows (Fig. 1) in every region of (k, z)
    from oracle.ma_definition import alpha_n_definition
    for n, k, z in [(0, 0.1, 0.3), (1, 0.1, 0.3), (2, 0.2, 0.9), (1, 0.1, 1.0), (3, 0.15, 0.0), (1, 0.3, 0.75), (4, 0.05, 1.02)]:
        ref = float(alpha_n_definition(n, k, z))
        err = [abs(oracle.gimenez_alpha(n, nj, k, z, "f128")[0] - ref) for nj in (5, 40, 100)]
        # the convergence oscillates (the partial sums overshoot alternately), so the pin is on the envelope
        assert err[0] > 5 * max(err[1], err[2]), (n, k, z, err)
        assert err[2] <= 1.5e-6 and err[1] <= 5e-6, (n, k, z, err)
    # n = 0 and n = 2 have elementary values inside the disk: α_0 = k², α_2 = k² - k²(k² + 2z²)/2
    a0 = oracle.gimenez_alpha(0, 100, 0.1, 0.4, "f128")[0]
    a2 = oracle.gimenez_alpha(2, 100, 0.1, 0.4, "f128")[0]
    assert abs(a0 - 0.01) <= 1e-6 and abs(a2 - (0.01 - 0.01 * (0.01 + 0.32) / 2)) <= 1e-6
    assert oracle.gimenez_alpha(1, 40, 0.1, 1.1, "f128")[0] == 0.0 and oracle.gimenez_alpha(1, 40, 0.1, 1.3, "f128")[0] == 0.0


def test_next4_quadratic_law_reduces_to_mandel_agol(oracle):
    # N = 2 with u_1 = a + 2b, u_2 = -b is the quadratic law: the Giménez flux tends to the Mandel-Agol flux of the same
    # oracle (independent code: closed forms + Carlson integrals) as N_J grows; supersampling and two passbands share the α_n
    t = np.linspace(-0.09, 0.09, 19)
    a, b = 0.4, 0.2
    pm = np.array([[0.0, 3.0, 8.0, math.radians(88.0), 0.0, 0.0, 0.1, a, b]])
    pg = np.array([[0.0, 3.0, 8.0, math.radians(88.0), 0.0, 0.0, 0.1, a + 2 * b, -b, 0.3, 0.0]])   # second passband: linear law u = 0.3
    fm = oracle.ma_quad_exact(t, pm, prec="f128")[0, 0]
    pl = pm.copy(); pl[0, 7:] = (0.3, 0.0)
    fl = oracle.ma_quad_exact(t, pl, prec="f128")[0, 0]
    errs = []
    for nj in (5, 40, 80):
        fg = oracle.gimenez_exact(t, pg, n_pb=2, n_ldc=2, n_j=nj, prec="f128")[0]
        errs.append(max(np.abs(fg[0] - fm).max(), np.abs(fg[1] - fl).max()))
    assert errs[0] > 5 * max(errs[1], errs[2]) and errs[1] <= 3e-5 and errs[2] <= 5e-6, errs
    # out of transit exactly 1; supersampled = mean of the subsample fluxes
    tt = np.array([0.03, 0.2])
    f1 = oracle.gimenez_exact(tt, pg, 2, 2, 30, 4, 0.02, prec="f128")
    offs = 0.02 * ((np.arange(4) + 0.5) / 4 - 0.5)
    fs = oracle.gimenez_exact((tt[:, None] + offs[None, :]).ravel(), pg, 2, 2, 30, prec="f128").reshape(2, 2, 4).mean(axis=2)
    assert np.abs(f1[0] - fs).max() <= 1e-15 and np.all(f1[0][:, 1] == 1.0)
