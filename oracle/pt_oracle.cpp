// pt_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, obviously-correct CPU oracle for the batched quadratic Mandel–Agol transit model that
// PyTransit (Parviainen 2015, arXiv 1504.07433; /root/reference/PAPER.md, cited "P:Ln") evaluates.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
// It shares NO code, header, table or constant generator with the CUDA path under
// paper_1504_07433_b200/csrc/, and neither side includes the other.
//
// What it computes (DESIGN.md §2 lists every reading of the paper that is taken here):
//   flux f(k,z) = 1 - [(1-c) λe + c λd + b ηd] / (1 - a/3 - b/6),  c = a + 2b          P:L136 (Eq. 13)
//   with (a,b) = (u1,u2) the quadratic limb-darkening coefficients of                 P:L86  (Eq. 6)
//   λe, λd, ηd "as defined in Mandel & Agol (2002)"
//   multi-passband: λ's once per (k,z), linear combine per passband
//   k-correction for per-passband radius ratios: evaluate at mean k, scale by k_i²/k̂²
//   supersampling: mean of n evenly distributed subsamples inside each exposure
//   interpolated model: bilinear interpolation in (k,z) tables of λe, λd, ηd
//   orbit: circular, and eccentric by a Kepler solve (paper names the solvers only)
//   the other orbit routines: fixed-point iteration, two series, e-based dispatch      P:L31 (R19)
//   the Giménez model with general limb darkening, Eq. 1-12 as printed                 P:L40-L128 (R20)
//
// Method choices that are deliberately DIFFERENT from the CUDA path (so that a shared mistake is unlikely):
//   * elliptic integrals K, E, Π by Carlson's symmetric forms R_F, R_D, R_J (duplication), not Bulirsch cel;
//   * the textbook closed forms of the three basis functions (acos for the angles, q = p² - z², Π(n|m) with
//     n and m formed directly), not the cancellation-free rearrangement the kernel uses;
//   * Kepler's equation by bisection, not Newton;
//   * every function is a template on the real type and instantiated for `double` (the timed CPU baseline)
//     and for `__float128` (libquadmath, ~34 digits: the PARITY ARBITER — the textbook forms lose up to ~1e-9
//     in double within 1e-6 of a case boundary, in quad they hold ~1e-24 there).
//
// Two operations are fixed to IEEE double on both sides of the parity comparison because the *inputs* are doubles
// and the result is ill-conditioned in them (readings H1, H2): the subsample time and the phase fold.
// This file is compiled with -ffp-contract=off so they are exactly the operations written.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): integral definitions of λe, λd*, ηd by quadrature
// (oracle/ma_definition.py: 1-D tanh-sinh with mpmath at 30 digits, 2-D Gauss–Legendre, 2-D pixel brute force),
// mpmath ellipk/ellipe/ellippi for the Carlson forms, closed forms (z=0, z<=1-k, u=0 lens area, k>=1 cover),
// symmetry/periodicity, Kepler residuals and the e->0 limit, z(t0) identity, the paper's interpolation error
// figures, linearity in (u1,u2).  Nothing here is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __float128 quad;

// ---------------------------------------------------------------------------------------------------------
// Real-type shims: the same source text serves double and __float128.
// ---------------------------------------------------------------------------------------------------------
static inline double x_sqrt(double x) { return std::sqrt(x); }
static inline double x_sin(double x) { return std::sin(x); }
static inline double x_cos(double x) { return std::cos(x); }
static inline double x_acos(double x) { return std::acos(x); }
static inline double x_atan(double x) { return std::atan(x); }
static inline double x_atanh(double x) { return std::atanh(x); }
static inline double x_atan2(double y, double x) { return std::atan2(y, x); }
static inline double x_fabs(double x) { return std::fabs(x); }
static inline double x_floor(double x) { return std::floor(x); }
static inline quad x_sqrt(quad x) { return sqrtq(x); }
static inline quad x_sin(quad x) { return sinq(x); }
static inline quad x_cos(quad x) { return cosq(x); }
static inline quad x_acos(quad x) { return acosq(x); }
static inline quad x_atan(quad x) { return atanq(x); }
static inline quad x_atanh(quad x) { return atanhq(x); }
static inline quad x_atan2(quad y, quad x) { return atan2q(y, x); }
static inline quad x_fabs(quad x) { return fabsq(x); }
static inline quad x_floor(quad x) { return floorq(x); }
static inline double x_pow(double x, double y) { return std::pow(x, y); }
static inline quad x_pow(quad x, quad y) { return powq(x, y); }
static inline double x_tgamma(double x) { return std::tgamma(x); }
static inline quad x_tgamma(quad x) { return tgammaq(x); }

template <class R> struct Real;
template <> struct Real<double> {
  static double pi() { return 3.141592653589793238462643383279502884; }
  static double eps() { return 1.1102230246251565e-16; }  // 2^-53
};
template <> struct Real<quad> {
  static quad pi() { return M_PIq; }
  static quad eps() { return FLT128_EPSILON / 2; }  // 2^-113
};

template <class R> static inline R x_max(R a, R b) { return a > b ? a : b; }
template <class R> static inline R x_min(R a, R b) { return a < b ? a : b; }

// ---------------------------------------------------------------------------------------------------------
// Carlson symmetric elliptic integrals by duplication (B. C. Carlson, Numer. Algorithms 10 (1995) 13; the series
// are the 5th-order truncations, error O(r^6) with r the largest relative deviation from the mean, so the loop runs
// until r^6 is below the unit roundoff of R).
// ---------------------------------------------------------------------------------------------------------
template <class R> static R conv_tol() {
  // r such that r^6 ~ eps/16: eps^(1/6) by repeated square/cube roots is overkill; these constants are safe.
  return sizeof(R) == sizeof(double) ? R(1.0e-3) : R(1.0e-6);
}

// R_C(1, 1+e), e > -1:  atan(sqrt(e))/sqrt(e)  (e>0),  atanh(sqrt(-e))/sqrt(-e)  (e<0),  1 (e=0).
template <class R> static R carlson_rc1(R e) {
  if (e == R(0)) return R(1);
  if (e > R(0)) { R s = x_sqrt(e); return x_atan(s) / s; }
  R s = x_sqrt(-e);
  return x_atanh(s) / s;
}

// R_F(x,y,z) = (1/2) ∫_0^∞ [(t+x)(t+y)(t+z)]^(-1/2) dt ; at most one argument zero.
template <class R> static R carlson_rf(R x, R y, R z) {
  const R tol = conv_tol<R>();
  for (int it = 0; it < 200; ++it) {
    R A = (x + y + z) / R(3);
    R X = (A - x) / A, Y = (A - y) / A, Z = (A - z) / A;
    if (x_max(x_max(x_fabs(X), x_fabs(Y)), x_fabs(Z)) < tol) {
      R E2 = X * Y - Z * Z, E3 = X * Y * Z;
      return (R(1) - E2 / R(10) + E3 / R(14) + E2 * E2 / R(24) - R(3) * E2 * E3 / R(44)) / x_sqrt(A);
    }
    R sx = x_sqrt(x), sy = x_sqrt(y), sz = x_sqrt(z);
    R lam = sx * sy + sy * sz + sz * sx;
    x = (x + lam) / R(4); y = (y + lam) / R(4); z = (z + lam) / R(4);
  }
  return std::numeric_limits<double>::quiet_NaN();
}

// R_D(x,y,z) = (3/2) ∫_0^∞ [(t+x)(t+y)]^(-1/2) (t+z)^(-3/2) dt ; z > 0.
template <class R> static R carlson_rd(R x, R y, R z) {
  const R tol = conv_tol<R>();
  R sum = R(0), fac = R(1);
  for (int it = 0; it < 200; ++it) {
    R A = (x + y + R(3) * z) / R(5);
    R X = (A - x) / A, Y = (A - y) / A, Z = (A - z) / A;
    if (x_max(x_max(x_fabs(X), x_fabs(Y)), x_fabs(Z)) < tol) {
      R E2 = X * Y - R(6) * Z * Z, E3 = (R(3) * X * Y - R(8) * Z * Z) * Z;
      R E4 = R(3) * (X * Y - Z * Z) * Z * Z, E5 = X * Y * Z * Z * Z;
      R ser = R(1) - R(3) * E2 / R(14) + E3 / R(6) + R(9) * E2 * E2 / R(88) - R(3) * E4 / R(22) -
              R(9) * E2 * E3 / R(52) + R(3) * E5 / R(26);
      return R(3) * sum + fac * ser / (A * x_sqrt(A));
    }
    R sx = x_sqrt(x), sy = x_sqrt(y), sz = x_sqrt(z);
    R lam = sx * sy + sy * sz + sz * sx;
    sum += fac / (sz * (z + lam));
    fac /= R(4);
    x = (x + lam) / R(4); y = (y + lam) / R(4); z = (z + lam) / R(4);
  }
  return std::numeric_limits<double>::quiet_NaN();
}

// R_J(x,y,z,p) = (3/2) ∫_0^∞ [(t+x)(t+y)(t+z)]^(-1/2) (t+p)^(-1) dt ; p > 0.
template <class R> static R carlson_rj(R x, R y, R z, R p) {
  const R tol = conv_tol<R>();
  const R delta = (p - x) * (p - y) * (p - z);
  R sum = R(0), fac = R(1), fac3 = R(1);  // fac = 4^-m, fac3 = 4^-3m
  for (int it = 0; it < 200; ++it) {
    R A = (x + y + z + R(2) * p) / R(5);
    R X = (A - x) / A, Y = (A - y) / A, Z = (A - z) / A, P = (A - p) / A;
    if (x_max(x_max(x_fabs(X), x_fabs(Y)), x_max(x_fabs(Z), x_fabs(P))) < tol) {
      R E2 = X * Y + X * Z + Y * Z - R(3) * P * P;
      R E3 = X * Y * Z + R(2) * E2 * P + R(4) * P * P * P;
      R E4 = (R(2) * X * Y * Z + E2 * P + R(3) * P * P * P) * P;
      R E5 = X * Y * Z * P * P;
      R ser = R(1) - R(3) * E2 / R(14) + E3 / R(6) + R(9) * E2 * E2 / R(88) - R(3) * E4 / R(22) -
              R(9) * E2 * E3 / R(52) + R(3) * E5 / R(26);
      return R(6) * sum + fac * ser / (A * x_sqrt(A));
    }
    R sx = x_sqrt(x), sy = x_sqrt(y), sz = x_sqrt(z), sp = x_sqrt(p);
    R lam = sx * sy + sy * sz + sz * sx;
    R dm = (sp + sx) * (sp + sy) * (sp + sz);
    R em = fac3 * delta / (dm * dm);
    sum += fac / dm * carlson_rc1<R>(em);
    fac /= R(4); fac3 /= R(64);
    x = (x + lam) / R(4); y = (y + lam) / R(4); z = (z + lam) / R(4); p = (p + lam) / R(4);
  }
  return std::numeric_limits<double>::quiet_NaN();
}

// Complete elliptic integrals in PARAMETER form (m = k², "minus" sign convention for n), m < 1, n < 1:
//   K(m) = ∫_0^{π/2} (1 - m sin²θ)^(-1/2) dθ,   E(m) = ∫_0^{π/2} (1 - m sin²θ)^(1/2) dθ,
//   Π(n|m) = ∫_0^{π/2} (1 - n sin²θ)^(-1) (1 - m sin²θ)^(-1/2) dθ.
template <class R> static R ell_K(R m) { return carlson_rf<R>(R(0), R(1) - m, R(1)); }
template <class R> static R ell_E(R m) {
  return carlson_rf<R>(R(0), R(1) - m, R(1)) - m / R(3) * carlson_rd<R>(R(0), R(1) - m, R(1));
}
template <class R> static R ell_Pi(R n, R m) {
  return carlson_rf<R>(R(0), R(1) - m, R(1)) + n / R(3) * carlson_rj<R>(R(0), R(1) - m, R(1), R(1) - n);
}

// ---------------------------------------------------------------------------------------------------------
// The three limb-darkening-independent basis functions of Eq. 13 at radius ratio p and projected
// separation z >= 0.  Definitions (from Eq. 6 + Eq. 13 alone, DESIGN.md §2 R1-R3), occ = part of the unit disk within
// distance p of the planet centre:
//     λe = (1/π) ∫_occ dA,   λd* = (1/π) ∫_occ sqrt(1-r²) dA,   ηd = (1/π) ∫_occ r² dA.
// λd* is Mandel & Agol's λd + (2/3)Θ(p-z): Eq. 13 as printed has no Θ term, so its "λd" is this continuous function.
// Closed forms: Mandel & Agol (2002) Table 1 with its published errata, written in textbook form.
// ---------------------------------------------------------------------------------------------------------
template <class R> static void ma_basis(R p, R z, R* le, R* ld, R* ed) {
  const R pi = Real<R>::pi();
  const R one = R(1), two = R(2), three = R(3);
  // no occultation: planet of zero size, or disks do not overlap
  if (p <= R(0) || z >= one + p) { *le = R(0); *ld = R(0); *ed = R(0); return; }
  // star completely covered
  if (p >= one && z <= p - one) { *le = one; *ld = two / three; *ed = one / two; return; }

  const R a = (z - p) * (z - p), b = (z + p) * (z + p), q = p * p - z * z;
  const R eta2 = p * p / two * (p * p + two * z * z);
  const R theta = (z < p) ? two / three : R(0);  // (2/3)Θ(p-z) for the generic rows (z != p)

  if (z <= one - p) {  // planet disk entirely inside the stellar disk (inner contact included)
    *le = p * p;
    *ed = eta2;
    if (z == one - p) {  // inner contact, any 0<p<1
      *ld = two / (three * pi) * x_acos(one - two * p) -
            R(4) / (R(9) * pi) * (three + two * p - R(8) * p * p) * x_sqrt(p * (one - p));
    } else if (z == R(0)) {  // concentric
      R w = one - p * p;
      *ld = two / three * (one - w * x_sqrt(w));
    } else if (z == p) {  // planet edge through the star centre, p < 1/2
      R m = R(4) * p * p;
      *ld = one / three + two / (R(9) * pi) * (R(4) * (two * p * p - one) * ell_E<R>(m) + (one - R(4) * p * p) * ell_K<R>(m));
    } else {
      R m = R(4) * z * p / (one - a);
      R n = (a - b) / a;
      R K = ell_K<R>(m), E = ell_E<R>(m), Pi = ell_Pi<R>(n, m);
      *ld = two / (R(9) * pi * x_sqrt(one - a)) *
                ((one - R(5) * z * z + p * p + q * q) * K + (one - a) * (z * z + R(7) * p * p - R(4)) * E -
                 three * q / a * Pi) + theta;
    }
    return;
  }

  // partial overlap |1-p| < z < 1+p
  const R kap0 = x_acos((p * p + z * z - one) / (two * p * z));
  const R kap1 = x_acos((one - p * p + z * z) / (two * z));
  const R T = x_sqrt((one - a) * (b - one));  // = sqrt(4z² - (1+z²-p²)²)
  *le = (p * p * kap0 + kap1 - T / two) / pi;
  *ed = (kap1 + two * eta2 * kap0 - (one + R(5) * p * p + z * z) / R(4) * T) / (two * pi);
  if (z == p) {  // p >= 1/2 here
    if (p == one / two) {
      *ld = one / three - R(4) / (R(9) * pi);
    } else {
      R m = one / (R(4) * p * p);
      *ld = one / three + R(16) * p / (R(9) * pi) * (two * p * p - one) * ell_E<R>(m) -
            (one - R(4) * p * p) * (three - R(8) * p * p) / (R(9) * pi * p) * ell_K<R>(m);
    }
  } else {
    R m = (one - a) / (R(4) * z * p);
    R n = (a - one) / a;
    R K = ell_K<R>(m), E = ell_E<R>(m), Pi = ell_Pi<R>(n, m);
    *ld = (((one - b) * (two * b + a - three) - three * q * (b - two)) * K +
           R(4) * p * z * (z * z + R(7) * p * p - R(4)) * E - three * q / a * Pi) / (R(9) * pi * x_sqrt(p * z)) + theta;
  }
}

// ---------------------------------------------------------------------------------------------------------
// Parameter rows: [t0, P, a/R*, i, e, w, k_0,u1_0,u2_0, k_1,u1_1,u2_1, ...]  (6 + 3 n_pb doubles), angles in radians.
// ---------------------------------------------------------------------------------------------------------
static bool row_is_valid(const double* pr, int n_pb) {
  for (int j = 0; j < 6 + 3 * n_pb; ++j) if (!std::isfinite(pr[j])) return false;
  if (!(pr[1] > 0.0)) return false;               // period
  if (!(pr[2] > 0.0)) return false;               // a/R*
  if (!(pr[4] >= 0.0 && pr[4] < 1.0)) return false;  // eccentricity
  for (int j = 0; j < n_pb; ++j) {
    const double* c = pr + 6 + 3 * j;
    if (!(c[0] >= 0.0)) return false;                          // radius ratio
    if (1.0 - c[1] / 3.0 - c[2] / 6.0 == 0.0) return false;    // unocculted flux must not vanish
  }
  return true;
}

// H2: subsample time, IEEE double, operations exactly as written (midpoints of n equal parts).
static inline double subsample_time(double t, double t_exp, int s, int n_ss) {
  if (n_ss == 1) return t;
  double off = t_exp * ((s + 0.5) / n_ss - 0.5);
  return t + off;
}
// H1: phase fold, IEEE double, one subtraction, one division, round-to-nearest-even, one subtraction.
static inline double fold_phase(double t, double t0, double P) {
  double x = (t - t0) / P;
  return x - std::nearbyint(x);
}

// Kepler's equation E - e sin E = M for M in [-π, π] by bisection on [M-e, M+e] (f is increasing in E).
template <class R> static R kepler_E(R M, R e) {
  R lo = M - e, hi = M + e;
  for (int it = 0; it < 400; ++it) {
    R mid = (lo + hi) / R(2);
    if (mid <= lo || mid >= hi) break;  // interval is one ulp wide
    R f = mid - e * x_sin(mid) - M;
    if (f > R(0)) hi = mid; else lo = mid;
  }
  return (lo + hi) / R(2);
}

// ---- the other orbit routines the paper names ("circular and elliptic orbits (using either Newton's method,
// iteration, or two series approximations) ... selects the most appropriate orbit calculation routine based on the
// eccentricity").  The paper gives no formulas; R19 fixes the reading:
//   iteration            the fixed-point iteration E <- M + e sin E from E = M (contraction with rate e), run to a fixed point
//   series, order 3 / 5  the classical expansion of the equation of the centre f - M in powers of e (e.g. Brouwer & Clemence
//                        1961, ch. II; Murray & Dermott 1999, eq. 2.88), truncated after e^3 and after e^5:
//     f = M + (2e - e^3/4 + 5e^5/96) sin M + (5e^2/4 - 11e^4/24) sin 2M + (13e^3/12 - 43e^5/64) sin 3M
//           + (103e^4/96) sin 4M + (1097e^5/960) sin 5M
//   The position then follows from the true anomaly f: r/a = (1-e^2)/(1 + e cos f).
enum { SOLVER_EXACT = 0, SOLVER_NEWTON = 1, SOLVER_ITER = 2, SOLVER_PS3 = 3, SOLVER_PS5 = 4, SOLVER_FAST = 5 };

template <class R> static R kepler_E_iteration(R M, R e) {
  R E = M;
  for (int it = 0; it < 100000; ++it) {
    const R En = M + e * x_sin(E);
    const R d = En > E ? En - E : E - En;
    E = En;
    if (d == R(0)) break;                       // a fixed point in this arithmetic
    const R scale = (E > R(0) ? E : -E) + R(1);
    if (d <= scale * Real<R>::eps()) break;     // moves by less than an ulp
  }
  return E;
}
template <class R> static R true_anomaly_series(R M, R e, int order) {
  const R e2 = e * e, e3 = e2 * e;
  if (order == 3)
    return M + (R(2) * e - e3 / R(4)) * x_sin(M) + (R(5) * e2 / R(4)) * x_sin(R(2) * M) + (R(13) * e3 / R(12)) * x_sin(R(3) * M);
  const R e4 = e2 * e2, e5 = e4 * e;
  return M + (R(2) * e - e3 / R(4) + R(5) * e5 / R(96)) * x_sin(M) + (R(5) * e2 / R(4) - R(11) * e4 / R(24)) * x_sin(R(2) * M) +
         (R(13) * e3 / R(12) - R(43) * e5 / R(64)) * x_sin(R(3) * M) + (R(103) * e4 / R(96)) * x_sin(R(4) * M) +
         (R(1097) * e5 / R(960)) * x_sin(R(5) * M);
}
// Which routine the eccentricity selects (R19): exact = circular for e == 0, else a full-precision Kepler
// solve; fast = the cheapest routine whose truncation error in the true anomaly stays below 2e-9 rad
// (order 3: 1.5 e^4 <= 2e-9 for e <= 0.006; order 5: 2.2 e^6 <= 2e-9 for e <= 0.03), else the Kepler solve.
static inline int dispatch_solver(int solver, double e) {
  if (solver == SOLVER_FAST) return e == 0.0 ? SOLVER_EXACT : (e <= 0.006 ? SOLVER_PS3 : (e <= 0.03 ? SOLVER_PS5 : SOLVER_NEWTON));
  return solver;
}

// Projected separation at folded phase ph (cycles, in [-1/2, 1/2]); sign: +z planet in front, -z behind the star.
// Observer on +Z; t0 is the time of inferior conjunction (true anomaly f = π/2 - w); standard two-body projection.
template <class R> struct Orbit {
  R a, cosi, e, sinw, cosw, rt1me2, Mtr;
  bool circular;
  explicit Orbit(const double* pr) {
    a = R(pr[2]);
    cosi = x_cos(R(pr[3]));
    e = R(pr[4]);
    circular = (pr[4] == 0.0);
    sinw = x_sin(R(pr[5])); cosw = x_cos(R(pr[5]));
    rt1me2 = x_sqrt((R(1) - e) * (R(1) + e));
    R ftr = Real<R>::pi() / R(2) - R(pr[5]);
    R Etr = R(2) * x_atan2(x_sqrt(R(1) - e) * x_sin(ftr / R(2)), x_sqrt(R(1) + e) * x_cos(ftr / R(2)));
    Mtr = Etr - e * x_sin(Etr);
  }
  // `solver`: SOLVER_EXACT / SOLVER_NEWTON = the Kepler solve of this oracle (bisection: "Newton" names the method of the
  // CUDA path, the root is the same), SOLVER_ITER, SOLVER_PS3, SOLVER_PS5; a non-exact routine is used as asked even for e == 0.
  R z_signed_solver(double ph, int solver) const {
    const R pi = Real<R>::pi();
    if (solver == SOLVER_EXACT || solver == SOLVER_NEWTON) return z_signed(ph);
    R M = R(2) * pi * R(ph) + Mtr;
    if (M > pi) M -= R(2) * pi;
    if (M <= -pi) M += R(2) * pi;
    R A, B;
    if (solver == SOLVER_ITER) {
      R E = kepler_E_iteration<R>(M, e);
      R cE = x_cos(E), sE = x_sin(E);
      A = cosw * (cE - e) - sinw * rt1me2 * sE;
      B = sinw * (cE - e) + cosw * rt1me2 * sE;
    } else {
      R f = true_anomaly_series<R>(M, e, solver == SOLVER_PS3 ? 3 : 5);
      R cf = x_cos(f), sf = x_sin(f);
      R rr = (R(1) - e) * (R(1) + e) / (R(1) + e * cf);       // r / a
      A = rr * (cosw * cf - sinw * sf);                       // (r/a) cos(w+f)
      B = rr * (sinw * cf + cosw * sf);
    }
    R Bc = B * cosi;
    R z = a * x_sqrt(A * A + Bc * Bc);
    return B > R(0) ? z : -z;
  }
  R z_signed(double ph) const {
    const R pi = Real<R>::pi();
    if (circular) {
      R phi = R(2) * pi * R(ph);
      R sn = x_sin(phi), cs = x_cos(phi);
      R z = a * x_sqrt(sn * sn + cosi * cosi * cs * cs);
      return cs > R(0) ? z : -z;
    }
    R M = R(2) * pi * R(ph) + Mtr;
    if (M > pi) M -= R(2) * pi;
    if (M <= -pi) M += R(2) * pi;
    R E = kepler_E<R>(M, e);
    R cE = x_cos(E), sE = x_sin(E);
    R A = cosw * (cE - e) - sinw * rt1me2 * sE;  // (r/a) cos(w+f)
    R B = sinw * (cE - e) + cosw * rt1me2 * sE;  // (r/a) sin(w+f)
    R Bc = B * cosi;
    R z = a * x_sqrt(A * A + Bc * Bc);
    return B > R(0) ? z : -z;
  }
};

// Per-passband constants of one parameter row.
template <class R> struct Passbands {
  R khat;
  std::vector<R> c, u2, norm, g;
  Passbands(const double* pr, int n_pb) : c(n_pb), u2(n_pb), norm(n_pb), g(n_pb) {
    R ksum = R(0);
    for (int j = 0; j < n_pb; ++j) ksum += R(pr[6 + 3 * j]);
    khat = ksum / R(n_pb);
    for (int j = 0; j < n_pb; ++j) {
      R k = R(pr[6 + 3 * j]), u1 = R(pr[7 + 3 * j]), v2 = R(pr[8 + 3 * j]);
      c[j] = u1 + R(2) * v2;
      u2[j] = v2;
      norm[j] = R(1) - u1 / R(3) - v2 / R(6);
      g[j] = (khat > R(0)) ? (k * k) / (khat * khat) : R(0);
    }
  }
  R flux(int j, R le, R ld, R ed) const {
    return R(1) - g[j] * ((R(1) - c[j]) * le + c[j] * ld + u2[j] * ed) / norm[j];
  }
};

// ---------------------------------------------------------------------------------------------------------
// Bilinear table lookup (R10, R12): table[n_k][n_z][n_fn], node (i,j) at
// k = k_min + i dk, z = j dz.
// ---------------------------------------------------------------------------------------------------------
struct TableView {
  const void* data; int dtype /*0 f64, 1 f32*/; int n_k, n_z, n_fn; double k_min, dk, dz;
  double at(int ik, int iz, int f) const {
    size_t o = ((size_t)ik * n_z + iz) * n_fn + f;
    return dtype == 0 ? ((const double*)data)[o] : (double)((const float*)data)[o];
  }
};
template <class R> static void interp_basis(const TableView& tb, R khat, R z, R* out3) {
  R rk = (khat - R(tb.k_min)) / R(tb.dk);
  int ik = (int)x_floor(rk); if (ik > tb.n_k - 2) ik = tb.n_k - 2; if (ik < 0) ik = 0;
  R fk = rk - R(ik);
  R rz = z / R(tb.dz);
  int iz = (int)x_floor(rz); if (iz > tb.n_z - 2) iz = tb.n_z - 2; if (iz < 0) iz = 0;
  R fz = rz - R(iz);
  for (int f = 0; f < 3; ++f) {
    R t00 = R(tb.at(ik, iz, f)), t01 = R(tb.at(ik, iz + 1, f));
    R t10 = R(tb.at(ik + 1, iz, f)), t11 = R(tb.at(ik + 1, iz + 1, f));
    out3[f] = (R(1) - fk) * ((R(1) - fz) * t00 + fz * t01) + fk * ((R(1) - fz) * t10 + fz * t11);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Drivers
// ---------------------------------------------------------------------------------------------------------
template <class R>
static int orbit_z_impl(const double* times, int64_t n_t, int64_t t_stride_pv, const double* params, int64_t n_pv,
                        int n_pb, int n_ss, double t_exp, double* z_out, int solver = SOLVER_EXACT) {
  if (!times || !params || !z_out) return 1;
  if (n_t <= 0 || n_pv <= 0 || n_pb < 1 || n_ss < 1) return 2;
  const int64_t row = 6 + 3 * (int64_t)n_pb;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t pv = 0; pv < n_pv; ++pv) {
    const double* pr = params + pv * row;
    const double* tt = times + pv * t_stride_pv;
    double* zo = z_out + pv * n_t * n_ss;
    if (!row_is_valid(pr, n_pb)) {
      for (int64_t j = 0; j < n_t * n_ss; ++j) zo[j] = std::numeric_limits<double>::quiet_NaN();
      continue;
    }
    Orbit<R> orb(pr);
    const int sv = dispatch_solver(solver, pr[4]);
    for (int64_t j = 0; j < n_t; ++j)
      for (int s = 0; s < n_ss; ++s) {
        double ts = subsample_time(tt[j], t_exp, s, n_ss);
        zo[j * n_ss + s] = (double)orb.z_signed_solver(fold_phase(ts, pr[0], pr[1]), sv);
      }
  }
  return 0;
}

// mode 0: exact; mode 1: interpolated from `tb`.  Rows whose mean k lies outside the table are evaluated exactly
// (R13).  flux_out[n_pv][n_pb][n_t] as double.
template <class R>
static int flux_impl(int mode, const TableView* tb, const double* times, int64_t n_t, int64_t t_stride_pv,
                     const double* params, int64_t n_pv, int n_pb, int n_ss, double t_exp, double* flux_out) {
  if (!times || !params || !flux_out) return 1;
  if (n_t <= 0 || n_pv <= 0 || n_pb < 1 || n_ss < 1) return 2;
  const int64_t row = 6 + 3 * (int64_t)n_pb;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t pv = 0; pv < n_pv; ++pv) {
    const double* pr = params + pv * row;
    const double* tt = times + pv * t_stride_pv;
    double* fo = flux_out + pv * n_pb * n_t;
    if (!row_is_valid(pr, n_pb)) {
      for (int64_t j = 0; j < n_pb * n_t; ++j) fo[j] = std::numeric_limits<double>::quiet_NaN();
      continue;
    }
    Orbit<R> orb(pr);
    Passbands<R> pb(pr, n_pb);
    bool use_table = false;
    if (mode == 1) {
      double kh = (double)pb.khat;
      use_table = (kh >= tb->k_min) && (kh <= tb->k_min + (tb->n_k - 1) * tb->dk);
    }
    std::vector<R> acc(n_pb);
    for (int64_t j = 0; j < n_t; ++j) {
      for (int q = 0; q < n_pb; ++q) acc[q] = R(0);
      for (int s = 0; s < n_ss; ++s) {
        double ts = subsample_time(tt[j], t_exp, s, n_ss);
        R zs = orb.z_signed(fold_phase(ts, pr[0], pr[1]));
        R b3[3] = {R(0), R(0), R(0)};
        if (zs >= R(0) && zs < R(1) + pb.khat) {  // in front of the star and overlapping (else F = 1, R6)
          if (use_table) interp_basis<R>(*tb, pb.khat, zs, b3);
          else ma_basis<R>(pb.khat, zs, &b3[0], &b3[1], &b3[2]);
        }
        for (int q = 0; q < n_pb; ++q) acc[q] += pb.flux(q, b3[0], b3[1], b3[2]);
      }
      for (int q = 0; q < n_pb; ++q) fo[(int64_t)q * n_t + j] = (double)(acc[q] / R(n_ss));
    }
  }
  return 0;
}

template <class R>
static int table_build_impl(double k_min, double k_max, int n_k, double z_max, int n_z, int dtype, int n_fn, void* table) {
  if (!table) return 1;
  if (n_k < 2 || n_z < 2 || (n_fn != 3 && n_fn != 4) || !(k_max > k_min) || !(z_max > 0.0) || !(k_min >= 0.0)) return 2;
  if (dtype != 0 && dtype != 1) return 3;
  const double dk = (k_max - k_min) / (n_k - 1), dz = z_max / (n_z - 1);
#pragma omp parallel for schedule(dynamic, 1)
  for (int i = 0; i < n_k; ++i) {
    double kd = i * dk; kd = k_min + kd;  // mul then add (no FMA: -ffp-contract=off)
    for (int j = 0; j < n_z; ++j) {
      double zd = j * dz;
      R v[4] = {R(0), R(0), R(0), R(0)};
      ma_basis<R>(R(kd), R(zd), &v[0], &v[1], &v[2]);
      size_t o = ((size_t)i * n_z + j) * n_fn;
      for (int f = 0; f < n_fn; ++f) {
        if (dtype == 0) ((double*)table)[o + f] = (double)v[f];
        else ((float*)table)[o + f] = (float)(double)v[f];
      }
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------------
// The Giménez model (Eq. 1-12), written out as printed.
//   f(k,z) = 1 - α(k,z),   α = Σ_{n=0}^{N} C_n α_n(b,c),   b = k/(1+k), c = z/(1+k)                     Eq. 1, 2
//   α_n(b,c) = b² (1-c²)^{ν+1} / (ν Γ(ν+1)) Σ_{j=0}^{N_J} (-1)^j (2j+ν+2) Γ(ν+j+1)/Γ(j+2)
//              G_j(ν+2, ν+1; 1-b)² G_j(ν+2, 1; c²),   ν = (n+2)/2                                       Eq. 3
//   C_0 = (1 - Σ u_n) / (1 - Σ n u_n/(n+2)),  C_n = u_n / (1 - Σ n u_n/(n+2))                           Eq. 7, 8
//   limb darkening I(μ)/I(1) = 1 - Σ_{n=1}^{N} u_n (1 - μ^n)                                            Eq. 4
// The paper names G_n(p,q;x) "Jacobi polynomials" without defining them; R20: they are Kopal's (1977), the
// polynomials of the series the model comes from: G_j(p,q;x) = 2F1(-j, j+p; q; x) = Σ_m (-j)_m (j+p)_m / ((q)_m m!) x^m.
// With this reading Eq. 3 converges, as N_J grows, to α_n = (1/π) ∫_occulted μ^n dA — the definition that follows from Eq. 4,
// 7, 8 alone (checked in tests/test_oracle_pins.py against 30-digit quadrature).  Here the polynomial is its defining
// finite sum, term by term (an alternating sum: use the __float128 instantiation beyond j ~ 25).
// The defining sum Σ_m (-j)_m (j+p)_m / ((q)_m m!) x^m alternates with terms up to ~1e40 at j = 60 (beyond even __float128), so
// the same polynomial is evaluated through its other textbook closed form, the two-binomial sum of the Jacobi polynomial it
// is a multiple of (e.g. Szegő, Orthogonal Polynomials, eq. 4.3.2):
//   G_j(p,q;x) = j! Γ(q)/Γ(j+q) P_j^{(q-1, p-q)}(1-2x),   P_j^{(α,β)}(1-2x) = Σ_s C(j+α, j-s) C(j+β, s) (-x)^s (1-x)^{j-s},
// whose terms stay below ~1e16 for x in [0,1] and j <= 60 (C(a,m) = Γ(a+1)/(Γ(m+1)Γ(a-m+1))).  tests/test_oracle_pins.py
// checks it against mpmath's 2F1 and against the defining sum for small j.
template <class R> static R gen_binom(R a, int m) { return x_tgamma(a + R(1)) / (x_tgamma(R(m + 1)) * x_tgamma(a - R(m) + R(1))); }
template <class R> static R kopal_G(int j, R p, R q, R x) {
  const R al = q - R(1), be = p - q;
  R sum = R(0);
  for (int s = 0; s <= j; ++s) {
    R t = gen_binom<R>(R(j) + al, j - s) * gen_binom<R>(R(j) + be, s) * x_pow(x, R(s)) * x_pow(R(1) - x, R(j - s));
    sum += (s & 1) ? -t : t;
  }
  return x_tgamma(R(j + 1)) * x_tgamma(q) / x_tgamma(R(j) + q) * sum;
}
template <class R> static R kopal_G_defining_sum(int j, R p, R q, R x) {
  R sum = R(1), term = R(1);
  for (int m = 0; m < j; ++m) {
    term *= R(m - j) * (R(j) + p + R(m)) / ((q + R(m)) * R(m + 1)) * x;
    sum += term;
  }
  return sum;
}
template <class R> static R gimenez_alpha_n(int n, int n_j, R k, R z) {
  if (!(z < R(1) + k) || !(k > R(0))) return R(0);
  const R b = k / (R(1) + k), c = z / (R(1) + k);
  const R nu = R(n + 2) / R(2);
  R s = R(0);
  for (int j = 0; j <= n_j; ++j) {
    const R g1 = kopal_G<R>(j, nu + R(2), nu + R(1), R(1) - b);
    const R g2 = kopal_G<R>(j, nu + R(2), R(1), c * c);
    const R a = R((j & 1) ? -1 : 1) * (R(2 * j) + nu + R(2)) * x_tgamma(nu + R(j + 1)) / x_tgamma(R(j + 2));
    s += a * g1 * g1 * g2;
  }
  return b * b * x_pow(R(1) - c * c, nu + R(1)) / (nu * x_tgamma(nu + R(1))) * s;
}
// Row layout of the Giménez entry points: [t0, P, a/R*, i, e, w, k,  u_1..u_N (passband 0), u_1..u_N (passband 1), ...].
static bool gimenez_row_is_valid(const double* pr, int n_pb, int n_ldc) {
  for (int j = 0; j < 7 + n_pb * n_ldc; ++j) if (!std::isfinite(pr[j])) return false;
  if (!(pr[1] > 0.0) || !(pr[2] > 0.0) || !(pr[4] >= 0.0 && pr[4] < 1.0) || !(pr[6] >= 0.0)) return false;
  for (int q = 0; q < n_pb; ++q) {
    double den = 1.0;
    for (int n = 1; n <= n_ldc; ++n) den -= n * pr[7 + q * n_ldc + n - 1] / (n + 2.0);
    if (den == 0.0) return false;
  }
  return true;
}
template <class R>
static int gimenez_exact_impl(const double* times, int64_t n_t, int64_t t_stride_pv, const double* params, int64_t n_pv,
                              int n_pb, int n_ldc, int n_j, int n_ss, double t_exp, double* flux_out) {
  if (!times || !params || !flux_out) return 1;
  if (n_t <= 0 || n_pv <= 0 || n_pb < 1 || n_ss < 1 || n_ldc < 1 || n_j < 0) return 2;
  const int64_t row = 7 + (int64_t)n_pb * n_ldc;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t pv = 0; pv < n_pv; ++pv) {
    const double* pr = params + pv * row;
    const double* tt = times + pv * t_stride_pv;
    double* fo = flux_out + pv * n_pb * n_t;
    if (!gimenez_row_is_valid(pr, n_pb, n_ldc)) {
      for (int64_t j = 0; j < n_pb * n_t; ++j) fo[j] = std::numeric_limits<double>::quiet_NaN();
      continue;
    }
    double orow[9] = {pr[0], pr[1], pr[2], pr[3], pr[4], pr[5], pr[6], 0.0, 0.0};
    Orbit<R> orb(orow);
    const R k = R(pr[6]);
    std::vector<R> C((size_t)n_pb * (n_ldc + 1));                      // Eq. 7, 8
    for (int q = 0; q < n_pb; ++q) {
      R su = R(0), den = R(1);
      for (int n = 1; n <= n_ldc; ++n) { const R u = R(pr[7 + q * n_ldc + n - 1]); su += u; den -= R(n) * u / R(n + 2); }
      C[(size_t)q * (n_ldc + 1)] = (R(1) - su) / den;
      for (int n = 1; n <= n_ldc; ++n) C[(size_t)q * (n_ldc + 1) + n] = R(pr[7 + q * n_ldc + n - 1]) / den;
    }
    std::vector<R> acc(n_pb), an(n_ldc + 1);
    for (int64_t j = 0; j < n_t; ++j) {
      for (int q = 0; q < n_pb; ++q) acc[q] = R(0);
      for (int s = 0; s < n_ss; ++s) {
        const double ts = subsample_time(tt[j], t_exp, s, n_ss);
        const R zs = orb.z_signed(fold_phase(ts, pr[0], pr[1]));
        if (zs >= R(0) && zs < R(1) + k && k > R(0)) {
          for (int n = 0; n <= n_ldc; ++n) an[n] = gimenez_alpha_n<R>(n, n_j, k, zs);
          for (int q = 0; q < n_pb; ++q) {
            R al = R(0);
            for (int n = 0; n <= n_ldc; ++n) al += C[(size_t)q * (n_ldc + 1) + n] * an[n];   // Eq. 9
            acc[q] += R(1) - al;
          } 
        } else {
          for (int q = 0; q < n_pb; ++q) acc[q] += R(1);
        }
      }
      for (int q = 0; q < n_pb; ++q) fo[(int64_t)q * n_t + j] = (double)(acc[q] / R(n_ss));
    }
  }
  return 0;
}

extern "C" {

int pto_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void pto_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// basis functions at n (k,z) pairs; prec: 0 = double, 1 = __float128 (result rounded to double)
int pto_ma_basis(int prec, const double* k, const double* z, int64_t n, double* le, double* ld, double* ed) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    if (prec == 0) { double a, b, c; ma_basis<double>(k[i], z[i], &a, &b, &c); le[i] = a; ld[i] = b; ed[i] = c; }
    else { quad a, b, c; ma_basis<quad>(quad(k[i]), quad(z[i]), &a, &b, &c); le[i] = (double)a; ld[i] = (double)b; ed[i] = (double)c; }
  }
  return 0;
}

// K(m), E(m), Π(n|m) at n_pts points (pins the Carlson forms)
int pto_ellip(int prec, const double* m, const double* n, int64_t n_pts, double* K, double* E, double* Pi) {
  for (int64_t i = 0; i < n_pts; ++i) {
    if (prec == 0) { K[i] = ell_K<double>(m[i]); E[i] = ell_E<double>(m[i]); Pi[i] = ell_Pi<double>(n[i], m[i]); }
    else { K[i] = (double)ell_K<quad>(m[i]); E[i] = (double)ell_E<quad>(m[i]); Pi[i] = (double)ell_Pi<quad>(n[i], m[i]); }
  }
  return 0;
}

// eccentric anomaly for (M, e) pairs (pins the Kepler solve)
int pto_kepler(int prec, const double* M, const double* e, int64_t n, double* E) {
  for (int64_t i = 0; i < n; ++i)
    E[i] = prec == 0 ? kepler_E<double>(M[i], e[i]) : (double)kepler_E<quad>(quad(M[i]), quad(e[i]));
  return 0;
}

int pto_orbit_z(int prec, const double* times, int64_t n_t, int64_t t_stride_pv, const double* params, int64_t n_pv,
                int32_t n_pb, int32_t n_ss, double t_exp, double* z_out) {
  return prec == 0 ? orbit_z_impl<double>(times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, z_out)
                   : orbit_z_impl<quad>(times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, z_out);
}

int pto_orbit_z_solver(int prec, int solver, const double* times, int64_t n_t, int64_t t_stride_pv, const double* params,
                        int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, double* z_out) {
  if (solver < SOLVER_EXACT || solver > SOLVER_FAST) return 3;
  return prec == 0 ? orbit_z_impl<double>(times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, z_out, solver)
                   : orbit_z_impl<quad>(times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, z_out, solver);
}

// E(M) by the fixed-point iteration and the true anomaly by the two series, on their own (tests/test_oracle_pins.py).
int pto_kepler_iter(int prec, const double* M, const double* e, int64_t n, double* E) {
  for (int64_t i = 0; i < n; ++i)
    E[i] = prec == 0 ? kepler_E_iteration<double>(M[i], e[i]) : (double)kepler_E_iteration<quad>(quad(M[i]), quad(e[i]));
  return 0;
}
int pto_true_anomaly_series(int prec, int order, const double* M, const double* e, int64_t n, double* f) {
  if (order != 3 && order != 5) return 3;
  for (int64_t i = 0; i < n; ++i)
    f[i] = prec == 0 ? true_anomaly_series<double>(M[i], e[i], order) : (double)true_anomaly_series<quad>(quad(M[i]), quad(e[i]), order);
  return 0;
}

int pto_gimenez_alpha(int prec, int n, int n_j, const double* k, const double* z, int64_t n_pts, double* out) {
  for (int64_t i = 0; i < n_pts; ++i)
    out[i] = prec == 0 ? gimenez_alpha_n<double>(n, n_j, k[i], z[i]) : (double)gimenez_alpha_n<quad>(n, n_j, quad(k[i]), quad(z[i]));
  return 0;
}
int pto_kopal_G(int prec, int j, double p, double q, const double* x, int64_t n_pts, double* out) {
  for (int64_t i = 0; i < n_pts; ++i)
    out[i] = prec == 0 ? kopal_G<double>(j, p, q, x[i]) : (prec == 1 ? (double)kopal_G<quad>(j, quad(p), quad(q), quad(x[i]))
                                                                     : (double)kopal_G_defining_sum<quad>(j, quad(p), quad(q), quad(x[i])));
  return 0;
}
int pto_gimenez_exact(int prec, const double* times, int64_t n_t, int64_t t_stride_pv, const double* params, int64_t n_pv,
                      int32_t n_pb, int32_t n_ldc, int32_t n_j, int32_t n_ss, double t_exp, double* flux_out) {
  return prec == 0 ? gimenez_exact_impl<double>(times, n_t, t_stride_pv, params, n_pv, n_pb, n_ldc, n_j, n_ss, t_exp, flux_out)
                   : gimenez_exact_impl<quad>(times, n_t, t_stride_pv, params, n_pv, n_pb, n_ldc, n_j, n_ss, t_exp, flux_out);
}

int pto_ma_quad_exact(int prec, const double* times, int64_t n_t, int64_t t_stride_pv, const double* params,
                      int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, double* flux_out) {
  return prec == 0
             ? flux_impl<double>(0, nullptr, times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, flux_out)
             : flux_impl<quad>(0, nullptr, times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, flux_out);
}

int pto_ma_table_build(int prec, double k_min, double k_max, int32_t n_k, double z_max, int32_t n_z, int32_t dtype,
                       int32_t n_fn, void* table) {
  return prec == 0 ? table_build_impl<double>(k_min, k_max, n_k, z_max, n_z, dtype, n_fn, table)
                   : table_build_impl<quad>(k_min, k_max, n_k, z_max, n_z, dtype, n_fn, table);
}

int pto_ma_quad_interp(int prec, const void* table, int32_t table_dtype, int32_t n_k, int32_t n_z, int32_t n_fn,
                       double k_min, double dk, double dz, const double* times, int64_t n_t, int64_t t_stride_pv,
                       const double* params, int64_t n_pv, int32_t n_pb, int32_t n_ss, double t_exp, double* flux_out) {
  if (!table) return 1;
  if (n_k < 2 || n_z < 2 || (n_fn != 3 && n_fn != 4) || !(dk > 0.0) || !(dz > 0.0)) return 4;
  TableView tb{table, table_dtype, n_k, n_z, n_fn, k_min, dk, dz};
  return prec == 0 ? flux_impl<double>(1, &tb, times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, flux_out)
                   : flux_impl<quad>(1, &tb, times, n_t, t_stride_pv, params, n_pv, n_pb, n_ss, t_exp, flux_out);
}

// bilinear rule alone at n (k,z) pairs (pins the cell choice and the clamps of interp_basis); out[n][3]
int pto_interp_basis(int prec, const void* table, int32_t table_dtype, int32_t n_k, int32_t n_z, int32_t n_fn, double k_min,
                     double dk, double dz, const double* k, const double* z, int64_t n, double* out) {
  if (!table || !k || !z || !out) return 1;
  if (n_k < 2 || n_z < 2 || (n_fn != 3 && n_fn != 4) || !(dk > 0.0) || !(dz > 0.0)) return 4;
  TableView tb{table, table_dtype, n_k, n_z, n_fn, k_min, dk, dz};
  for (int64_t i = 0; i < n; ++i) {
    if (prec == 0) { double v[3]; interp_basis<double>(tb, k[i], z[i], v); for (int f = 0; f < 3; ++f) out[3 * i + f] = v[f]; }
    else { quad v[3]; interp_basis<quad>(tb, quad(k[i]), quad(z[i]), v); for (int f = 0; f < 3; ++f) out[3 * i + f] = (double)v[f]; }
  }
  return 0;
}

}  // extern "C"
