"""Generator of the polynomial coefficients in pt_math.cuh (kernel side only; the oracle uses libm/libquadmath).

    python paper_1504_07433_b200/csrc/gen_poly.py

atan(t) = t + t u P(u), u = t², |t| <= tan(π/8): P is the degree-10 polynomial obtained from the degree-11 interpolant of
atan(√u)/√u at the Chebyshev nodes of [0, tan²(π/8)] (near-minimax; max error 4e-18 with double-rounded coefficients),
computed with mpmath at 60 digits.  The interpolant's constant term is 1 - 1.3e-18 and is replaced by exactly 1.
sin/cos use plain Taylor coefficients ±1/n! (|r| <= π/4: truncation < 5e-17).
"""
import mpmath as mp

mp.mp.dps = 60


def atan_coeffs(n_terms=12):
    a = mp.tan(mp.pi / 8) ** 2

    def f(u):
        if u == 0:
            return mp.mpf(1)
        t = mp.sqrt(u)
        return mp.atan(t) / t

    xs = [(a / 2) * (1 + mp.cos(mp.pi * (2 * k + 1) / (2 * n_terms))) for k in range(n_terms)]
    A = mp.matrix(n_terms, n_terms)
    for i, x in enumerate(xs):
        for j in range(n_terms):
            A[i, j] = x ** j
    return list(mp.lu_solve(A, mp.matrix([f(x) for x in xs])))


if __name__ == "__main__":
    c = atan_coeffs()
    print("// atan: P(u) coefficients, highest power first (u^10 ... u^0 of P; c[j+1] of the interpolant)")
    for j in range(len(c) - 1, 0, -1):
        print("  %s," % mp.nstr(c[j], 20))
    print("// sin: -1/3!, 1/5!, ... ; cos: 1/4!, -1/6!, ...")
    for k in (15, 13, 11, 9, 7, 5, 3):
        print("  %s,  // sin 1/%d!" % (mp.nstr((-1) ** ((k - 1) // 2) / mp.factorial(k), 20), k))
    for k in (16, 14, 12, 10, 8, 6, 4):
        print("  %s,  // cos 1/%d!" % (mp.nstr((-1) ** (k // 2) / mp.factorial(k), 20), k))
