"""Writes the stored expected values under tests/golden/ — calls ONLY oracle/ma_definition.py (+ mpmath).

    python tests/golden/make_golden.py

ma_basis_definition.txt : λe, λd, ηd from their integral definitions (Eq. 6 + Eq. 13 of PAPER.md) by
                          30-digit tanh-sinh quadrature, at (k, z) pairs covering every region of the Mandel–Agol case
                          split, incl. points 1e-6 / 1e-9 from each boundary.  k and z are the IEEE doubles printed.
config1_worked.txt      : BASELINE.json configs[0] (t0=0, P=3 d, a/R*=8, i=88 deg, k=0.1, u=(0.4,0.2), circular):
                          z(t) from the circular-orbit projection and the flux from Eq. 13 with the quadrature values.
Nothing here touches oracle/pt_oracle.cpp or the CUDA path; the files pin both.
"""
import os
import sys

import mpmath as mp

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))
from oracle.ma_definition import basis_mp  # noqa: E402

PAIRS = [
    (0.1, 0.0), (0.1, 0.05), (0.1, 0.1), (0.1, 0.5), (0.1, 0.95), (0.1, 1.05), (0.2, 0.85), (0.25, 0.75), (0.3, 0.3),
    (0.5, 0.25), (0.5, 0.5), (0.7, 0.5), (0.7, 0.7), (0.75, 0.25), (1.5, 1.0),
    # near the case boundaries (z = k, 1-k, 1+k, 0) and near k = 1/2
    (0.1, 0.1 + 1e-6), (0.1, 0.1 - 1e-6), (0.1, 0.1 + 1e-9), (0.1, 0.9 + 1e-6), (0.1, 0.9 - 1e-6), (0.1, 0.9 - 1e-9),
    (0.1, 1.1 - 1e-6), (0.1, 1.1 - 1e-9), (0.1, 1e-6), (0.1, 1e-9), (0.01, 0.99 - 1e-6), (0.01, 0.99 + 1e-6),
    (0.5 + 1e-6, 0.5), (0.5 - 1e-6, 0.5), (0.5 + 1e-9, 0.5 - 1e-9), (0.45, 0.45), (0.45, 0.55), (0.45, 0.55 + 1e-7),
    (0.3, 0.7), (0.3, 1.2999), (0.05, 1.0), (0.2, 1.0), (0.4, 0.6), (0.6, 0.4), (0.6, 0.4 + 1e-7), (0.6, 0.6 - 1e-7),
    # k >= 1
    (1.0, 0.5), (1.2, 0.1), (1.2, 0.5), (1.5, 0.3), (2.0, 1.5), (2.0, 2.9),
    (0.0123456789, 0.3), (0.33, 0.0), (0.9, 0.05), (0.9, 0.1), (0.9, 1.5),
]


def main():
    mp.mp.dps = 40
    with open(os.path.join(HERE, "ma_basis_definition.txt"), "w") as f:
        f.write("# k z lambda_e lambda_d eta_d   (integral definitions, P:L86 Eq.6 + P:L136 Eq.13; 30-digit quadrature)\n")
        for k, z in PAIRS:
            le, ld, ed = basis_mp(k, z, dps=30)
            f.write("%r %r %s %s %s\n" % (k, z, mp.nstr(le, 25), mp.nstr(ld, 25), mp.nstr(ed, 25)))
    # config 1 worked example
    t0, P, a, inc, k, u1, u2 = 0.0, 3.0, 8.0, 88.0 * 3.141592653589793 / 180.0, 0.1, 0.4, 0.2
    times = [0.0, 0.01, 0.03, 0.05, 0.055, 0.06, 0.0625, 0.064, 0.1, 0.15, -0.03, -0.06]
    with open(os.path.join(HERE, "config1_worked.txt"), "w") as f:
        f.write("# t z flux   (BASELINE.json configs[0]; circular projection + Eq. 13 with quadrature values)\n")
        for t in times:
            x = (t - t0) / P          # IEEE double, as both implementations fold the phase (H1)
            ph = x - round(x)
            phi = 2 * mp.pi * mp.mpf(ph)
            ci = mp.cos(mp.mpf(inc))
            z = mp.mpf(a) * mp.sqrt(mp.sin(phi) ** 2 + ci ** 2 * mp.cos(phi) ** 2)
            zf = float(z)
            if z >= 1 + mp.mpf(k):
                flux = mp.mpf(1)
            else:
                le, ld, ed = basis_mp(mp.mpf(k), z, dps=30)
                c = mp.mpf(u1) + 2 * mp.mpf(u2)
                flux = 1 - ((1 - c) * le + c * ld + mp.mpf(u2) * ed) / (1 - mp.mpf(u1) / 3 - mp.mpf(u2) / 6)
            f.write("%r %s %s\n" % (t, mp.nstr(z, 20), mp.nstr(flux, 20)))


if __name__ == "__main__":
    main()
