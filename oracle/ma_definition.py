"""The plain DEFINITION of the three Mandel–Agol basis functions, by quadrature.  TEST INFRASTRUCTURE.

PAPER.md gives the quadratic limb-darkening law (Eq. 6)  I(mu)/I(1) = 1 - a(1-mu) - b(1-mu)^2, mu = sqrt(1-r^2),
and the flux (Eq. 13)  f = 1 - [(1-c) λe + c λd + b ηd] / (1 - a/3 - b/6), c = a + 2b, but defers λe, λd, ηd to
Mandel & Agol (2002).  Expanding Eq. 6 with mu^2 = 1 - r^2 gives

    I(r) = (1 - c) + c sqrt(1 - r^2) + b r^2 ,       ∫_{r<1} I dA = π (1 - a/3 - b/6)      (the denominator of Eq. 13)

so Eq. 13 is  f = 1 - (∫_occ I dA)/(∫_disk I dA)  and, term by term, with occ = {points of the unit disk within distance k
of the planet centre, itself at distance z from the disk centre}:

    λe(k,z) = (1/π) ∫_occ dA      λd(k,z) = (1/π) ∫_occ sqrt(1-r²) dA      ηd(k,z) = (1/π) ∫_occ r² dA

These integrals are what this module evaluates, three independent ways, none of which shares anything with the closed
forms in oracle/pt_oracle.cpp (which they pin) or with the CUDA path:

  * `basis_mp`     — 1-D tanh-sinh quadrature (mpmath, 30 digits) of ∫ g(r) r φ(r) dr with φ(r) the angle of the arc of
                     radius r that lies inside the planet's disk;  writes tests/golden/ma_basis_definition.txt.
  * `basis_gl2d`   — 2-D tensor Gauss–Legendre quadrature (numpy, fp64) in star-centred polar coordinates (r, θ).
  * `basis_pixels` — brute force: midpoint sum over a Cartesian grid covering the planet's disk (accuracy ~1e-5).
  * `flux_pixels`  — brute-force flux straight from Eq. 6 as printed (no expansion), to catch a wrong weight in Eq. 13.
"""
from __future__ import annotations

import numpy as np


def _arc_angle_mp(mp, r, k, z):
    """Angle (0..2π) of the circle of radius r about the star centre that lies within k of the planet centre."""
    if r <= k - z:
        return 2 * mp.pi
    if r <= z - k or r >= z + k:
        return mp.mpf(0)
    x = (r * r + z * z - k * k) / (2 * r * z)
    x = max(mp.mpf(-1), min(mp.mpf(1), x))
    return 2 * mp.acos(x)


def basis_mp(k, z, dps: int = 30):
    """(λe, λd, ηd) from the integral definitions with mpmath at `dps` digits.  k, z: Python floats (exact doubles)."""
    import mpmath as mp
    mp.mp.dps = dps + 10
    k = mp.mpf(k)
    z = mp.mpf(z)
    lo = max(mp.mpf(0), z - k)
    hi = min(mp.mpf(1), z + k)
    if k == 0 or lo >= hi:
        return mp.mpf(0), mp.mpf(0), mp.mpf(0)
    # panel break points: where the arc becomes a full circle, and the midpoint (tanh-sinh handles the endpoint roots)
    pts = [lo]
    if k > z and lo < k - z < hi:
        pts.append(k - z)
    pts.append(hi)
    full = []
    for a, b in zip(pts[:-1], pts[1:]):
        full += [a, (a + b) / 2]
    full.append(hi)
    out = []
    for g in (lambda r: mp.mpf(1), lambda r: mp.sqrt(max(mp.mpf(0), 1 - r * r)), lambda r: r * r):
        val = mp.quad(lambda r: g(r) * r * _arc_angle_mp(mp, r, k, z), full)
        out.append(val / mp.pi)
    return tuple(out)


def _panels(k, z):
    lo, hi = max(0.0, z - k), min(1.0, z + k)
    if k <= 0 or lo >= hi:
        return []
    pts = [lo]
    if k > z and lo < k - z < hi:
        pts.append(k - z)
    pts.append(hi)
    return list(zip(pts[:-1], pts[1:]))


def basis_gl2d(k: float, z: float, n_r: int = 200, n_th: int = 8):
    """2-D Gauss–Legendre in star-centred polar coordinates: ∫∫ g(r) r dθ dr over the occulted region.

    r-panels are mapped by r = lo + (hi-lo) sin²(πu/2) so the square-root behaviour at the ends becomes smooth.
    """
    xr, wr = np.polynomial.legendre.leggauss(n_r)
    xt, wt = np.polynomial.legendre.leggauss(n_th)
    u = 0.5 * (xr + 1.0)
    wu = 0.5 * wr
    acc = np.zeros(3)
    for lo, hi in _panels(k, z):
        r = lo + (hi - lo) * np.sin(0.5 * np.pi * u) ** 2
        jac = (hi - lo) * np.pi * np.sin(0.5 * np.pi * u) * np.cos(0.5 * np.pi * u)
        # half-opening angle of the arc inside the planet's disk
        with np.errstate(invalid="ignore", divide="ignore"):
            cosang = (r * r + z * z - k * k) / (2.0 * r * z) if z > 0 else np.full_like(r, -1.0)
        half = np.where(r <= k - z, np.pi, np.arccos(np.clip(cosang, -1.0, 1.0)))
        half = np.where((r <= z - k) | (r >= z + k), 0.0, half)
        for f, g in enumerate((np.ones_like(r), np.sqrt(np.clip(1.0 - r * r, 0.0, None)), r * r)):
            # θ-integral over [-half, half] by Gauss–Legendre (the integrand does not depend on θ)
            th_int = np.outer(half, wt).sum(axis=1)
            acc[f] += np.sum(wu * jac * g * r * th_int)
    return tuple(acc / np.pi)


def _pixel_grid(k: float, z: float, n: int):
    h = 2.0 * k / n
    c = -k + h * (np.arange(n) + 0.5)
    x, y = np.meshgrid(z + c, c, indexing="ij")
    r2 = x * x + y * y
    inside = ((x - z) ** 2 + y * y <= k * k) & (r2 <= 1.0)
    return h, r2, inside


def basis_pixels(k: float, z: float, n: int = 2000):
    """Brute force: midpoint sum over an n×n Cartesian grid on the planet's bounding square."""
    if k <= 0:
        return 0.0, 0.0, 0.0
    h, r2, inside = _pixel_grid(k, z, n)
    mu = np.sqrt(np.clip(1.0 - r2, 0.0, None))
    w = h * h / np.pi
    return float(np.sum(inside) * w), float(np.sum(mu[inside]) * w), float(np.sum(r2[inside]) * w)


def flux_pixels(k: float, z: float, a: float, b: float, n: int = 2000):
    """Brute-force relative flux directly from Eq. 6 as printed: 1 - ∫_occ I dA / ∫_disk I dA."""
    if k <= 0:
        return 1.0
    h, r2, inside = _pixel_grid(k, z, n)
    mu = np.sqrt(np.clip(1.0 - r2[inside], 0.0, None))
    inten = 1.0 - a * (1.0 - mu) - b * (1.0 - mu) ** 2
    blocked = float(np.sum(inten) * h * h)
    # unocculted flux of the same law: 2π ∫_0^1 I(mu) mu dmu, by Gauss–Legendre in mu (polynomial => exact)
    x, w = np.polynomial.legendre.leggauss(8)
    m = 0.5 * (x + 1.0)
    total = 2.0 * np.pi * np.sum(0.5 * w * (1.0 - a * (1.0 - m) - b * (1.0 - m) ** 2) * m)
    return 1.0 - blocked / total


def alpha_n_definition(n: int, k: float, z: float):
    """The Giménez basis function by its definition (Eq. 4 with Eq. 7-8: the flux lost to the μ^n term of the limb
    darkening law, in units of π): α_n(k, z) = (1/π) ∫_occulted μ^n dA, μ = sqrt(1 - r²), as a 1-D integral over the
    star-centred radius with the arc of the circle of radius r that lies inside the planet's disk (30-digit tanh-sinh)."""
    import mpmath as mp
    mp.mp.dps = 30
    k, z = mp.mpf(k), mp.mpf(z)
    lo, hi = max(mp.mpf(0), z - k), min(mp.mpf(1), z + k)
    if hi <= lo:
        return mp.mpf(0)

    def arc(r):
        if r <= k - z:
            return 2 * mp.pi
        if r <= z - k or r >= z + k:
            return mp.mpf(0)
        return 2 * mp.acos((r * r + z * z - k * k) / (2 * r * z))

    pts = [lo, hi]
    if k > z and k - z < hi:
        pts = [lo, k - z, hi]
    pts = sorted(set(pts + [(pts[0] + pts[-1]) / 2]))
    return mp.quad(lambda r: (1 - r * r) ** (mp.mpf(n) / 2) * r * arc(r), pts) / mp.pi
