"""Seeded synthetic workloads for the five BASELINE.json configs (shapes, cadences and priors only).

This module serves BOTH the CUDA path (tests, bench.py) and the CPU oracle (tests) and therefore holds none of the
method's arithmetic: no limb darkening, no basis functions, no orbit solve, no interpolation.  Where a generator
needs projected separations (config 5 aims 30 % of its times at the case boundaries) the caller passes an `orbit_z`
callable in; tests pass the oracle's.  The paper measures on synthetic light curves (35 % in transit) and
BASELINE.json names Kepler long cadence / spectrophotometry only as shapes, so these stand in for those workloads
(DESIGN.md §4 states the full recipe).

Random draws: numpy.random.Generator(PCG64(SEED0 + config [+ 1000*stream])), one vector per named quantity, in the
order written below, float64.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np

SEED0 = 15040743300
LC_CADENCE = 29.4 / 1440.0  # Kepler long cadence, days


@dataclass
class Workload:
    name: str
    times: np.ndarray            # [n_t] shared, or [n_pv][n_t] per parameter vector
    params: np.ndarray           # [n_pv][6 + 3 n_pb] = t0, P, a/R*, i, e, w, (k, u1, u2) per passband
    n_pb: int = 1
    n_ss: int = 1
    t_exp: float = 0.0
    table: Optional[dict] = None  # config 4: k_min, k_max, n_k, z_max, n_z
    meta: dict = field(default_factory=dict)

    @property
    def n_pv(self) -> int:
        return self.params.shape[0]

    @property
    def n_t(self) -> int:
        return self.times.shape[-1]

    @property
    def n_eval(self) -> int:
        """z-evaluations (supersamples counted)."""
        return self.n_pv * self.n_t * self.n_ss


def _rng(config: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED0 + config + 1000 * stream))


def kipping_to_quadratic(q1, q2):
    """Kipping's triangular sampling (named in BASELINE.json configs[1]): (q1,q2) in [0,1]² -> (u1,u2)."""
    sq = np.sqrt(q1)
    return 2.0 * sq * q2, sq * (1.0 - 2.0 * q2)


def config1() -> Workload:
    """1 parameter set, circular, 1000 times uniform on [-0.15, 0.15] d (BASELINE.json configs[0])."""
    params = np.array([[0.0, 3.0, 8.0, 88.0 * np.pi / 180.0, 0.0, 0.0, 0.1, 0.4, 0.2]])
    j = np.arange(1000, dtype=np.float64)
    times = -0.15 + 0.3 * j / 999.0
    return Workload("config1", times, params)


def _population_cfg2(rng: np.random.Generator, n_pv: int) -> np.ndarray:
    P = rng.uniform(1.0, 10.0, n_pv)
    t0 = P * rng.uniform(0.0, 1.0, n_pv)
    k = rng.uniform(0.05, 0.2, n_pv)
    b = rng.uniform(0.0, 0.9, n_pv)
    a = rng.uniform(5.0, 20.0, n_pv)
    q1 = rng.uniform(0.0, 1.0, n_pv)
    q2 = rng.uniform(0.0, 1.0, n_pv)
    u1, u2 = kipping_to_quadratic(q1, q2)
    inc = np.arccos(b / a)
    z = np.zeros(n_pv)
    return np.stack([t0, P, a, inc, z, z, k, u1, u2], axis=1)


def config2(n_pv: int = 64, n_t: int = 60000, stream: int = 0) -> Workload:
    """Kepler long-cadence-like: 29.4-min cadence, 10 supersamples, circular orbits (BASELINE.json configs[1])."""
    rng = _rng(2, stream)
    start = rng.uniform(0.0, 10.0)
    times = start + np.arange(n_t, dtype=np.float64) * LC_CADENCE
    params = _population_cfg2(rng, n_pv)
    return Workload("config2", times, params, n_pb=1, n_ss=10, t_exp=LC_CADENCE, meta={"start": start})


def config3(n_pv: int = 512, n_pb: int = 20, n_t: int = 600, stream: int = 0) -> Workload:
    """Spectrophotometric multi-passband: 20 passbands x 600 exposures on [-0.12, 0.12] d (BASELINE.json configs[2])."""
    rng = _rng(3, stream)
    t0 = rng.normal(0.0, 1e-3, n_pv)
    P = np.full(n_pv, 2.5)
    a = rng.uniform(6.0, 12.0, n_pv)
    b = rng.uniform(0.0, 0.8, n_pv)
    k = rng.normal(0.12, 0.005, (n_pv, n_pb))
    q1 = rng.uniform(0.0, 1.0, (n_pv, n_pb))
    q2 = rng.uniform(0.0, 1.0, (n_pv, n_pb))
    u1, u2 = kipping_to_quadratic(q1, q2)
    inc = np.arccos(b / a)
    z = np.zeros(n_pv)
    head = np.stack([t0, P, a, inc, z, z], axis=1)
    tail = np.stack([k, u1, u2], axis=2).reshape(n_pv, 3 * n_pb)
    params = np.concatenate([head, tail], axis=1)
    # a single exposure sits at mid-transit (0/0 otherwise)
    times = -0.12 + 0.24 * np.arange(n_t, dtype=np.float64) / (n_t - 1) if n_t > 1 else np.zeros(1)
    return Workload("config3", times, params, n_pb=n_pb)


def config4(n_pv: int = 4096, n_t: int = 100000, stream: int = 0) -> Workload:
    """Interpolated path: table k in [0.05,0.25] step 5e-4, z in [0,1.25] step 1e-4; population as config 2, n_ss = 1."""
    rng = _rng(4, stream)
    start = rng.uniform(0.0, 10.0)
    times = start + np.arange(n_t, dtype=np.float64) * LC_CADENCE
    params = _population_cfg2(rng, n_pv)
    table = dict(k_min=0.05, k_max=0.25, n_k=401, z_max=1.25, n_z=12501)
    return Workload("config4", times, params, table=table, meta={"start": start})


def transit_duration_t14(P, a, inc, e, w, k):
    """Approximate first-to-fourth-contact duration, used only to place config 5's time windows."""
    fac = (1.0 - e * e) / (1.0 + e * np.sin(w))
    b = a * np.cos(inc) * fac
    arg = np.sqrt(np.clip((1.0 + k) ** 2 - b * b, 0.0, None)) / (a * np.sin(inc))
    return P / np.pi * np.arcsin(np.clip(arg, 0.0, 1.0)) * fac / np.sqrt(1.0 - e * e)


def config5(orbit_z: Callable[[np.ndarray, np.ndarray], np.ndarray], n_pv: int = 4096, n_t: int = 4096,
            order: str = "sorted", stream: int = 0) -> Workload:
    """Edge-case and eccentric stress (BASELINE.json configs[4]); per-pv times.

    orbit_z(times[n_pv][m], params[n_pv][9]) -> signed z[n_pv][m] is supplied by the caller (the oracle's, in tests).
    order: "sorted" (times ascending per pv) or "shuffled" (a seeded permutation: divergence stress).
    """
    rng = _rng(5, stream)
    P = rng.uniform(1.0, 10.0, n_pv)
    t0 = P * rng.uniform(0.0, 1.0, n_pv)
    a = rng.uniform(5.0, 20.0, n_pv)
    e = rng.uniform(0.0, 0.6, n_pv)
    w = rng.uniform(0.0, 2.0 * np.pi, n_pv)
    q1 = rng.uniform(0.0, 1.0, n_pv)
    q2 = rng.uniform(0.0, 1.0, n_pv)
    u1, u2 = kipping_to_quadratic(q1, q2)
    # groups: 1/2 generic, 1/4 grazing, 1/8 central (b = 0 exactly), 1/8 k within 1e-6 of 0.5
    grp = np.zeros(n_pv, dtype=np.int64)
    n2, n4, n8 = n_pv // 2, n_pv // 4, n_pv // 8
    grp[n2:n2 + n4] = 1
    grp[n2 + n4:n2 + n4 + n8] = 2
    grp[n2 + n4 + n8:] = 3
    k = rng.uniform(0.01, 0.5, n_pv)
    b = rng.uniform(0.0, 0.8, n_pv)
    b_graze = rng.uniform(0.8, 1.2, n_pv)
    k_half = 0.5 + rng.uniform(-1e-6, 1e-6, n_pv)
    b_half = rng.uniform(0.0, 0.4, n_pv)
    b = np.where(grp == 1, b_graze, b)
    b = np.where(grp == 2, 0.0, b)
    b = np.where(grp == 3, b_half, b)
    k = np.where(grp == 3, k_half, k)
    idx3 = np.flatnonzero(grp == 3)
    k[idx3[: max(1, len(idx3) // 8)]] = 0.5  # some exactly 0.5
    cosi = b * (1.0 + e * np.sin(w)) / (a * (1.0 - e * e))
    inc = np.where(grp == 2, np.pi / 2.0, np.arccos(np.clip(cosi, -1.0, 1.0)))
    params = np.stack([t0, P, a, inc, e, w, k, u1, u2], axis=1)

    t14 = transit_duration_t14(P, a, inc, e, w, k)
    t14 = np.where(t14 > 0, t14, 0.02 * P)  # non-transiting grazers still get a window
    half = 0.75 * t14
    n_uni = int(round(0.7 * n_t))
    n_tgt = n_t - n_uni
    t_uni = t0[:, None] + half[:, None] * rng.uniform(-1.0, 1.0, (n_pv, n_uni))

    # boundary-targeted times: z(t) = |z* + delta|, z* in {0, k, 1-k, 1+k}, on the ingress (side=-1) or egress (+1)
    delta = rng.uniform(-1e-6, 1e-6, (n_pv, n_tgt))
    side = np.where(rng.uniform(0.0, 1.0, (n_pv, n_tgt)) < 0.5, -1.0, 1.0)
    prio = rng.uniform(0.0, 1.0, (4, n_pv, n_tgt))
    # bracket: [mid-transit, edge of the window] on the chosen side; z grows away from mid-transit
    t_in = np.broadcast_to(t0[:, None], delta.shape).copy()
    t_out = t0[:, None] + side * 1.2 * half[:, None]
    z_in = np.abs(orbit_z(t_in, params))
    z_out = np.abs(orbit_z(t_out, params))
    kk = k[:, None]
    cand = np.stack([np.abs(0.0 + delta), np.abs(kk + delta), np.abs(1.0 - kk + delta), np.abs(1.0 + kk + delta)])
    reach = (cand > z_in[None]) & (cand < z_out[None])          # z* reachable on this chord and side
    which = np.argmax(np.where(reach, prio, -1.0), axis=0)      # a random reachable boundary
    ztgt = np.take_along_axis(cand, which[None], axis=0)[0]
    ok = np.take_along_axis(reach, which[None], axis=0)[0]
    # Illinois-type bracketed secant on g(t) = z(t) - ztgt (monotone on the branch): g(t_in) < 0 < g(t_out)
    g_in, g_out = z_in - ztgt, z_out - ztgt
    t_best = 0.5 * (t_in + t_out)
    g_best = np.full(ztgt.shape, np.inf)
    last = np.zeros(ztgt.shape, dtype=np.int8)  # which end moved last: -1 inner, +1 outer
    for _ in range(60):
        denom = np.where(g_out - g_in != 0, g_out - g_in, 1.0)
        t_new = t_out - g_out * (t_out - t_in) / denom
        bad = ~np.isfinite(t_new) | ((t_new - t_in) * (t_new - t_out) > 0)
        t_new = np.where(bad | ~ok, 0.5 * (t_in + t_out), t_new)
        g_new = np.abs(orbit_z(t_new, params)) - ztgt
        better = np.abs(g_new) < g_best
        t_best = np.where(better, t_new, t_best)
        g_best = np.where(better, np.abs(g_new), g_best)
        inner = g_new < 0
        g_out = np.where(inner, np.where(last == -1, 0.5 * g_out, g_out), g_new)
        g_in = np.where(inner, g_new, np.where(last == 1, 0.5 * g_in, g_in))
        t_in = np.where(inner, t_new, t_in)
        t_out = np.where(inner, t_out, t_new)
        last = np.where(inner, -1, 1).astype(np.int8)
        if np.all(~ok | (g_best < 1e-9)):
            break
    # unreachable targets (grazing chords, z* below the impact parameter) fall back to uniform-in-window times
    t_fallback = t0[:, None] + half[:, None] * rng.uniform(-1.0, 1.0, (n_pv, n_tgt))
    t_tgt = np.where(ok, t_best, t_fallback)

    times = np.concatenate([t_uni, t_tgt], axis=1)
    if order == "sorted":
        times = np.sort(times, axis=1)
    elif order == "shuffled":
        perm = np.argsort(rng.uniform(0.0, 1.0, times.shape), axis=1)
        times = np.take_along_axis(times, perm, axis=1)
    else:
        raise ValueError(order)
    meta = {"groups": grp, "targeted_fraction": float(np.mean(ok)) * n_tgt / n_t}
    return Workload("config5", np.ascontiguousarray(times), params, meta=meta)


def dense_transit(n_pv: int = 4096, n_t: int = 4096, eccentric: bool = True, stream: int = 0) -> Workload:
    """Config-5-like population with every time inside t0 ± 0.75 T14 (no boundary targeting, so no orbit callable is
    needed): the FP64-bound bench workload."""
    rng = _rng(6, stream)
    P = rng.uniform(1.0, 10.0, n_pv)
    t0 = P * rng.uniform(0.0, 1.0, n_pv)
    a = rng.uniform(5.0, 20.0, n_pv)
    e = rng.uniform(0.0, 0.6, n_pv) if eccentric else np.zeros(n_pv)
    w = rng.uniform(0.0, 2.0 * np.pi, n_pv) if eccentric else np.zeros(n_pv)
    q1 = rng.uniform(0.0, 1.0, n_pv)
    q2 = rng.uniform(0.0, 1.0, n_pv)
    u1, u2 = kipping_to_quadratic(q1, q2)
    k = rng.uniform(0.01, 0.5, n_pv)
    b = rng.uniform(0.0, 0.8, n_pv)
    cosi = b * (1.0 + e * np.sin(w)) / (a * (1.0 - e * e))
    inc = np.arccos(np.clip(cosi, -1.0, 1.0))
    params = np.stack([t0, P, a, inc, e, w, k, u1, u2], axis=1)
    half = 0.75 * transit_duration_t14(P, a, inc, e, w, k)
    times = np.sort(t0[:, None] + half[:, None] * rng.uniform(-1.0, 1.0, (n_pv, n_t)), axis=1)
    return Workload("dense_transit", np.ascontiguousarray(times), params)
