"""Seeded synthetic TESS-shaped light-curve batches (numpy only).

This module is the one thing the CPU oracle's tests and the CUDA path's tests share: it makes
INPUTS.  It holds none of the search arithmetic (no grid, no folding, no SR, no S/N) and imports
neither ``oracle/`` nor the CUDA binding.

The recipes follow BASELINE.json ``configs[0..4]`` (called config 1..5 here)
and stand in for the QLP multi-sector light curves of PAPER.md:7,59 (27.4-d sectors, 30-min /
10-min / 200-s FFI cadence), which are not available offline.  Every star is generated from
``numpy.random.default_rng([seed, config_id, star_id])`` so that any star can be reproduced alone.

Layout returned by :func:`make_batch` (ragged CSR over stars, "determined for each
star"): ``row_ptr`` int64[S+1]; ``t``, ``y``, ``dy`` float64[row_ptr[S]] (days, relative flux,
flux error); ``rho``, ``rstar`` float64[S] in solar units; ``truth`` = per-star injected signal
(period, t0, depth, duration; period 0 = none).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SECTOR_DAYS = 27.4
T_OFFSET = 2000.0             # BTJD-like zero point, days
GAP_LO, GAP_HI = 13.2, 14.2   # sector-relative data gap between the two 13.7-d orbits
CADENCES_S = (200.0, 600.0, 1800.0)

# G * rho_sun * (86400 s/d)^2 in d^-2 (IAU nominal GM_sun, R_sun); used only to give injected
# transits a physically sensible duration.
_K_RHO = 3.0 * 1.3271244e20 / (4.0 * math.pi * 6.957e8 ** 3) * 86400.0 ** 2


@dataclasses.dataclass
class Batch:
    config: int
    seed: int
    star_ids: np.ndarray      # int64[S]
    row_ptr: np.ndarray       # int64[S+1]
    t: np.ndarray             # float64
    y: np.ndarray             # float64
    dy: np.ndarray            # float64
    rho: np.ndarray           # float64[S]
    rstar: np.ndarray         # float64[S]
    truth: np.ndarray         # structured [S]: period, t0, depth, duration

    @property
    def n_stars(self) -> int:
        return int(self.row_ptr.shape[0] - 1)

    @property
    def n_points(self) -> int:
        return int(self.row_ptr[-1])

    def star(self, s: int):
        a, b = int(self.row_ptr[s]), int(self.row_ptr[s + 1])
        return self.t[a:b], self.y[a:b], self.dy[a:b]


TRUTH_DTYPE = np.dtype([("period", "f8"), ("t0", "f8"), ("depth", "f8"), ("duration", "f8")])

N_STARS = {1: 1, 2: 1000, 3: 10000, 4: 1000, 5: 200000}


def sector_times(sector_index: int, cadence_s: float) -> np.ndarray:
    """Timestamps of one sector: samples every cadence from the sector start, mid-sector gap removed."""
    step = cadence_s / 86400.0
    n = int(math.floor(SECTOR_DAYS / step - 1e-9)) + 1
    rel = np.arange(n, dtype=np.float64) * step
    rel = rel[rel < SECTOR_DAYS]
    keep = (rel < GAP_LO) | (rel >= GAP_HI)
    return T_OFFSET + SECTOR_DAYS * sector_index + rel[keep]


def kepler_duration_days(period: float, rho: float) -> float:
    """Central, circular-orbit transit duration (small-angle): P/pi * R*/a, a/R* = (G rho P^2 / 3 pi)^(1/3)."""
    a_over_r = (_K_RHO * rho * period * period / (3.0 * math.pi)) ** (1.0 / 3.0)
    return period / (math.pi * a_over_r)


def _ar1(rng: np.random.Generator, n: int, phi: float, std: float) -> np.ndarray:
    if std <= 0.0 or n == 0:
        return np.zeros(n)
    e = rng.standard_normal(n) * (std * math.sqrt(1.0 - phi * phi))
    e[0] = e[0] / math.sqrt(1.0 - phi * phi)
    try:
        from scipy.signal import lfilter
        return lfilter([1.0], [1.0, -phi], e)
    except Exception:  # pragma: no cover - scipy is in the image; keep a plain fallback
        out = np.empty(n)
        acc = 0.0
        for i in range(n):
            acc = phi * acc + e[i]
            out[i] = acc
        return out


def _inject(t, y, period, t0, depth, duration):
    ph = np.mod(t - t0 + 0.5 * duration, period)
    y[ph < duration] -= depth


def _log_uniform(rng, lo, hi):
    return math.exp(rng.uniform(math.log(lo), math.log(hi)))


def _star_layout(config: int, star_id: int, seed: int = 0):
    """The part of a star that does not depend on its flux: timestamps (after the quality-flag drops), density,
    radius, white-noise level and the injection ranges.  Consumes the star's random stream up to and including
    the drop mask, so that :func:`make_star` continues from the same state.  Configs 2-5 only."""
    rng = np.random.default_rng([seed, config, star_id])
    rho = math.exp(rng.normal(0.0, 0.5))
    rstar = math.exp(rng.normal(0.0, 0.3))
    sigma = _log_uniform(rng, 2e-4, 1e-2)
    drop = 0.0
    red_fac = 0.3
    if config == 2:
        t = sector_times(0, 200.0)
        inj_frac, p_lo, p_hi, d_lo, d_hi = 0.10, 0.5, 12.0, 3e-4, 1e-2
    elif config == 3:
        t = np.concatenate([sector_times(s, 600.0) for s in range(3)])
        inj_frac, p_lo, p_hi, d_lo, d_hi = 0.10, 0.5, 40.0, 3e-4, 1e-2
        drop = 0.02
    elif config == 4:
        t = np.concatenate([sector_times(s, 200.0) for s in range(13)])
        inj_frac, p_lo, p_hi, d_lo, d_hi = 0.10, 1.0, 150.0, 2e-4, 5e-3
        red_fac = rng.uniform(0.0, 1.0)
    elif config == 5:
        n_sec = min(int(rng.geometric(1.0 / 3.0)), 40)
        cadence = CADENCES_S[int(rng.choice(3, p=[0.5, 0.3, 0.2]))]
        sectors = [0]
        for _ in range(n_sec - 1):
            hole = 0 if rng.random() < 0.6 else int(rng.geometric(1.0 / 6.0))
            nxt = sectors[-1] + 1 + hole
            if nxt >= 70:
                break
            sectors.append(nxt)
        t = np.concatenate([sector_times(s, cadence) for s in sectors])
        inj_frac, p_lo, d_lo, d_hi = 0.05, 0.5, 3e-4, 1e-2
        # injected periods run up to the star's own longest stretch (its P_max scale)
        brk = np.nonzero(np.diff(t) > SECTOR_DAYS)[0]
        edges = np.concatenate([[0], brk + 1, [t.size]])
        longest = max(t[edges[i + 1] - 1] - t[edges[i]] for i in range(edges.size - 1))
        p_hi = max(1.0, longest if brk.size else 0.5 * longest)
        drop = 0.02
    else:
        raise ValueError(f"unknown config {config}")
    if drop > 0.0:
        t = t[rng.random(t.size) >= drop]
    return rng, t, rho, rstar, sigma, red_fac, (inj_frac, p_lo, p_hi, d_lo, d_hi)


def star_times(config: int, star_id: int, seed: int = 0):
    """Timestamps and density of one star without generating its flux -> (t, rho).  What a cost estimate needs
    (points x frequencies, for sharding stars over GPUs) at a fraction of the cost of :func:`make_star`."""
    if config == 1:
        return sector_times(0, 1800.0), 1.0
    _, t, rho, _, _, _, _ = _star_layout(config, star_id, seed)
    return t, rho


def make_star(config: int, star_id: int, seed: int = 0):
    """One star of the given config -> (t, y, dy, rho, rstar, truth tuple)."""
    truth = (0.0, 0.0, 0.0, 0.0)
    if config == 1:
        rng = np.random.default_rng([seed, config, star_id])
        t = sector_times(0, 1800.0)
        sigma = 1e-3
        rho, rstar = 1.0, 1.0
        dy = np.full(t.shape, sigma)
        y = rng.standard_normal(t.size) * sigma
        period, depth, duration = 3.7, 2e-3, 2.5 / 24.0
        t0 = t[0] + rng.uniform(0.0, period)
        _inject(t, y, period, t0, depth, duration)
        return t, y, dy, rho, rstar, (period, t0, depth, duration)

    rng, t, rho, rstar, sigma, red_fac, (inj_frac, p_lo, p_hi, d_lo, d_hi) = _star_layout(config, star_id, seed)
    n = t.size
    dy = sigma * np.exp(0.1 * rng.standard_normal(n))
    y = rng.standard_normal(n) * dy + _ar1(rng, n, 0.9, red_fac * sigma)
    if rng.random() < inj_frac:
        period = _log_uniform(rng, p_lo, p_hi)
        depth = _log_uniform(rng, d_lo, d_hi)
        duration = kepler_duration_days(period, rho)
        t0 = t[0] + rng.uniform(0.0, period)
        _inject(t, y, period, t0, depth, duration)
        truth = (period, t0, depth, duration)
    return t, y, dy, rho, rstar, truth


def make_batch(config: int, star_ids=None, seed: int = 0, n_stars: int | None = None) -> Batch:
    """CSR batch of the given stars (default: the first ``n_stars`` ids, or the whole config)."""
    if star_ids is None:
        if n_stars is None:
            n_stars = N_STARS[config]
        star_ids = np.arange(n_stars, dtype=np.int64)
    star_ids = np.asarray(star_ids, dtype=np.int64)
    ts, ys, dys = [], [], []
    S = star_ids.size
    rho = np.empty(S)
    rstar = np.empty(S)
    truth = np.zeros(S, dtype=TRUTH_DTYPE)
    row_ptr = np.zeros(S + 1, dtype=np.int64)
    for i, sid in enumerate(star_ids):
        t, y, dy, r, rs, tr = make_star(config, int(sid), seed)
        ts.append(t); ys.append(y); dys.append(dy)
        rho[i], rstar[i] = r, rs
        truth[i] = tr
        row_ptr[i + 1] = row_ptr[i] + t.size
    cat = (lambda xs: np.concatenate(xs) if xs else np.zeros(0))
    return Batch(config, seed, star_ids, row_ptr, cat(ts), cat(ys), cat(dys), rho, rstar, truth)


def from_arrays(stars, rho=None, rstar=None) -> Batch:
    """Pack hand-built (t, y, dy) triples into a Batch (used by edge-case tests)."""
    S = len(stars)
    row_ptr = np.zeros(S + 1, dtype=np.int64)
    for i, (t, _, _) in enumerate(stars):
        row_ptr[i + 1] = row_ptr[i] + len(t)
    cat = lambda k: (np.concatenate([np.asarray(s[k], dtype=np.float64) for s in stars])
                     if S else np.zeros(0))
    rho = np.ones(S) if rho is None else np.asarray(rho, dtype=np.float64)
    rstar = np.ones(S) if rstar is None else np.asarray(rstar, dtype=np.float64)
    return Batch(0, 0, np.arange(S, dtype=np.int64), row_ptr, cat(0), cat(1), cat(2), rho, rstar,
                 np.zeros(S, dtype=TRUTH_DTYPE))
