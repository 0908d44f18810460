"""Pins for the oracle's fold + box-scan (O2-O4): exact-rational bin indices, the aligned closed
form SR = delta^2 r (1 - r), invariants, unbinned brute force on tiny inputs, injection recovery.

The brute-force searches below are written independently in numpy/Python (sorted phases, cyclic
contiguous subsets); they share nothing with oracle/qlp_oracle.c.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from paper_2302_01293_b200 import synth


# ------------------------------------------------------------------ O3: bin index
def test_bin_index_against_exact_rationals(orc):
    """O3 (reading A17): b = floor(nb * frac(p)) exactly, p = fl64(f * tau) the only rounding.
    Checked on every point with Python rationals; and against the exact (unrounded) product f*tau
    wherever that is not within 1e-9 bin of an edge (the rounding of p cannot matter there)."""
    rng = np.random.default_rng(7)
    tau = np.sort(rng.uniform(0.0, 400.0, 4000))
    checked = 0
    for f, nb in ((0.0731, 433), (0.91, 97), (3.05, 38), (1.0 / 3.0, 150), (16.7, 38), (0.0056, 7814)):
        b = orc.bins(f, nb, tau)
        assert b.min() >= 0 and b.max() <= nb - 1
        for i in range(0, tau.size, 3):
            p = Fraction(float(f) * float(tau[i]))                  # the rounded FP64 product, exactly
            assert b[i] == math.floor((p - math.floor(p)) * nb)
            pe = Fraction(float(f)) * Fraction(float(tau[i]))       # exact product of the two doubles
            x = (pe - math.floor(pe)) * nb
            if min(x - math.floor(x), math.ceil(x) - x) > Fraction(1, 10 ** 9):   # away from a bin edge
                assert b[i] == math.floor(x)
                checked += 1
    assert checked > 6000


def test_bin_index_no_double_rounding(orc):
    """The case that separates the exact floor from floor(fl64(ph*nb)): ph*nb just below an integer."""
    ph = np.nextafter(1.0, 0.0)                  # 1 - 2^-53
    for nb in (38, 91, 455, 7814):
        assert orc.bins(1.0, nb, np.array([ph]))[0] == nb - 1
    # ph = (n - eps)/nb with eps tiny: fl64(ph*nb) may round up to n, the exact floor is n-1 or n
    rng = np.random.default_rng(11)
    for nb in (97, 433):
        for n in rng.integers(1, nb, 200):
            ph = np.nextafter(float(n) / nb, 0.0)
            want = math.floor(Fraction(ph) * nb)
            assert orc.bins(1.0, nb, np.array([ph]))[0] == want


def test_bin_index_edges(orc):
    # integer phase -> bin 0; phase just below 1 -> last bin (exact floor: never reaches nb)
    tau = np.array([0.0, 1.0, 2.0, 4.0, 0.5, 0.25, np.nextafter(1.0, 0.0), np.nextafter(3.0, 0.0)])
    b = orc.bins(1.0, 40, tau)
    assert list(b) == [0, 0, 0, 0, 20, 10, 39, 39]
    # monotone staircase over one cycle
    tau = np.linspace(0.0, 1.0, 1001)[:-1]
    b = orc.bins(1.0, 38, tau)
    assert np.all(np.diff(b) >= 0) and b[0] == 0 and b[-1] == 37
    assert np.all(np.bincount(b, minlength=38) >= 26)


# ------------------------------------------------------------------ O4: closed form
@pytest.mark.parametrize("kfrac,j,m", [(0.1, 0, 3), (0.5, 17, 7), (0.9, 30, 11), (0.3, -2, 5)])
def test_aligned_box_closed_form(orc, cfg, kfrac, j, m):
    """Noiseless box aligned with the fine bins: SR = delta^2 r (1 - r), best (m, j) returned."""
    t, _, _, rho, _, _ = synth.make_star(2, 1)
    t = t[::4]
    rng = np.random.default_rng(3)
    dy = 1e-3 * np.exp(0.3 * rng.standard_normal(t.size))
    g = orc.grid(cfg, t, rho)
    k = int(kfrac * g["n_freq"])
    (f,), (nb,) = orc.freqs(cfg, g, k, k + 1)
    j = j % nb
    tau, w, _ = orc.prep(t, np.zeros_like(t), dy, g["t_ref"])
    b = orc.bins(f, nb, tau)
    inside = ((b - j) % nb) < m
    assert inside.any() and not inside.all()
    delta = 2.5e-3
    y = np.where(inside, -delta, 0.0) + 0.75       # any constant offset drops out
    sr, mb, jb = orc.spectrum_star(cfg, g, t, y, dy)
    r = w[inside].sum()
    assert sr[k] == pytest.approx(delta ** 2 * r * (1.0 - r), rel=1e-11)
    assert (mb[k], jb[k]) == (m, j)
    rec = orc.peak_record(cfg, g, t, y, dy, k, 0.0)
    assert rec["depth"] == pytest.approx(delta, rel=1e-10)
    assert rec["q"] == pytest.approx(m / nb)
    assert rec["t0"] == pytest.approx(g["t_ref"] + ((j + 0.5 * m) / nb) / f, rel=1e-14)


def test_constant_series_gives_zero(orc, cfg):
    t, _, dy, rho, _, _ = synth.make_star(1, 0)
    g = orc.grid(cfg, t, rho)
    for c in (0.0, 1.0, -37.5):
        sr, mb, jb = orc.spectrum_star(cfg, g, t, np.full_like(t, c), dy)
        assert sr.max() <= 1e-25 * max(1.0, c * c)
    sr, mb, jb = orc.spectrum_star(cfg, g, t, np.zeros_like(t), dy)
    assert np.all(sr == 0.0) and np.all(mb == 3) and np.all(jb == 0)     # all-zero convention


def test_shift_and_scale_invariances(orc, cfg):
    t, y, dy, rho, _, _ = synth.make_star(3, 2)
    t, y, dy = t[:3000], y[:3000], dy[:3000]
    g = orc.grid(cfg, t, rho)
    sr, mb, jb = orc.spectrum_star(cfg, g, t, y, dy)
    sr_c, *_ = orc.spectrum_star(cfg, g, t, y + 0.5, dy)
    assert np.allclose(sr_c, sr, rtol=1e-8, atol=1e-12 * sr.max())
    sr_a, *_ = orc.spectrum_star(cfg, g, t, -3.0 * y, dy)
    assert np.allclose(sr_a, 9.0 * sr, rtol=1e-12)
    sr_d, *_ = orc.spectrum_star(cfg, g, t, y, 7.0 * dy)
    assert np.allclose(sr_d, sr, rtol=1e-11)


# ------------------------------------------------------------------ brute force
def brute_all_subsets(phase, w, wy):
    """max s^2/(r(1-r)) over ALL cyclic contiguous subsets in phase order (unbinned BLS)."""
    o = np.argsort(phase, kind="stable")
    w, wy = w[o], wy[o]
    n = w.size
    best = 0.0
    for a in range(n):
        r = s = 0.0
        for L in range(1, n):
            i = (a + L - 1) % n
            r += w[i]; s += wy[i]
            if 0.0 < r < 1.0:
                best = max(best, s * s / (r * (1.0 - r)))
    return best


def test_binned_sr_never_beats_unbinned_brute_force(orc, cfg):
    rng = np.random.default_rng(11)
    hits = 0
    for trial in range(6):
        n = 40 + trial * 4
        t = 2000.0 + np.sort(rng.uniform(0.0, 30.0, n))
        y = rng.standard_normal(n)
        dy = np.exp(0.2 * rng.standard_normal(n))
        g = orc.grid(cfg, t, 1.0)
        sr, mb, jb = orc.spectrum_star(cfg, g, t, y, dy)
        f, nb = orc.freqs(cfg, g)
        tau, w, wy = orc.prep(t, y, dy, g["t_ref"])
        for k in range(0, f.size, max(1, f.size // 25)):
            p = f[k] * tau
            bf = brute_all_subsets(p - np.floor(p), w, wy)
            assert sr[k] <= bf * (1.0 + 1e-12)
            assert sr[k] >= 0.2 * bf            # and it is not trivially small
            hits += sr[k] >= bf * (1.0 - 1e-12)
    assert hits >= 1   # equality happens when the best subset is exactly a bin window


def brute_windows(phase, w, wy, lmin, lmax):
    """Unbinned search restricted to phase windows [a, a + l), lmin <= l <= lmax: a contiguous run
    of points (cyclic, phase order) is selectable iff it fits in lmax and its two outside
    neighbours are more than lmin apart."""
    o = np.argsort(phase, kind="stable")
    ph, w, wy = phase[o], w[o], wy[o]
    n = ph.size
    best = 0.0
    for a in range(n):
        r = s = 0.0
        for L in range(1, n - 1):
            i = (a + L - 1) % n
            r += w[i]; s += wy[i]
            extent = (ph[i] - ph[a]) % 1.0
            outer = (ph[(i + 1) % n] - ph[(a - 1) % n]) % 1.0
            if extent < lmax and outer > lmin and 0.0 < r < 1.0:
                best = max(best, s * s / (r * (1.0 - r)))
    return best


def test_fine_bins_converge_to_width_restricted_brute_force(orc):
    """Generalised oracle call (arbitrary nb, M): as nb grows the binned search selects exactly the
    point subsets of the continuous window search, up to the 1/nb edge quantisation (sandwich)."""
    rng = np.random.default_rng(5)
    nb = 1500
    M = np.arange(60, 121)            # windows 0.04 .. 0.08 of the phase
    for trial in range(4):
        n = 24
        tau = np.sort(rng.uniform(0.0, 50.0, n))
        y = rng.standard_normal(n); dy = np.ones(n)
        _, w, wy = orc.prep(tau, y, dy, 0.0)
        f = 0.1 + 0.37 * trial
        sr, m, j, r, s = orc.sr_one(tau, w, wy, f, nb, M)
        p = f * tau
        ph = p - np.floor(p)
        eps = 2.0 / nb
        lo = brute_windows(ph, w, wy, M[0] / nb + eps, M[-1] / nb - eps)   # surely reachable
        hi = brute_windows(ph, w, wy, M[0] / nb - eps, M[-1] / nb + eps)   # everything reachable
        assert lo * (1 - 1e-12) <= sr <= hi * (1 + 1e-12)
        assert sr == pytest.approx(s * s / (r * (1 - r)), rel=1e-13)


# ------------------------------------------------------------------ injection recovery (config 1)
def test_injection_recovery_config1(orc, cfg):
    b = synth.make_batch(1)
    t, y, dy = b.star(0)
    tr = b.truth[0]
    out = orc.batch(cfg, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3)
    g = out["grid"][0]
    pk = out["peaks"][0, 0]
    f, nb = orc.freqs(cfg, g)
    k = int(pk["k"])
    grid_step_P = abs(1.0 / f[k] - 1.0 / f[k + 1])
    assert abs(pk["period"] - tr["period"]) <= 1.5 * grid_step_P
    assert abs(pk["q"] - tr["duration"] / tr["period"]) <= 1.0 / pk["nb"]
    dt = (pk["t0"] - tr["t0"] + 0.5 * pk["period"]) % pk["period"] - 0.5 * pk["period"]
    assert abs(dt) <= pk["period"] / pk["nb"]
    assert pk["depth"] == pytest.approx(tr["depth"], rel=0.25)
    assert pk["snr"] > 9.0                      # PAPER.md:55 detection threshold
    # noiseless expectation delta^2 r (1-r) with r ~ duration/period
    r = tr["duration"] / tr["period"]
    assert 0.5 < pk["sr"] / (tr["depth"] ** 2 * r * (1 - r)) < 2.0


# ------------------------------------------------------------------ test helpers of the oracle
def test_sampled_spectrum_and_box_values_helpers(orc, cfg):
    """orc_spectrum_samples is orc_spectrum_star restricted to some k (bitwise); orc_box_values agrees with a numpy
    evaluation of the same box written here from the definition (weights, bins from exact rationals' floor)."""
    b = synth.make_batch(2, n_stars=1)
    t, y, dy = b.star(0)
    t, y, dy = t[::8], y[::8], dy[::8]
    g = orc.grid(cfg, t, float(b.rho[0]))
    sr, m, j = orc.spectrum_star(cfg, g, t, y, dy)
    rng = np.random.default_rng(5)
    ks = np.unique(np.concatenate([[0, int(g["n_freq"]) - 1], rng.integers(0, int(g["n_freq"]), 40)]))
    s2, m2, j2 = orc.spectrum_samples(cfg, g, t, y, dy, ks)
    assert np.array_equal(s2, sr[ks]) and np.array_equal(m2, m[ks]) and np.array_equal(j2, j[ks])
    # the best box re-evaluated point by point reproduces SR (summation order differs: 1e-12)
    v = orc.box_values(cfg, g, t, y, dy, ks, m[ks], j[ks])
    assert np.abs(v - sr[ks]).max() <= 1e-12 * sr.max()
    # an arbitrary other box, from the definition in numpy
    w = dy ** -2.0 / np.sum(dy ** -2.0)
    yt = y - np.sum(w * y)
    for k in ks[:10]:
        (f,), (nb,) = orc.freqs(cfg, g, int(k), int(k) + 1)
        mm, jj = int(rng.integers(3, 12)), int(rng.integers(0, nb))
        ph = np.array([float(Fraction(float(f) * float(x)) % 1) for x in (t - t[0])])
        bins = np.floor(ph * nb).astype(np.int64)
        sel = ((bins - jj) % nb) < mm
        r, s = w[sel].sum(), (w * yt)[sel].sum()
        want = s * s / (r * (1 - r)) if 0 < r < 1 else 0.0
        got = orc.box_values(cfg, g, t, y, dy, [k], [mm], [jj])[0]
        assert abs(got - want) <= 1e-9 * max(want, 1e-30)
        assert got <= sr[k] * (1 + 1e-12)      # no box beats the maximum
