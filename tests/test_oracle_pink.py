"""Pins of oracle O9: sigma_w, sigma_r on the transit-duration timescale, S/N_pink (Eq. 2) and the detection
criteria (O9).

Pinned to things other than the oracle: closed forms on constructed residuals (equal bins of four points), the
positivity floor, a brute force with numpy's grouping routines (np.unique / np.bincount) on gappy random data, the
statistics of white noise, the O7 counts (another code path, pinned on its own), and the paper's formula evaluated
on numbers known by construction."""
import numpy as np
import pytest

from oracle import oracle

CAD = 1.0 / 64.0            # cadence in days: a power of two, so times and bin edges are exact


def regular(n):
    return np.arange(n) * CAD


def test_closed_form_bins_of_four():
    """Residual +a in even bins, -a in odd bins, bins of exactly four points, no transit (depth 0):
    sigma_w = a, bin means +-a, sigma_bin = a, mean(1/n_b) = 1/4  =>  sigma_r^2 = a^2 (1 - 1/4)."""
    n, a, z = 4 * 200, 0.003, 1.0
    t = regular(n)
    r = np.where((np.arange(n) // 4) % 2 == 0, a, -a)
    P = 8.0
    q = 4 * CAD / P                                # D = q P = four cadences exactly
    o = oracle.pink_noise(t, z + r, 1.0 / P, 1.0, 0.0, q, 0.25, z, 20.0)
    assert o["n_bins"] == 200
    assert o["sigma_w"] == pytest.approx(a, rel=1e-12)
    assert o["sigma_r"] == pytest.approx(a * np.sqrt(0.75), rel=1e-12)
    assert o["depth_eff"] == 0.0 and o["snr_pink"] == 0.0 and o["detected"] == 0


def test_white_part_is_removed_and_floored_at_zero():
    """Residuals alternating +-a inside every bin of four: all bin means are 0, so sigma_bin^2 - sigma_w^2/4 < 0."""
    n, a = 4 * 100, 0.01
    t = regular(n)
    r = np.where(np.arange(n) % 2 == 0, a, -a)
    P = 8.0
    o = oracle.pink_noise(t, r, 1.0 / P, 1.0, 0.0, 4 * CAD / P, 0.0, 0.0, 20.0)
    assert o["sigma_w"] == pytest.approx(a, rel=1e-12) and o["sigma_r"] == 0.0


def brute(t, y, P, T0, delta, q, q_in, z):
    x = (t - T0) / P
    cyc = np.floor(x + 0.5)
    dt = (x - cyc) * P
    D = q * P
    if q_in > 0:
        sh = np.interp(dt, [-0.5 * D, -0.5 * D + q_in * D, 0.5 * D - q_in * D, 0.5 * D], [0.0, 1.0, 1.0, 0.0])
    else:
        sh = (np.abs(dt) < 0.5 * D).astype(float)
    r = y - (z - delta * sh)
    var_w = np.var(r)
    b = np.floor((t - t[0]) / D).astype(np.int64)
    _, inv, cnt = np.unique(b, return_inverse=True, return_counts=True)
    mb = np.bincount(inv, weights=r) / cnt
    var_r = max(0.0, np.var(mb) - var_w * np.mean(1.0 / cnt))
    intr = np.abs(dt) <= 0.5 * D
    n_t = int(intr.sum())
    N_t = int(np.unique(cyc[intr]).size)
    return np.sqrt(var_w), np.sqrt(var_r), n_t, N_t, int(cnt.size)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_brute_force_with_numpy_grouping_on_gappy_red_noise(seed):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0.0, 27.0, 6000))
    t = t[(t < 12.5) | (t > 14.0)]                                     # a gap: empty bins must not count
    P, T0, delta, q, q_in, z = 3.3 + seed, 1.1, 0.004, 0.03, [0.0, 0.2, 0.5][seed], 1.0
    red = 0.002 * np.sin(2 * np.pi * t / 0.7)
    x = (t - T0) / P
    dt = (x - np.floor(x + 0.5)) * P
    y = z - delta * (np.abs(dt) < 0.5 * q * P) + red + 0.001 * rng.standard_normal(t.size)
    o = oracle.pink_noise(t, y, 1.0 / P, T0, delta, q, q_in, z, 12.0)
    sw, sr, n_t, N_t, nb = brute(t, y, P, T0, delta, q, q_in, z)
    assert (o["n_t"], o["n_transits"], o["n_bins"]) == (n_t, N_t, nb)
    assert o["sigma_w"] == pytest.approx(sw, rel=1e-10) and o["sigma_r"] == pytest.approx(sr, rel=1e-9)
    assert o["sigma_r"] > 0.5 * 0.002 / np.sqrt(2)                     # the injected red noise is seen
    # PAPER.md Eq. 2 with delta replaced by the trapezoid integral, on the brute-force numbers
    want = delta * (1.0 - q_in) / np.sqrt(sw ** 2 / n_t + sr ** 2 / N_t)
    assert o["snr_pink"] == pytest.approx(want, rel=1e-9)
    assert o["depth_eff"] == pytest.approx(delta * (1.0 - q_in), rel=1e-15)


def test_white_noise_has_little_red_noise():
    rng = np.random.default_rng(5)
    t = regular(20000)
    y = 0.001 * rng.standard_normal(t.size)
    P = 2.0
    o = oracle.pink_noise(t, y, 1.0 / P, 0.3, 0.0, 16 * CAD / P, 0.1, 0.0, 0.0)
    assert o["sigma_w"] == pytest.approx(0.001, rel=0.03)
    assert o["sigma_r"] < 0.1 * o["sigma_w"]                           # ~ sigma_w / sqrt(16) / (2 N_b)^(1/4) at most


def test_counts_agree_with_o7_and_detection_criteria():
    rng = np.random.default_rng(9)
    t = regular(1700)
    P, T0, m, nb = 3.0, 0.7, 5, 200
    q = m / nb
    x = (t - T0) / P
    dt = (x - np.floor(x + 0.5)) * P
    dy = np.full(t.size, 1e-3)
    depth = 0.01
    y = 1.0 - depth * (np.abs(dt) <= 0.5 * q * P) + 1e-3 * rng.standard_normal(t.size)
    st = oracle.peak_statistics(t, y, dy, 1.0 / P, m, nb, T0)
    o = oracle.pink_noise(t, y, 1.0 / P, T0, depth, q, 0.0, 1.0, 15.0)
    assert (o["n_t"], o["n_transits"]) == (st["n_in"], st["n_transits"])
    assert o["n_transits"] >= 2 and o["snr_pink"] > 9.0 and o["detected"] == 1
    assert oracle.pink_noise(t, y, 1.0 / P, T0, depth, q, 0.0, 1.0, 8.9)["detected"] == 0      # S/N <= 9
    assert oracle.pink_noise(t, y, 1.0 / P, T0, 1e-4, q, 0.0, 1.0, 15.0)["detected"] == 0      # S/N_pink <= 9
    one = t < T0 + 0.5 * P                                                               # a single transit
    o1 = oracle.pink_noise(t[one], y[one], 1.0 / P, T0, depth, q, 0.0, 1.0, 15.0)
    assert o1["n_transits"] == 1 and o1["detected"] == 0
    # V-shaped transit of the same depth: half the signal (grazing transits)
    ov = oracle.pink_noise(t, y, 1.0 / P, T0, depth, q, 0.5, 1.0, 15.0)
    assert ov["depth_eff"] == pytest.approx(0.5 * depth)
