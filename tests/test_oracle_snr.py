"""Pins for the oracle's S/N spectrum and peaks (O5/O6; PAPER.md:37-42 and footnote 3 at :65).

Library special cases: the trend equals numpy's ``interp`` through per-bin ``median`` values and
sigma equals 1.4826 * numpy MAD.  Peaks are checked against a brute-force sort of local maxima.
"""
import math

import numpy as np
import pytest


def test_sturges_values_by_hand(orc):
    # N = 1 + 3.322 log10 n, rounded to nearest: 13.13, 14.89, 17.14, 20.54 -> 13, 15, 17, 21
    for n, N in ((4489, 13), (15138, 15), (72098, 17), (763623, 21), (1, 1), (2, 2), (10, 4), (100, 8)):
        assert orc.sturges(n) == N
        assert N == int(math.floor(1 + 3.322 * math.log10(n) + 0.5))


def numpy_snr(f, sr):
    n = f.size
    N = int(math.floor(1 + 3.322 * math.log10(n) + 0.5))
    edges = np.linspace(f[0], f[-1], N + 1)
    which = np.minimum(np.searchsorted(edges, f, side="right") - 1, N - 1)
    cx, cy = [], []
    for b in range(N):
        sel = sr[which == b]
        if sel.size:
            cx.append(0.5 * (edges[b] + edges[b + 1])); cy.append(np.median(sel))
    trend = np.interp(f, cx, cy)
    sigma = 1.4826 * np.median(np.abs(sr - np.median(sr)))
    return (sr - trend) / sigma, trend, sigma


@pytest.mark.parametrize("n", [1, 2, 3, 10, 57, 4489, 20001])
def test_snr_equals_numpy_interp_of_binned_medians(orc, n):
    rng = np.random.default_rng(n)
    u = np.sort(rng.uniform(0.3, 1.4, n))
    f = u ** 3                                   # non-uniform, like the real grid
    sr = rng.gamma(3.0, 1e-8, n) * (1.0 + 2.0 / (0.2 + f))   # rising toward low frequency
    snr, trend, sigma = orc.snr(f, sr)
    if n >= 3:
        ref, rtrend, rsigma = numpy_snr(f, sr)
        # bin edges from linspace vs (f-f0)/span*N may differ for a point exactly on an edge: none here
        assert sigma == pytest.approx(rsigma, rel=1e-14)
        assert np.allclose(trend, rtrend, rtol=1e-12, atol=0)
        assert np.allclose(snr, ref, rtol=1e-9, atol=1e-9)
    else:
        assert np.all(np.isfinite(snr))


def test_snr_invariances(orc):
    rng = np.random.default_rng(2)
    f = np.sort(rng.uniform(0.1, 3.0, 5000))
    sr = rng.gamma(2.0, 1.0, 5000)
    s0, _, _ = orc.snr(f, sr)
    s1, _, _ = orc.snr(f, 3.5 * sr + 11.0)
    assert np.allclose(s0, s1, rtol=1e-9, atol=1e-9)
    flat, _, sig = orc.snr(f, np.full(5000, 2.0))
    assert sig == 0.0 and np.all(flat == 0.0)
    # the median-binned trend removes a rise toward low frequency
    sr2 = 1.0 + 5.0 / f + 0.01 * rng.standard_normal(5000)
    s2, tr, _ = orc.snr(f, sr2)
    assert abs(np.median(s2[:500])) < 5.0 and abs(np.median(s2[-500:])) < 1.0


def brute_peaks(snr, K):
    n = snr.size
    k1 = int(np.argmax(snr))
    cand = []
    for k in range(n):
        if n == 1:
            break
        left = k == 0 or snr[k] > snr[k - 1]
        right = k == n - 1 or snr[k] >= snr[k + 1]
        if left and right and k != k1:
            cand.append(k)
    cand.sort(key=lambda k: (-snr[k], k))
    return [k1] + cand[:K - 1]


def test_peaks_against_bruteforce(orc):
    rng = np.random.default_rng(9)
    for n in (1, 2, 5, 50, 1000):
        for rep in range(5):
            snr = np.round(rng.standard_normal(n), 1)      # rounding makes ties and plateaus common
            for K in (1, 3, 8):
                got = list(orc.peak_indices(snr, K))
                assert got == brute_peaks(snr, K)
