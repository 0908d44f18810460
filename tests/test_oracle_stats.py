"""Pins of the oracle's per-peak statistics (O7; "Other statistics").  None of these re-types the
oracle's loop: they are closed forms on regular grids, brute force by set arithmetic, and invariants."""
import numpy as np


def _lc(n=2000, cad=0.02, seed=0):
    rng = np.random.default_rng(seed)
    t = 1000.0 + np.arange(n) * cad
    return t, rng.standard_normal(n) * 1e-3 + 7.0, np.full(n, 1e-3)


def test_closed_form_counts_on_a_regular_grid(orc):
    # cadence 0.02 d, P = 2 d = 100 samples, duration D = m/nb * P = 21/200 * 2 = 0.21 d (window edges fall
    # between samples), mid-transit on a sample: |dt| <= 0.105 d holds for 11 samples per transit
    t, y, dy = _lc()
    P, m, nb = 2.0, 21, 200
    t0 = t[50]
    s = orc.peak_statistics(t, y, dy, 1.0 / P, m, nb, t0)
    n_tr = 20                                  # mid-times at samples 50, 150, ..., 1950: all inside the data
    assert s["n_transits"] == n_tr
    assert s["n_in"] == 11 * n_tr
    assert s["n_before"] == 10 * n_tr and s["n_after"] == 10 * n_tr   # (0.105, 0.315] d -> samples 6..15
    assert abs(s["duration"] - 0.21) < 1e-15


def test_transit_needs_data_near_mid_time(orc):
    # a transit counts only with data within 0.5 durations of the expected mid-time
    t, y, dy = _lc()
    P, m, nb = 2.0, 21, 200
    t0 = t[50]
    keep = np.ones(t.size, bool)
    keep[150 - 5:150 + 6] = False              # remove every in-transit point of the 2nd transit
    keep[250 - 5:250 + 5] = False              # 3rd transit: one in-transit point survives
    s = orc.peak_statistics(t[keep], y[keep], dy[keep], 1.0 / P, m, nb, t0)
    assert s["n_transits"] == 19
    assert s["n_in"] == 11 * 20 - 11 - 10


def test_brute_force_by_sets(orc):
    rng = np.random.default_rng(3)
    t = np.sort(1000 + rng.uniform(0, 60, 700))
    y = rng.standard_normal(700); dy = rng.uniform(0.5, 2.0, 700)
    f, m, nb, t0 = 1 / 3.3, 7, 120, 1001.234
    s = orc.peak_statistics(t, y, dy, f, m, nb, t0)
    P = 1 / f; D = m / nb * P
    cyc = np.floor((t - t0) / P + 0.5)
    dt = t - t0 - cyc * P                      # mathematically the same quantity, formed differently
    edge = np.minimum.reduce([np.abs(np.abs(dt) - 0.5 * D), np.abs(np.abs(dt) - 1.5 * D)])
    assert edge.min() > 1e-9                   # no point sits on a window edge: the counts are unambiguous
    inn = np.abs(dt) <= 0.5 * D
    assert s["n_in"] == inn.sum()
    assert s["n_before"] == ((dt < -0.5 * D) & (dt >= -1.5 * D)).sum()
    assert s["n_after"] == ((dt > 0.5 * D) & (dt <= 1.5 * D)).sum()
    assert s["n_transits"] == np.unique(cyc[inn]).size
    w = dy[~inn] ** -2.0
    assert abs(s["oot_level"] - np.sum(w * y[~inn]) / np.sum(w)) < 1e-12


def test_invariants(orc):
    t, y, dy = _lc(seed=5)
    f, m, nb, t0 = 1 / 2.7, 5, 90, t[3] + 0.0123
    a = orc.peak_statistics(t, y, dy, f, m, nb, t0)
    b = orc.peak_statistics(t, y + 3.0, dy * 2.0, f, m, nb, t0)     # offset in y, scale in dy
    for k in ("n_in", "n_before", "n_after", "n_transits"):
        assert a[k] == b[k]
    assert abs((b["oot_level"] - a["oot_level"]) - 3.0) < 1e-12
    c = orc.peak_statistics(t, y, dy, f, m, nb, t0 + 5 / f)         # epoch shifted by whole periods
    for k in ("n_in", "n_before", "n_after", "n_transits"):
        assert a[k] == c[k]
    assert a["n_in"] + a["n_before"] + a["n_after"] <= t.size
