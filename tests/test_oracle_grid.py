"""Pins for the oracle's grid stage (O0/O1): closed forms, hand-built timestamp sets, invariants.

Nothing here re-types the oracle's formulas: P_min and C_q are checked against Kepler's third
law in SI units, counts against direct enumeration, P_max against hand-built gap patterns
(PAPER.md:19, 23, 35).
"""
import math

import numpy as np
import pytest

from paper_2302_01293_b200 import synth

GM_SUN = 1.3271244e20   # m^3 s^-2 (IAU nominal)
R_SUN = 6.957e8         # m


def a_over_r(period_days, rho_solar):
    """Kepler III with M = rho * 4/3 pi R^3 (R cancels): a/R for a given period, SI units."""
    P = period_days * 86400.0
    R = R_SUN  # any radius: it cancels
    M_G = GM_SUN * rho_solar * (R / R_SUN) ** 3
    a = (M_G * P * P / (4.0 * math.pi ** 2)) ** (1.0 / 3.0)
    return a / R


def uniform_t(n, step, t0=2000.0):
    return t0 + step * np.arange(n)


def test_cbrt_det_exact_cases(orc):
    for i in range(1, 40):
        assert orc.cbrt_det(float(i ** 3)) == float(i)
    for e in range(-30, 31):
        assert orc.cbrt_det(8.0 ** e) == 2.0 ** e


def test_cbrt_det_accuracy(orc):
    rng = np.random.default_rng(1)
    x = np.exp(rng.uniform(-40, 40, 20000))
    y = np.array([orc.cbrt_det(v) for v in x])
    ref = np.cbrt(x)
    ulp = np.spacing(ref)
    assert np.max(np.abs(y - ref) / ulp) <= 1.0
    # y within 1 ulp of the true root => y^3 within 3*(1 ulp relative) of x: at most 4 ulp(x); exact rationals
    from fractions import Fraction
    for v, r in zip(x[:300], y[:300]):
        err = abs(Fraction(r) ** 3 - Fraction(v))
        assert err <= 4 * Fraction(float(np.spacing(v)))


def test_pmin_is_where_a_equals_k_rstar(orc):
    t = synth.sector_times(0, 1800.0)
    for k, expect in ((2.0, 0.327634), (3.0, 0.601901)):
        for rho in (1.0, 0.3, 4.2):
            g = orc.grid(orc.default_config(a_over_rstar_min=k), t, rho)
            assert a_over_r(g["p_min"], rho) == pytest.approx(k, rel=1e-7)
        g = orc.grid(orc.default_config(a_over_rstar_min=k), t, 1.0)
        assert g["p_min"] == pytest.approx(expect, abs=1e-6)


def test_cq_is_circular_central_duty_cycle(orc, cfg):
    t = synth.sector_times(0, 1800.0)
    for rho in (1.0, 0.2, 7.0):
        g = orc.grid(cfg, t, rho)
        for P in (0.7, 3.0, 11.0):
            q_circ = g["c_q"] * (1.0 / P) ** (2.0 / 3.0)
            assert q_circ == pytest.approx(1.0 / (math.pi * a_over_r(P, rho)), rel=1e-7)
    assert orc.grid(cfg, t, 1.0)["c_q"] == pytest.approx(0.0756390, abs=1e-7)


def test_missing_density_is_solar(orc, cfg):
    t = synth.sector_times(0, 1800.0)
    ref = orc.grid(cfg, t, 1.0)
    for bad in (float("nan"), 0.0, -1.0, float("inf")):
        assert orc.grid(cfg, t, bad) == ref


def test_pmax_rule(orc, cfg):
    step = 0.02
    # no gap at all: half the stretch
    t = uniform_t(2001, step)
    assert orc.grid(cfg, t)["p_max"] == pytest.approx(0.5 * (t[-1] - t[0]), rel=1e-15)
    # 1-d gaps only (shorter than a sector): still one stretch -> half of the full span
    t1 = np.concatenate([uniform_t(600, step), uniform_t(600, step, 2000.0 + 600 * step + 1.0)])
    assert orc.grid(cfg, t1)["p_max"] == pytest.approx(0.5 * (t1[-1] - t1[0]), rel=1e-15)
    # one 30-d gap: longest side, not halved
    a, b = uniform_t(500, step), uniform_t(900, step, 2000.0 + 500 * step + 30.0)
    t2 = np.concatenate([a, b])
    assert orc.grid(cfg, t2)["p_max"] == pytest.approx(b[-1] - b[0], rel=1e-15)
    t2r = np.concatenate([uniform_t(900, step), uniform_t(500, step, 2000.0 + 900 * step + 30.0)])
    assert orc.grid(cfg, t2r)["p_max"] == pytest.approx(899 * step, rel=1e-12)
    # a gap of exactly one sector is not a break; one cadence more is (dyadic numbers: exact)
    sd = 27.5
    c = orc.default_config(sector_days=sd)
    left = 1000.0 + 0.25 * np.arange(100)
    for extra, is_break in ((0.0, False), (0.25, True)):
        right = left[-1] + sd + extra + 0.25 * np.arange(300)
        tt = np.concatenate([left, right])
        assert (tt[100] - tt[99] > sd) == is_break
        want = (right[-1] - right[0]) if is_break else 0.5 * (tt[-1] - tt[0])
        assert orc.grid(c, tt)["p_max"] == want


def test_grid_closed_forms(orc, cfg):
    for conf, sid in ((1, 0), (2, 3), (3, 5)):
        t, y, dy, rho, rstar, _ = synth.make_star(conf, sid)
        g = orc.grid(cfg, t, rho)
        assert g["status"] == 0
        f, nb = orc.freqs(cfg, g)
        n = f.size
        assert n == g["n_freq"] and n > 1000
        # ends: first frequency is 1/P_max (cube-root round trip), last one does not pass 1/P_min
        assert f[0] == pytest.approx(1.0 / g["p_max"], rel=4e-16 * 4)
        assert f[-1] <= (1.0 / g["p_min"]) * (1 + 1e-15)
        u1 = (1.0 / g["p_min"]) ** (1.0 / 3.0)
        assert u1 - (g["u0"] + n * g["h"]) < 0  # one more step would overshoot
        assert np.all(np.diff(f) > 0)
        # spacing law: df = q_lo(f) / (samples_per_peak * T), q_lo = 0.5 q_circ
        q_lo = 0.5 * g["c_q"] * f ** (2.0 / 3.0)
        df = np.diff(f)
        assert np.allclose(df, (q_lo[:-1] / (2.0 * g["baseline"])), rtol=3e-3)
        # fine bins: narrowest searched box is exactly noverlap = 3 bins; grid ends at a/R* = 2
        assert np.all(nb == np.ceil(3.0 / q_lo - 1e-9)) or np.mean(nb == np.ceil(3.0 / q_lo)) > 0.999
        assert nb[-1] == 38 == math.ceil(3 * 4 * math.pi)
        assert nb[0] == g["nb_max"] == nb.max()
        assert np.all(np.diff(nb) <= 0)


def test_grid_sizes_match_design(orc, cfg):
    # config 1: one 27.4-d sector at 30 min, solar star
    t, *_ = synth.make_star(1, 0)
    g = orc.grid(cfg, t, 1.0)
    assert t.size == 1268 and g["n_freq"] == 4489 and g["nb_max"] == 455
    # a 40-sector 200-s star stays within "up to ~10 times" 80,000 frequencies
    t40 = 2000.0 + np.arange(0.0, 40 * 27.4, 1.0)   # continuous 40-sector baseline
    assert 1e5 < orc.grid(cfg, t40, 1.0)["n_freq"] < 1.2e6


def test_comparison_grid_caps(orc, cfg):
    """O1.10: the earlier search's grid, "an under-sampled frequency grid on the order of 80,000
    frequencies or less" with "periods up to only ~56 days".  Pins: caps that do not bite change nothing;
    the period cap moves only the low-frequency end; the frequency cap keeps both ends and the f^(1/3) law
    and stretches the step by (n - 1)/(M - 1)."""
    t = 2000.0 + np.arange(0.0, 13 * 27.4, 1.0 / 48.0)          # 13 continuous sectors, 30-min cadence
    g0 = orc.grid(cfg, t, 1.0)
    n0 = int(g0["n_freq"])
    assert g0["p_max"] == pytest.approx(0.5 * (t[-1] - t[0]), rel=1e-15) and g0["p_max"] > 56.0
    # caps that do not bite: bit-identical descriptor
    loose = orc.grid(orc.default_config(max_period_days=1e4, max_freq=n0), t, 1.0)
    assert loose.tobytes() == g0.tobytes()
    # period cap: P_max = 56 exactly, same step, same high end, fewer frequencies
    gp = orc.grid(orc.default_config(max_period_days=56.0), t, 1.0)
    assert gp["p_max"] == 56.0 and gp["h"] == g0["h"] and gp["p_min"] == g0["p_min"] and gp["c_q"] == g0["c_q"]
    assert gp["u0"] == pytest.approx((1.0 / 56.0) ** (1.0 / 3.0), rel=1e-15)
    assert gp["n_freq"] < n0 and gp["nb_max"] < g0["nb_max"]
    # the dropped frequencies are exactly those below 1/56 (counted on the uncapped grid, +-1 for the offset)
    f0, _ = orc.freqs(cfg, g0)
    assert abs((n0 - int(gp["n_freq"])) - int(np.sum(f0 < 1.0 / 56.0))) <= 1
    # frequency cap: exactly M frequencies over the same range
    for M in (80000, 1000, 2):
        cm = orc.default_config(max_freq=M)
        gm = orc.grid(cm, t, 1.0)
        if n0 <= M:
            assert gm.tobytes() == g0.tobytes()
            continue
        assert gm["n_freq"] == M and gm["u0"] == g0["u0"] and gm["nb_max"] == g0["nb_max"]
        u1 = (1.0 / g0["p_min"]) ** (1.0 / 3.0)
        assert gm["h"] == pytest.approx((u1 - g0["u0"]) / (M - 1), rel=1e-14)
        assert gm["h"] > g0["h"]                                 # under-sampled
        f, nb = orc.freqs(cm, gm)
        assert f.size == M and f[0] == f0[0]
        assert f[-1] == pytest.approx(1.0 / g0["p_min"], rel=1e-13)
        assert np.all(np.diff(f) > 0) and np.all(np.diff(nb) <= 0) and nb[-1] == 38
        # uniform in u = f^(1/3)
        du = np.diff(np.cbrt(f))
        assert np.allclose(du, gm["h"], rtol=1e-9)
    # both caps together = the comparison workload; a short light curve is untouched by it
    both = orc.default_config(max_period_days=56.0, max_freq=80000)
    t1, *_ = synth.make_star(1, 0)
    assert orc.grid(both, t1, 1.0).tobytes() == orc.grid(cfg, t1, 1.0).tobytes()
    gb = orc.grid(both, 2000.0 + np.arange(0.0, 13 * 27.4, 200.0 / 86400.0), 8.0)   # dense star, 200 s: > 80,000
    assert gb["n_freq"] == 80000 and gb["p_max"] == 56.0
    # context of PAPER.md:59 ("up to ~10 times more frequencies" on the GPU grid): longest baseline (40 sectors),
    # a dense (rho* = 10) star; a solar star gets ~3 times more, a single-sector star the same grid
    t40 = 2000.0 + np.arange(0.0, 40 * 27.4, 1.0 / 48.0)
    ratio = lambda rho: orc.grid(cfg, t40, rho)["n_freq"] / orc.grid(both, t40, rho)["n_freq"]
    assert 5.0 < ratio(10.0) < 15.0 and 2.0 < ratio(1.0) < 4.0


def test_comparison_grid_uniform_in_frequency(orc, cfg):
    """O1.10c: the comparison grid with equal steps in frequency.  Pins, none of
    them the oracle's own formula: the frequencies are an arithmetic progression from 1/P_max to (at most) 1/P_min;
    uncapped, its step is the smallest step of the GPU grid (the one at its low-frequency end); capped, exactly
    max_freq points over the same range; nb_k is the Keplerian ceil(noverlap / (0.5 q_circ(f_k))) with q_circ from
    Kepler's third law in SI units; nb_k is monotone; the descriptor marks the kind of grid by the sign of h."""
    t = 2000.0 + np.arange(0.0, 2 * 27.4, 1.0 / 48.0)           # 2 continuous sectors, 30-min cadence
    rho = 1.7
    g0 = orc.grid(cfg, t, rho)
    f0, nb0 = orc.freqs(cfg, g0)
    cu = orc.default_config(uniform_freq=1)
    gu = orc.grid(cu, t, rho)
    fu, nbu = orc.freqs(cu, gu)
    assert gu["status"] == 0 and gu["h"] < 0 < g0["h"] and gu["u0"] == 1.0 / g0["p_max"]
    for k in ("t_ref", "baseline", "p_min", "p_max", "c_q", "nb_max"):
        assert gu[k] == g0[k]
    # arithmetic progression over the same range
    assert fu[0] == 1.0 / g0["p_max"] and fu[0] == pytest.approx(f0[0], rel=1e-15)
    assert fu[-1] <= (1.0 / g0["p_min"]) * (1 + 1e-12)
    assert fu[-1] + (-gu["h"]) > 1.0 / g0["p_min"]
    assert np.allclose(np.diff(fu), -gu["h"], rtol=1e-9) and np.all(np.diff(fu) > 0)
    assert fu.size == gu["n_freq"] == int(math.floor((1.0 / g0["p_min"] - fu[0]) / -gu["h"])) + 1
    # its step = the finest step of the GPU grid (at the low-frequency end): 3 u0^2 h to first order
    assert -gu["h"] == pytest.approx(f0[1] - f0[0], rel=3.0 * g0["h"] / g0["u0"])
    assert -gu["h"] < np.diff(f0).min() * (1 + 1e-12)
    assert fu.size > 3 * f0.size                                 # uniform steps need many more points
    # Keplerian nb at f_k, from Kepler III in SI units (exact ceil except within 1e-9 of an integer)
    q_lo = 0.5 / (math.pi * a_over_r(1.0 / fu, rho))
    x = 3.0 / q_lo
    safe = np.abs(x - np.round(x)) > 1e-6
    assert safe.mean() > 0.999 and np.array_equal(nbu[safe], np.ceil(x[safe]).astype(np.int32))
    assert nbu[0] == gu["nb_max"] and nbu[-1] == 38 and np.all(np.diff(nbu) <= 0)
    # capped: exactly M points, both ends kept
    for M in (80000, 1000, 2):
        cm = orc.default_config(uniform_freq=1, max_freq=M)
        gm = orc.grid(cm, t, rho)
        fm, nbm = orc.freqs(cm, gm)
        if gu["n_freq"] <= M:
            assert gm.tobytes() == gu.tobytes()
            continue
        assert fm.size == gm["n_freq"] == M and fm[0] == fu[0]
        assert fm[-1] == pytest.approx(1.0 / g0["p_min"], rel=1e-13)
        assert np.allclose(np.diff(fm), (1.0 / g0["p_min"] - fm[0]) / (M - 1), rtol=1e-9)
        assert np.all(np.diff(nbm) <= 0) and nbm[0] == gu["nb_max"] and nbm[-1] == 38
    # the comparison workload as SURVEY.md 8(f) words it: uniform, <= 80,000 frequencies, P <= 56 d; context of
    # PAPER.md:59 ("up to ~10 times more frequencies" on the GPU grid) on the longest baseline
    comp = orc.default_config(uniform_freq=1, max_period_days=56.0, max_freq=80000)
    t40 = 2000.0 + np.arange(0.0, 40 * 27.4, 1.0 / 48.0)
    for rho_s, lo, hi in ((10.0, 5.0, 15.0), (1.0, 2.0, 4.0)):
        gc = orc.grid(comp, t40, rho_s)
        assert gc["n_freq"] == 80000 and gc["p_max"] == 56.0 and gc["h"] < 0
        assert lo < orc.grid(cfg, t40, rho_s)["n_freq"] / 80000 < hi
    # a step below 1e-9 f_max is refused
    tiny = orc.grid(orc.default_config(uniform_freq=1, samples_per_peak=1e9), t, rho)
    assert tiny["status"] == 3 and tiny["n_freq"] == 0
    # degenerate stars keep their status
    assert orc.grid(cu, t[:1], rho)["status"] == 1


def test_search_on_the_uniform_comparison_grid_recovers_an_injection(orc):
    """End to end on the frequency-uniform grid: the spectrum at index k is the spectrum of (f_k, nb_k) of that grid
    (brute force through sr_one), and the injected period of BASELINE.json configs[0] is found to within one step."""
    comp = orc.default_config(uniform_freq=1, max_freq=3000)
    b = synth.make_batch(1, n_stars=1)
    t, y, dy = b.star(0)
    out = orc.batch(comp, b.row_ptr, b.t, b.y, b.dy, b.rho, K=1, want_snr=True)
    g = out["grid"][0:1]
    f, nb = orc.freqs(comp, g)
    assert f.size == 3000 and g["h"][0] < 0
    tau, w, wy = orc.prep(t, y, dy, float(g["t_ref"][0]))[:3]
    M = orc.widths(comp)
    for k in (0, 1, 1499, 2999):
        sr, m, j = orc.sr_one(tau, w, wy, float(f[k]), int(nb[k]), M)[:3]
        assert out["sr"][k] == sr and out["m"][k] == m and out["j"][k] == j
    pk = out["peaks"][0][0]
    truth = b.truth[0]
    assert pk["freq"] == f[pk["k"]]
    n = round(pk["period"] / truth["period"]) if pk["period"] > truth["period"] else 1
    assert abs(1.0 / pk["period"] - 1.0 / (n * truth["period"])) < 2.0 * -g["h"][0]


def test_grid_invariances(orc, cfg):
    t, *_ = synth.make_star(3, 11)
    g = orc.grid(cfg, t, 1.7)
    g2 = orc.grid(cfg, t + 4096.0, 1.7)   # time zero point is arbitrary
    assert abs(int(g2["n_freq"]) - int(g["n_freq"])) <= 1
    assert g2["p_max"] == pytest.approx(g["p_max"], rel=1e-11)
    assert g2["u0"] == pytest.approx(g["u0"], rel=1e-11)


def test_degenerate_stars(orc, cfg):
    assert orc.grid(cfg, np.array([]))["status"] == 1
    assert orc.grid(cfg, np.array([5.0]))["status"] == 1
    g = orc.grid(cfg, 2000.0 + 0.02 * np.arange(20))   # 0.4 d of data: P_max < P_min
    assert g["status"] == 3 and g["n_freq"] == 0


def test_widths(orc):
    assert list(orc.widths(orc.default_config())) == list(range(3, 12))
    # by hand: J = floor(ln 4 / ln 1.1) + 1 = 15 rungs, 3 * 1.1^14 = 11.39 -> 11
    assert math.floor(math.log(4.0) / math.log(1.1)) + 1 == 15
    assert list(orc.widths(orc.default_config(dlogq=0.5))) == [3, 5, 7, 10]
