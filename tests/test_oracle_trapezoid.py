"""Pins of oracle O8, the trapezoid fit (O8).

The oracle is pinned to things other than itself:
  * closed form: noise-free data drawn from a trapezoid are fitted back to the generating parameters, chi2 -> 0;
  * library routines: chi2 and the linear part (z, depth) at the oracle's solution equal numpy.linalg.lstsq on a
    design matrix whose shape column comes from numpy.interp over the four contact points (the definition of a
    trapezoid by its contacts, not the oracle's branchy formula);
  * optimality: scipy's Nelder-Mead from several starts on that independent chi2 finds nothing better;
  * invariants: affine maps of y and shifts of t move (z, depth, chi2, T0) the way the model says;
  * the bounds of PAPER.md:44 (q in [0, 1], q_in in [0, 0.5]) and the +-2 duration data window.
"""
import numpy as np
import pytest
from scipy.optimize import minimize

from oracle import oracle


def phase_dt(t, P, T0):
    x = (t - T0) / P
    return (x - np.floor(x + 0.5)) * P


def trapezoid_curve(t, P, T0, delta, q, q_in, z):
    """Trapezoid by its contact points: 1st/4th contact at +-D/2, 2nd/3rd at +-(D/2 - q_in D)."""
    dt = phase_dt(t, P, T0)
    D = q * P
    t1, t2 = -0.5 * D, -0.5 * D + q_in * D
    return z - delta * np.interp(dt, [t1, t2, -t2, -t1], [0.0, 1.0, 1.0, 0.0])


def independent_chi2(t, y, dy, P, t0_bls, D0, c, q, q_in):
    dt = phase_dt(t, P, t0_bls)
    sel = np.abs(dt) <= 2.0 * D0
    dt, yy, sw = dt[sel], y[sel], 1.0 / dy[sel]
    D = q * P
    t1, t2 = -0.5 * D, -0.5 * D + q_in * D
    if q_in > 0 and D > 0:
        sh = np.interp(dt - c, [t1, t2, -t2, -t1], [0.0, 1.0, 1.0, 0.0])
    else:
        sh = (np.abs(dt - c) < 0.5 * D).astype(float)
    A = np.stack([np.ones_like(sh), -sh], axis=1) * sw[:, None]
    sol = np.linalg.lstsq(A, yy * sw, rcond=None)[0]
    r = A @ sol - yy * sw
    return float(r @ r), sol, int(sel.sum())


def make_case(q_in, noise, seed, P=2.5, q=0.03, delta=0.01, z=1.0003, T0=1.234, days=27.0):
    rng = np.random.default_rng(seed)
    t = np.arange(0.0, days, 200.0 / 86400.0)
    dy = np.full_like(t, max(noise, 1e-3))
    y = trapezoid_curve(t, P, T0, delta, q, q_in, z) + noise * rng.standard_normal(t.size)
    m, nb = 5, 150                                   # BLS guess: q0 = 1/30, epoch off by 0.15 durations
    return dict(t=t, y=y, dy=dy, P=P, m=m, nb=nb, t0_bls=T0 + 0.15 * q * P, truth=(T0, delta, q, q_in, z))


@pytest.mark.parametrize("q_in", [0.05, 0.2, 0.3, 0.45])
def test_noise_free_trapezoid_is_recovered(q_in):
    c = make_case(q_in, 0.0, 0)
    r = oracle.trapezoid_fit(c["t"], c["y"], c["dy"], 1.0 / c["P"], c["m"], c["nb"], c["t0_bls"])
    T0, delta, q, qi, z = c["truth"]
    assert r["status"] == 0 and r["n_eval"] <= 605
    assert abs(r["t0"] - T0) < 1e-7
    assert abs(r["q"] - q) < 1e-7 and abs(r["q_in"] - qi) < 1e-5
    # The search (O8, round-2 reading) stops when no neighbour lowers chi2 by more than 1e-12 G, i.e. at
    # chi2 ~ 1e-11 G: the linear parameters are then within a few 1e-6 of their scale (depth 0.01, level 1).
    assert abs(r["depth"] - delta) < 5e-8 and abs(r["z"] - z) < 5e-9
    assert r["chi2"] < 1e-9 * r["chi2_init"]


@pytest.mark.parametrize("q_in,noise,seed", [(0.2, 0.001, 1), (0.05, 0.001, 2), (0.45, 0.003, 3), (0.3, 0.003, 4)])
def test_chi2_and_linear_part_match_lstsq_and_nelder_mead_finds_nothing_better(q_in, noise, seed):
    c = make_case(q_in, noise, seed)
    t, y, dy, P = c["t"], c["y"], c["dy"], c["P"]
    r = oracle.trapezoid_fit(t, y, dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"])
    q0 = c["m"] / c["nb"]
    D0 = q0 * P
    chi2, sol, n_sel = independent_chi2(t, y, dy, P, c["t0_bls"], D0, r["t0"] - c["t0_bls"], r["q"], r["q_in"])
    assert r["n_fit"] == n_sel
    assert r["chi2"] == pytest.approx(chi2, rel=1e-9)
    assert r["z"] == pytest.approx(sol[0], rel=1e-9) and r["depth"] == pytest.approx(sol[1], rel=1e-7)
    at = oracle.trapezoid_chi2_at(t, y, dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"], r["t0"] - c["t0_bls"], r["q"], r["q_in"])
    assert at[0] == pytest.approx(chi2, rel=1e-9) and at[1] == pytest.approx(sol[1], rel=1e-7)
    assert r["chi2"] <= r["chi2_init"]
    assert 0.0 <= r["q"] <= 1.0 and 0.0 <= r["q_in"] <= 0.5 and abs(r["t0"] - c["t0_bls"]) <= D0

    def fun(th):
        return independent_chi2(t, y, dy, P, c["t0_bls"], D0, float(np.clip(th[0], -1, 1)) * D0,
                                float(np.clip(th[1], 0, 1 / q0)) * q0, float(np.clip(th[2], 0, 0.5)))[0]
    best = min(minimize(fun, x0, method="Nelder-Mead", options=dict(xatol=1e-7, fatol=1e-12, maxiter=3000)).fun
               for x0 in ([0.0, 1.0, 0.25], [0.1, 0.9, 0.1], [-0.1, 1.1, 0.4]))
    assert r["chi2"] <= best * (1.0 + 1e-4)


def test_affine_map_of_y_and_shift_of_t():
    c = make_case(0.25, 0.002, 7)
    t, y, dy, P = c["t"], c["y"], c["dy"], c["P"]
    r0 = oracle.trapezoid_fit(t, y, dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"])
    a, b = 4.0, -2.5                                     # powers of two / exactly representable: same path
    r1 = oracle.trapezoid_fit(t, a * y + b, dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"])
    assert r1["q"] == pytest.approx(r0["q"], rel=1e-6) and r1["q_in"] == pytest.approx(r0["q_in"], abs=1e-6)
    assert r1["depth"] == pytest.approx(a * r0["depth"], rel=1e-6)
    assert r1["z"] == pytest.approx(a * r0["z"] + b, rel=1e-9)
    assert r1["chi2"] == pytest.approx(a * a * r0["chi2"], rel=1e-9)
    r2 = oracle.trapezoid_fit(t + 64.0, y, dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"] + 64.0)
    assert r2["t0"] == pytest.approx(r0["t0"] + 64.0, abs=1e-7)
    assert r2["chi2"] == pytest.approx(r0["chi2"], rel=1e-7)


def test_box_and_v_shapes_hit_the_bounds_of_q_in():
    cadence = 200.0 / 86400.0
    # V-shaped data: the fit ends next to the upper bound 0.5 (a flat bottom shorter than the cadence is all
    # the sampled data leave open) and never beyond it
    c = make_case(0.5, 0.0, 0)
    r = oracle.trapezoid_fit(c["t"], c["y"], c["dy"], 1.0 / c["P"], c["m"], c["nb"], c["t0_bls"])
    assert 0.49 <= r["q_in"] <= 0.5 and (1.0 - 2.0 * r["q_in"]) * r["q"] * c["P"] <= 2.0 * cadence
    assert r["chi2"] < 1e-9 * r["chi2_init"]
    # box-shaped data: ingress shorter than the cadence is all the data can say
    c = make_case(0.0, 0.0, 0)
    r = oracle.trapezoid_fit(c["t"], c["y"], c["dy"], 1.0 / c["P"], c["m"], c["nb"], c["t0_bls"])
    assert 0.0 <= r["q_in"] and r["q_in"] * r["q"] * c["P"] <= 2.0 * cadence
    assert r["depth"] == pytest.approx(0.01, rel=1e-3)


def test_too_few_points_and_flat_data():
    t = np.array([0.0, 1.0, 2.0, 3.0, 4.0, 5.0])
    y = np.ones(6)
    dy = np.full(6, 0.1)
    r = oracle.trapezoid_fit(t, y, dy, 1.0 / 2.9, 3, 300, 0.45)      # window 2 q0 P = 0.058 d: no point inside
    assert r["status"] == 2 and r["n_fit"] < 5 and r["q"] == pytest.approx(0.01)
    t = np.arange(0.0, 10.0, 0.01)
    y = np.full_like(t, 3.0)
    dy = np.full_like(t, 0.5)
    r = oracle.trapezoid_fit(t, y, dy, 1.0 / 2.0, 5, 100, 1.0)      # constant series: nothing to fit
    assert r["status"] == 0 and r["depth"] == 0.0 and r["z"] == pytest.approx(3.0) and r["chi2"] == 0.0
    assert r["q"] == pytest.approx(0.05) and r["q_in"] == 0.25      # no move was accepted


@pytest.mark.parametrize("q_in,noise,seed", [(0.2, 0.001, 1), (0.05, 0.001, 2), (0.45, 0.003, 3), (0.3, 0.003, 4),
                                             (0.25, 0.02, 5), (0.25, 0.05, 6)])
def test_search_path_is_insensitive_to_rounding_noise(q_in, noise, seed):
    """The rule of the search (neighbour within tol of the best, move only if chi2 drops by more than tol = 1e-12 G)
    exists so that rounding noise cannot decide a move.  An affine map of y by numbers that are NOT powers of two
    changes every rounding error of every sum; the search must take the same path: same number of evaluations, same
    (T0, q, q_in) to 1e-9 -- also on data that are almost pure noise (the last two cases), where chi2 is flat."""
    c = make_case(q_in, noise, seed)
    t, y, dy, P = c["t"], c["y"], c["dy"], c["P"]
    r0 = oracle.trapezoid_fit(t, y, dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"])
    for a, b in ((3.0, 0.7), (1.0 / 7.0, -11.3)):
        r1 = oracle.trapezoid_fit(t, a * y + b, a * dy, 1.0 / P, c["m"], c["nb"], c["t0_bls"])
        assert r1["n_eval"] == r0["n_eval"]
        assert abs(r1["t0"] - r0["t0"]) <= 1e-9 * c["m"] / c["nb"] * P
        assert abs(r1["q"] - r0["q"]) <= 1e-9 * r0["q"] and abs(r1["q_in"] - r0["q_in"]) <= 1e-9
        assert r1["chi2"] == pytest.approx(r0["chi2"], rel=1e-9)
        assert r1["depth"] == pytest.approx(a * r0["depth"], rel=1e-6)
