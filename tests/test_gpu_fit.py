"""O8 parity on the GPU: trapezoid fit of every peak against the oracle, through the C ABI.

Both sides run the same compass search in FP64 on the same points.  The window membership is an integer decision
taken with the same unfused operations (n_fit: bit-exact).  The search rule (O8, round-2 reading) takes no
decision that rounding noise could flip: a sweep evaluates the six neighbours, takes the first one within
tol = 1e-12 G of the best and moves only if chi2 drops by more than tol.  So both implementations follow the SAME path
although they add the points up in different orders: the same number of evaluations, parameters equal to 1e-6,
chi2 to 1e-9 -- on every fit, noise peaks with flat chi2 included.  The GPU's result is also validated on its own:
the ORACLE's chi2, depth and level evaluated AT the GPU's parameters are the GPU's."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2302_01293_b200 import build, bls
    build.build()
    return bls


def run_search(gpu, ctx, b):
    dev = gpu.upload(b)
    grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
    sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
    _, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best, want_snr=False)
    fits = gpu.fits_to_numpy(ctx.trapezoid_fit(dev[0], dev[1], dev[2], dev[3], peaks), ctx.top_k)
    return gpu.peaks_to_numpy(peaks, ctx.top_k), fits


def compare(orc, star, g, o, p):
    """g: GPU fit, o: oracle fit, p: the peak."""
    t, y, dy = star
    D0 = p["m"] / p["nb"] * p["period"]
    assert g["n_fit"] == o["n_fit"] and g["status"] == o["status"]
    if o["status"] != 0:
        assert g["t0"] == o["t0"] and g["q"] == o["q"] and g["q_in"] == o["q_in"]
        return
    floor = 1e-12 * o["chi2_init"]
    assert abs(g["chi2_init"] - o["chi2_init"]) <= 1e-9 * o["chi2_init"]
    # the same path: same number of chi2 evaluations, same end point
    assert int(g["n_eval"]) == int(o["n_eval"]), (int(g["n_eval"]), int(o["n_eval"]))
    assert abs(g["t0"] - o["t0"]) <= 1e-6 * D0
    assert abs(g["q"] - o["q"]) <= 1e-6 * o["q"] and abs(g["q_in"] - o["q_in"]) <= 1e-6
    assert abs(g["chi2"] - o["chi2"]) <= 1e-9 * o["chi2"] + floor
    scale = max(abs(o["depth"]), 1e-12)
    assert abs(g["depth"] - o["depth"]) <= 1e-6 * scale and abs(g["z"] - o["z"]) <= 1e-6 * scale + 1e-12 * abs(o["z"])
    # the GPU's parameters are valid on their own: the oracle's chi2, depth and level AT those parameters
    c2, depth, z = orc.trapezoid_chi2_at(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]),
                                         float(g["t0"] - p["t0"]), float(g["q"]), float(g["q_in"]))
    assert abs(g["chi2"] - c2) <= 1e-9 * c2 + floor
    assert abs(g["depth"] - depth) <= 1e-6 * max(abs(depth), 1e-12)
    assert g["chi2"] <= g["chi2_init"] and 0.0 <= g["q"] <= 1.0 and 0.0 <= g["q_in"] <= 0.5
    assert abs(g["t0"] - p["t0"]) <= D0 and g["n_eval"] <= 605


@pytest.mark.parametrize("config,ids", [(1, [0]), (2, list(range(40))), (4, [0, 1]), (5, [0, 1, 2, 3, 19, 28])])
def test_trapezoid_fit_matches_oracle(gpu, orc, config, ids):
    from paper_2302_01293_b200 import synth
    b = synth.make_batch(config, star_ids=np.array(ids))
    ctx = gpu.QlpBls(top_k=3)
    try:
        pk, fits = run_search(gpu, ctx, b)
        checked = 0
        for s in range(b.n_stars):
            t, y, dy = b.star(s)
            for r in range(ctx.top_k):
                p, g = pk[s][r], fits[s][r]
                if p["k"] < 0:
                    assert g["status"] == 1 and g["n_fit"] == 0
                    continue
                o = orc.trapezoid_fit(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]))
                compare(orc, (t, y, dy), g, o, p)
                checked += 1
        assert checked >= b.n_stars
        if config == 1:  # the injected transit of BASELINE.json configs[0]: the fit keeps the BLS depth within 2x
            assert fits[0][0]["status"] == 0 and 0.5 * pk[0][0]["depth"] < fits[0][0]["depth"] < 2.0 * pk[0][0]["depth"]
            assert fits[0][0]["chi2"] < fits[0][0]["chi2_init"]
    finally:
        ctx.close()


def test_trapezoid_fit_recovers_an_injected_trapezoid(gpu, orc):
    """End to end on the device: search + fit of a noise-free trapezoid gives back its shape."""
    from paper_2302_01293_b200 import synth
    t = synth.sector_times(0, 200.0)
    P, T0, q, q_in, depth = 3.1, t[0] + 1.3, 0.02, 0.3, 0.004
    x = (t - T0) / P
    dt = (x - np.floor(x + 0.5)) * P
    D = q * P
    sh = np.interp(dt, [-0.5 * D, -0.5 * D + q_in * D, 0.5 * D - q_in * D, 0.5 * D], [0.0, 1.0, 1.0, 0.0])
    y = 1.0 - depth * sh
    b = synth.from_arrays([(t, y, np.full(t.size, 1e-3))])
    ctx = gpu.QlpBls(top_k=1)
    try:
        pk, fits = run_search(gpu, ctx, b)
        p, g = pk[0][0], fits[0][0]
        n = round(p["period"] / P)                       # the search may settle on a multiple of P
        assert n >= 1 and abs(p["period"] - n * P) < 0.02 * P
        if n == 1:
            x0 = (g["t0"] - T0) / P
            # the grid period differs from P by a fraction of the grid step, which shifts the best epoch of the
            # first transit and smears the ingress: loose bounds here, the exact check is the oracle's below
            assert abs(x0 - round(x0)) * P < 0.25 * D
            assert abs(g["q"] * p["period"] - D) < 0.2 * D and abs(g["depth"] - depth) < 0.1 * depth
            assert abs(g["z"] - 1.0) < 1e-4 and 0.0 < g["q_in"] <= 0.5
            assert g["chi2"] < g["chi2_init"]
        dy = np.full(t.size, 1e-3)
        o = orc.trapezoid_fit(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]))
        compare(orc, (t, y, dy), g, o, p)
    finally:
        ctx.close()


def test_trapezoid_fit_empty_and_invalid(gpu):
    from paper_2302_01293_b200 import synth
    t = synth.sector_times(0, 1800.0)
    b = synth.from_arrays([(t[:1], np.zeros(1), np.ones(1)), (t, np.zeros(t.size), np.ones(t.size))])
    ctx = gpu.QlpBls()
    try:
        pk, fits = run_search(gpu, ctx, b)
        assert fits[0]["status"].tolist() == [1, 1, 1] and fits[0]["n_fit"].tolist() == [0, 0, 0]
        for r in range(ctx.top_k):                        # constant series: every peak fits depth 0 exactly
            if pk[1][r]["k"] >= 0 and fits[1][r]["status"] == 0:
                assert fits[1][r]["depth"] == 0.0 and fits[1][r]["chi2"] == 0.0
        import torch
        empty = torch.zeros(1, dtype=torch.int64, device="cuda")
        assert ctx.trapezoid_fit(empty, empty.double(), empty.double(), empty.double(), empty).numel() == 0
    finally:
        ctx.close()


def test_trapezoid_fit_on_random_irregular_stars(gpu, orc):
    """The fit, the statistics and the noise row on 60 random irregular stars (exponential spacings, gaps, outliers,
    5 to 4,000 points: windows of a handful of points, q at its bounds, peaks without a fit) against the oracle:
    the same strict comparison as above on every fit."""
    from paper_2302_01293_b200 import synth
    rng = np.random.default_rng(777)
    stars, rho = [], []
    for i in range(60):
        n = int(rng.integers(5, 4000))
        dt = rng.exponential(rng.choice([200.0, 600.0, 1800.0]) / 86400.0, n) + 1e-5
        for _ in range(int(rng.integers(0, 3))):
            dt[int(rng.integers(0, n))] += rng.choice([0.7, 3.0, 29.0])
        t = 2000.0 + np.cumsum(dt)
        dy = 1e-3 * 10.0 ** rng.uniform(-0.3, 0.3, n)
        y = rng.standard_normal(n) * dy + 1.0
        if i % 3 == 0:
            p = rng.uniform(0.4, 5.0)
            y -= rng.uniform(2e-3, 1e-2) * (np.mod(t - t[0], p) < 0.04 * p)
        stars.append((t, y, dy))
        rho.append(10.0 ** rng.uniform(-1.0, 1.0))
    b = synth.from_arrays(stars, rho=np.array(rho))
    ctx = gpu.QlpBls(top_k=3)
    try:
        pk, fits = run_search(gpu, ctx, b)
        dev = gpu.upload(b)
        checked = 0
        for s in range(b.n_stars):
            t, y, dy = b.star(s)
            for r in range(ctx.top_k):
                p, g = pk[s][r], fits[s][r]
                if p["k"] < 0:
                    assert g["status"] == 1 and g["n_fit"] == 0
                    continue
                o = orc.trapezoid_fit(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]))
                compare(orc, (t, y, dy), g, o, p)
                checked += 1
        assert checked > 120
    finally:
        ctx.close()
