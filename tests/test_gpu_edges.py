"""Edge cases and full-size checks of the CUDA path (run with -m gpu).

  * flags bit0 input validation (QLP_BLS_EVALIDATION);
  * a star that would need more phase bins than QLP_BLS_MAX_NB is skipped with status 4, its neighbours untouched;
  * the exact launch configuration bench.py times (BASELINE.json configs[1]: 1,000 stars) checked against the
    oracle on sampled (star, frequency) outputs and on whole spectra of a few stars.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SR_RTOL = 1e-4


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2302_01293_b200 import build, bls
    build.build()
    return bls


def test_validation_flag(gpu):
    from paper_2302_01293_b200 import synth
    t = synth.sector_times(0, 1800.0)
    rng = np.random.default_rng(0)
    good = (t, rng.standard_normal(t.size) * 1e-3, np.full(t.size, 1e-3))
    ctx = gpu.QlpBls(flags=1)
    try:
        dev = gpu.upload(synth.from_arrays([good, good]))
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)  # valid inputs pass
        t_bad = t.copy(); t_bad[100] = t_bad[99]                    # not strictly increasing
        dev = gpu.upload(synth.from_arrays([good, (t_bad, good[1], good[2])]))
        with pytest.raises(gpu.QlpBlsError, match="validation"):
            ctx.grid(dev[0], dev[1], dev[4], dev[5])
        dy_bad = good[2].copy(); dy_bad[5] = 0.0                    # dy must be > 0
        dev = gpu.upload(synth.from_arrays([good, (t, good[1], dy_bad)]))
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        with pytest.raises(gpu.QlpBlsError, match="validation"):
            ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        y_bad = good[1].copy(); y_bad[7] = np.nan
        dev = gpu.upload(synth.from_arrays([(t, y_bad, good[2])]))
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        with pytest.raises(gpu.QlpBlsError, match="validation"):
            ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
    finally:
        ctx.close()


def test_star_above_bin_cap_is_skipped(gpu, orc, cfg):
    """70 contiguous 30-min sectors and a very dense star: nb at the longest period exceeds QLP_BLS_MAX_NB."""
    from paper_2302_01293_b200 import synth
    t_long = np.concatenate([synth.sector_times(s, 1800.0) for s in range(70)])
    rng = np.random.default_rng(1)
    mk = lambda t: (t, rng.standard_normal(t.size) * 1e-3, np.full(t.size, 1e-3))
    t_short = synth.sector_times(0, 1800.0)
    b = synth.from_arrays([mk(t_short), mk(t_long), mk(t_short)], rho=np.array([1.0, 200.0, 1.0]))
    ctx = gpu.QlpBls()
    try:
        dev = gpu.upload(b)
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        g = gpu.grid_to_numpy(grid)
        go = orc.grid(cfg, t_long, 200.0)
        assert go["nb_max"] > 24576                       # the oracle's descriptor says so too
        assert g["status"].tolist() == [0, 4, 0] and g["n_freq"][1] == 0
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        snr, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best)
        pk = gpu.peaks_to_numpy(peaks, ctx.top_k)
        assert pk[1][0]["k"] == -1 and pk[0][0]["k"] >= 0 and pk[2][0]["k"] >= 0
        # the neighbours are unaffected: identical inputs -> identical spectra
        fpn = fp.cpu().numpy()
        s0 = sr[fpn[0]:fpn[1]].cpu().numpy()
        so, _, _ = orc.spectrum_star(cfg, orc.grid(cfg, t_short, 1.0), *b.star(0))
        assert np.abs(s0 - so).max() <= SR_RTOL * so.max()
    finally:
        ctx.close()


def test_bench_configuration_sampled(gpu, orc, cfg):
    """BASELINE.json configs[1] at full size (1,000 stars), in the launch configuration bench.py times."""
    from paper_2302_01293_b200 import synth
    b = synth.make_batch(2, n_stars=1000)
    ctx = gpu.QlpBls(top_k=3)
    try:
        dev = gpu.upload(b)
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        snr, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best)
        g = gpu.grid_to_numpy(grid)
        sr, fpn, snr = sr.cpu().numpy(), fp.cpu().numpy(), snr.cpu().numpy()
        pk = gpu.peaks_to_numpy(peaks, ctx.top_k)
        assert np.all(g["status"] == 0) and np.all(np.isfinite(sr)) and np.all(sr >= 0)
        M = orc.widths(cfg)
        rng = np.random.default_rng(2)
        # (a) 60 sampled (star, frequency) outputs, one oracle evaluation each
        for s in rng.integers(0, 1000, 20):
            t, y, dy = b.star(int(s))
            go = orc.grid(cfg, t, float(b.rho[s]))
            assert go.tobytes() == g[s].tobytes()
            tau, w, wy = orc.prep(t, y, dy, float(go["t_ref"]))
            peak = float(sr[fpn[s]:fpn[s + 1]].max())
            for k in rng.integers(0, int(go["n_freq"]), 3):
                f, nb = orc.freqs(cfg, go, int(k), int(k) + 1)
                v = orc.sr_one(tau, w, wy, float(f[0]), int(nb[0]), M)[0]
                assert abs(float(sr[fpn[s] + k]) - v) <= SR_RTOL * peak
        # (b) three whole stars: spectrum, S/N and top peak
        for s in (0, 499, 999):
            t, y, dy = b.star(s)
            go = orc.grid(cfg, t, float(b.rho[s]))
            so, mo, jo = orc.spectrum_star(cfg, go, t, y, dy)
            assert np.abs(sr[fpn[s]:fpn[s + 1]] - so).max() <= SR_RTOL * so.max()
            sn_o, _, _ = orc.snr(orc.freqs(cfg, go)[0], so)
            scale = np.abs(sn_o).max()
            assert np.abs(snr[fpn[s]:fpn[s + 1]] - sn_o).max() <= 5e-4 * scale + 1e-3
            top2 = np.sort(sn_o)[-2:]
            if top2[1] - top2[0] > 1e-3 * scale:
                assert pk[s][0]["k"] == int(np.argmax(sn_o))
        # (c) properties that hold at any size: injected transits are recovered at the right period
        inj = np.nonzero(b.truth["period"] > 0)[0]
        deep = [s for s in inj if b.truth["depth"][s] > 20 * np.median(b.star(int(s))[2]) / np.sqrt(50)]
        hits = 0
        for s in deep:
            ratio = pk[s][0]["period"] / b.truth["period"][s]
            hits += any(abs(ratio - h) < 0.02 * h for h in (0.5, 1.0, 2.0, 1 / 3, 3.0))
        assert len(deep) > 20 and hits >= 0.8 * len(deep), (hits, len(deep))
    finally:
        ctx.close()


@pytest.mark.parametrize("span", [0.6553, 0.66, 0.7, 0.8])
def test_tiny_grids(gpu, orc, cfg, span):
    """Baselines barely longer than 2 P_min: grids of one to a few dozen frequencies (Sturges N = 1, 2, ...)."""
    from paper_2302_01293_b200 import synth
    rng = np.random.default_rng(4)
    t = 100.0 + np.arange(0.0, span, 200.0 / 86400.0)
    b = synth.from_arrays([(t, rng.standard_normal(t.size) * 1e-3, np.full(t.size, 1e-3))])
    go = orc.grid(cfg, t, 1.0)
    ctx = gpu.QlpBls(top_k=3)
    try:
        dev = gpu.upload(b)
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        assert gpu.grid_to_numpy(grid)[0].tobytes() == go.tobytes()
        assert tf == int(go["n_freq"])
        if tf == 0:
            return
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        snr, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best)
        ob = orc.batch(cfg, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True)
        assert np.abs(sr.cpu().numpy() - ob["sr"]).max() <= SR_RTOL * ob["sr"].max()
        scale = np.abs(ob["snr"]).max()
        assert np.abs(snr.cpu().numpy() - ob["snr"]).max() <= 5e-4 * scale + 1e-3
        pk = gpu.peaks_to_numpy(peaks, 3)
        n_o = int((ob["peaks"][0]["k"] >= 0).sum())
        assert int((pk[0]["k"] >= 0).sum()) == n_o
        assert pk[0][0]["k"] == ob["peaks"][0][0]["k"] or abs(np.sort(ob["snr"])[-1] - np.sort(ob["snr"])[-2]) < 1e-3 * scale
    finally:
        ctx.close()


def test_star_above_point_cap_is_skipped(gpu):
    """QLP_BLS_MAX_POINTS = 2^22 points per star (32-bit fixed-point weights): longer series get status 5."""
    from paper_2302_01293_b200 import synth
    n = 1 << 22
    t_big = 100.0 + np.arange(n, dtype=np.float64) * 1e-4
    t_ok = synth.sector_times(0, 1800.0)
    rng = np.random.default_rng(6)
    b = synth.from_arrays([(t_big, np.zeros(n), np.ones(n)), (t_ok, rng.standard_normal(t_ok.size), np.ones(t_ok.size))])
    ctx = gpu.QlpBls()
    try:
        dev = gpu.upload(b)
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        g = gpu.grid_to_numpy(grid)
        assert g["status"].tolist() == [5, 0] and g["n_freq"][0] == 0 and g["n_freq"][1] > 0
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        _, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best, want_snr=False)
        pk = gpu.peaks_to_numpy(peaks, ctx.top_k)
        assert pk[0][0]["k"] == -1 and pk[1][0]["k"] >= 0
    finally:
        ctx.close()


def test_tile_classes_cover_every_star_and_frequency_once(gpu):
    """The per-class work counters of the fold/scan kernel (qlp_bls_fold_class_counters, what bench.py's roofline
    entry is built from): over a ragged production-shaped batch the evaluations of all tile classes add up to
    sum_s N_s n_freq,s exactly -- every (star, frequency) is folded once, by one tile of one class."""
    from paper_2302_01293_b200 import synth
    b = synth.make_batch(5, star_ids=np.arange(80))
    ctx = gpu.QlpBls(top_k=3)
    try:
        dev = gpu.upload(b)
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        g = gpu.grid_to_numpy(grid)
        ctx.fold_timing(True)
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        cc = ctx.fold_class_counters()
        n_timed, ms = ctx.fold_elapsed_ms()
        ctx.fold_timing(False)
        want = int((g["n_freq"].astype(np.int64) * np.diff(b.row_ptr)).sum())
        assert int(cc[:, 3].sum()) == want
        assert n_timed == 1 and ms > 0.0
        assert int((cc[:, 4] > 0).sum()) >= 4                      # several tile classes are populated
        assert np.all(cc[cc[:, 4] == 0][:, :4] == 0)               # a class without tiles did no work
        # the trapezoid fits count their work too while timing is on
        _, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best, want_snr=False)
        ctx.fold_timing(True)
        fits = gpu.fits_to_numpy(ctx.trapezoid_fit(dev[0], dev[1], dev[2], dev[3], peaks), ctx.top_k)
        pairs = ctx.fit_work()
        ctx.fold_timing(False)
        assert pairs > 0 and pairs <= int((fits["n_fit"].astype(np.int64) * fits["n_eval"]).sum())
    finally:
        ctx.close()
