"""Bounds-check build of the CUDA path (run with -m gpu): compute-sanitizer is closed on this GPU pool, so the library
can be built with -DQLP_BOUNDS_CHECK (`python -m paper_2302_01293_b200.build --check`): every guarded shared-memory and
workspace access of the fold, scan and fit kernels tests its index against the extent it must stay in and counts a
violation instead of performing the access (include/qlp_bls.h qlp_bls_debug_violations).  The cases below drive every
tile class (forced on a small star and natively on long ones), ragged production-shaped stars, degenerate stars and the
single-CTA and cluster fits through that build: no violation, and the results equal the normal build's bit for bit."""
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
    build.build_check()
    return bls


def _run(gpu, ctx, b, path=0, fit=True):
    dev = gpu.upload(b)
    ctx.debug_set_path(path)
    try:
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
    finally:
        ctx.debug_set_path(0)
    snr, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best)
    out = [sr.cpu().numpy().tobytes(), best.cpu().numpy().tobytes(), snr.cpu().numpy().tobytes(),
           peaks.cpu().numpy().tobytes()]
    if fit:
        fits = ctx.trapezoid_fit(dev[0], dev[1], dev[2], dev[3], peaks)
        out.append(fits.cpu().numpy().tobytes())
        out.append(ctx.pink_noise(dev[0], dev[1], dev[2], peaks, fits).cpu().numpy().tobytes())
    return out


def test_normal_build_reports_unsupported(gpu):
    ctx = gpu.QlpBls()
    try:
        with pytest.raises(gpu.QlpBlsError, match="unsupported"):
            ctx.debug_violations()
    finally:
        ctx.close()


def test_no_violation_in_any_tile_class_and_same_results(gpu):
    from paper_2302_01293_b200 import synth
    chk, ref = gpu.QlpBls(check=True, top_k=3), gpu.QlpBls(top_k=3)
    try:
        assert chk.debug_violations().sum() == 0
        rng = np.random.default_rng(12)
        cases = [(synth.make_batch(1), p) for p in range(0, 10)]                        # every class forced
        cases.append((synth.make_batch(5, star_ids=np.arange(60)), 0))                  # ragged, classes 0-5 natively
        cases.append((synth.make_batch(2, n_stars=40), 0))                              # single-CTA and cluster fits
        cases.append((synth.make_batch(4, n_stars=2), 0))                               # 13 sectors: large fit windows
        t_long = np.concatenate([synth.sector_times(s, 1800.0) for s in list(range(40)) + [42]])
        mk = lambda t: (t, rng.standard_normal(t.size) * 1e-3, 1e-3 * np.exp(0.1 * rng.standard_normal(t.size)))
        t_short = synth.sector_times(0, 1800.0)
        cases.append((synth.from_arrays([mk(t_short), mk(t_long), mk(t_short[:3]), mk(t_short[:0])],
                                        rho=np.array([1.0, 10.0, 1.0, 1.0])), 0))       # class 8 natively + degenerate
        for b, path in cases:
            got = _run(gpu, chk, b, path)
            v = chk.debug_violations()
            assert v.sum() == 0, (path, v)
            want = _run(gpu, ref, b, path)
            assert got == want                                                           # integer accumulators: bitwise
    finally:
        chk.close(); ref.close()
