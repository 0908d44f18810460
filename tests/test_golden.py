"""Regression pins from tests/golden/config1_oracle.txt (written by tests/golden/make_golden.py, which calls only
oracle/).  CPU: the oracle still reproduces its stored values bit for bit.  GPU: the CUDA path agrees with them
(grid bit-exact, SR within 1e-4 of the peak, same top peak, identical per-peak counts)."""
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    d = {}
    for ln in open(os.path.join(HERE, "golden", "config1_oracle.txt")):
        if ln.startswith("#") or not ln.strip():
            continue
        k, *rest = ln.split()
        d[k] = rest
    return d


def test_oracle_reproduces_golden(orc, cfg):
    from paper_2302_01293_b200 import synth
    gold = _golden()
    b = synth.make_batch(1)
    ob = orc.batch(cfg, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True)
    g = ob["grid"][0]
    assert int(gold["n_points"][0]) == b.n_points and int(gold["n_freq"][0]) == g["n_freq"]
    for k in ("t_ref", "baseline", "p_min", "p_max", "c_q", "u0", "h"):
        assert float.fromhex(gold[f"grid.{k}"][0]) == float(g[k]), k
    assert float.fromhex(gold["sr.max"][0]) == float(ob["sr"].max())
    assert int(gold["sr.argmax"][0]) == int(np.argmax(ob["sr"]))
    assert float.fromhex(gold["snr.max"][0]) == float(ob["snr"].max())
    p0 = dict(kv.split("=") for kv in gold["peak0"])
    assert int(p0["k"]) == ob["peaks"][0][0]["k"] and abs(float.fromhex(p0["period"]) - 3.7) < 0.02


@pytest.mark.gpu
def test_gpu_matches_golden():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2302_01293_b200 import build, bls, synth
    build.build()
    gold = _golden()
    b = synth.make_batch(1)
    ctx = bls.QlpBls(top_k=3)
    try:
        dev = bls.upload(b)
        grid, fp, tf, _ = ctx.grid(dev[0], dev[1], dev[4], dev[5])
        g = bls.grid_to_numpy(grid)[0]
        assert tf == int(gold["n_freq"][0]) and g["nb_max"] == int(gold["nb_max"][0])
        for k in ("t_ref", "baseline", "p_min", "p_max", "c_q", "u0", "h"):
            assert float.fromhex(gold[f"grid.{k}"][0]) == float(g[k]), k
        sr, best = ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        snr, peaks = ctx.snr(dev[0], dev[1], dev[2], dev[3], grid, fp, sr, best)
        stats = bls.stats_to_numpy(ctx.peak_stats(dev[0], dev[1], dev[2], dev[3], peaks), 3)
        pk = bls.peaks_to_numpy(peaks, 3)
        srh = sr.cpu().numpy()
        peak = float.fromhex(gold["sr.max"][0])
        assert abs(float(srh.max()) - peak) <= 1e-4 * peak and int(np.argmax(srh)) == int(gold["sr.argmax"][0])
        assert abs(float(srh.astype(np.float64).sum()) - float.fromhex(gold["sr.sum"][0])) <= 1e-4 * peak * srh.size
        assert abs(float(snr.max()) - float.fromhex(gold["snr.max"][0])) <= 5e-4 * float.fromhex(gold["snr.max"][0]) + 1e-3
        for r in range(3):
            p = dict(kv.split("=") for kv in gold[f"peak{r}"])
            assert pk[0][r]["k"] == int(p["k"]) and pk[0][r]["m"] == int(p["m"]) and pk[0][r]["j"] == int(p["j"])
            assert pk[0][r]["period"] == float.fromhex(p["period"]) and pk[0][r]["t0"] == float.fromhex(p["t0"])
            for k in ("n_in", "n_before", "n_after", "n_transits"):
                assert stats[0][r][k] == int(p[k]), (r, k)
    finally:
        ctx.close()
