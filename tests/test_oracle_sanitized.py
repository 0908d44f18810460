"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (gcc): every routine of oracle/qlp_oracle.c runs on
a small injected star, on the degenerate stars (1, 2 points; constant; a gap longer than a sector) and on the test
helpers, in a child process that has libasan preloaded.  Any out-of-bounds access, signed overflow, bad shift or
invalid float-to-int conversion aborts the child.  The child also checks that the instrumented build gives the same
peak table as the normal one (the sanitizers do not change FP64 arithmetic at -ffp-contract=off)."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r'''
import sys
import numpy as np
sys.path.insert(0, sys.argv[1])
from oracle import oracle as O
from paper_2302_01293_b200 import synth
assert O.sanitized() and O.build().endswith("_san.so")
cfg = O.default_config()
b = synth.make_batch(1, n_stars=1)
t, y, dy = b.star(0)
out = O.batch(cfg, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True, threads=2)
pk = out["peaks"][0]
np.save(sys.argv[2], out["peaks"])
g = out["grid"][0:1]
# every single-purpose routine on the best peak
p = pk[0]
O.widths(cfg); O.cbrt_det(2.0); O.sturges(4489)
f, nb = O.freqs(cfg, g)
tau, w, wy = O.prep(t, y, dy, float(g["t_ref"][0]))[:3]
O.bins(float(f[0]), int(nb[0]), tau); O.bins(float(f[-1]), int(nb[-1]), tau)
O.sr_one(tau, w, wy, float(f[-1]), int(nb[-1]), O.widths(cfg))
ks = np.array([0, 1, f.size // 2, f.size - 1], dtype=np.int64)
sr_s, m_s, j_s = O.spectrum_samples(cfg, g, t, y, dy, ks)[:3]
O.box_values(cfg, g, t, y, dy, ks, m_s, j_s)
O.snr(f, out["sr"][:f.size]); O.snr(f[:3], out["sr"][:3]); O.snr(f[:1], out["sr"][:1])
O.peak_indices(np.array([1.0, 1.0, 0.5, 1.0, 2.0, 2.0]), 3); O.peak_indices(np.zeros(0), 3)
O.peak_record(cfg, g, t, y, dy, int(p["k"]), float(p["snr"]))
O.peak_statistics(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]))
fit = O.trapezoid_fit(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]))
O.trapezoid_chi2_at(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]), 0.0, float(fit["q"]),
                    float(fit["q_in"]))
O.pink_noise(t, y, float(p["freq"]), float(fit["t0"]), float(fit["depth"]), float(fit["q"]), float(fit["q_in"]),
             float(fit["z"]), float(p["snr"]))
# degenerate stars through the whole chain: 1 point, 2 points, constant, two sectors with a long gap, 3 close points
ts = synth.sector_times(0, 1800.0)
stars = [(ts[:1], np.ones(1), np.ones(1)), (ts[:2], np.ones(2), np.ones(2)),
         (ts, np.ones(ts.size), np.full(ts.size, 1e-3)),
         (np.concatenate([ts[:300], ts[:300] + 400.0]), np.r_[np.ones(300), np.zeros(300)], np.full(600, 1e-3)),
         (ts[:3], np.array([1.0, 0.9, 1.0]), np.full(3, 1e-3))]
bb = synth.from_arrays(stars)
o2 = O.batch(cfg, bb.row_ptr, bb.t, bb.y, bb.dy, bb.rho, K=3, want_snr=True, threads=2)
for s in range(bb.n_stars):
    tt, yy, dd = bb.star(s)
    for r in range(3):
        q = o2["peaks"][s][r]
        if q["k"] < 0:
            continue
        O.peak_statistics(tt, yy, dd, float(q["freq"]), int(q["m"]), int(q["nb"]), float(q["t0"]))
        ft = O.trapezoid_fit(tt, yy, dd, float(q["freq"]), int(q["m"]), int(q["nb"]), float(q["t0"]))
        O.pink_noise(tt, yy, float(q["freq"]), float(ft["t0"]), float(ft["depth"]), float(ft["q"]), float(ft["q_in"]),
                     float(ft["z"]), float(q["snr"]))
# the comparison grid's caps
cc = O.default_config(max_period_days=12.0, max_freq=500)
O.batch(cc, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True, threads=1)
cu = O.default_config(uniform_freq=1, max_period_days=12.0, max_freq=500)   # O1.10c: equal steps in frequency
O.batch(cu, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True, threads=1)
print("sanitized oracle ok")
'''


def _libasan():
    try:
        path = subprocess.run(["gcc", "-print-file-name=libasan.so"], check=True, capture_output=True,
                              text=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return None
    return os.path.realpath(path) if os.path.isabs(path) and os.path.exists(path) else None


def test_oracle_runs_clean_under_asan_and_ubsan(orc, cfg, tmp_path):
    asan = _libasan()
    if asan is None:
        pytest.skip("gcc's libasan is not installed")
    env = dict(os.environ, QLP_ORACLE_SANITIZE="1", LD_PRELOAD=asan, OMP_NUM_THREADS="2",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    out = tmp_path / "peaks.npy"
    r = subprocess.run([sys.executable, "-c", CHILD, ROOT, str(out)], env=env, capture_output=True, text=True,
                       timeout=600)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
    from paper_2302_01293_b200 import synth
    b = synth.make_batch(1, n_stars=1)
    want = orc.batch(cfg, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True)["peaks"]
    assert np.load(out).tobytes() == want.tobytes()
