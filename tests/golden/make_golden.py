"""Writes tests/golden/config1_oracle.txt: the oracle's results for BASELINE.json configs[0] (one star, one
27.4-d sector at 30-min cadence, injected 3.7-d box transit; seed 0).  Calls ONLY oracle/ and the input generator.
The paper (arXiv:2302.01293) prints no spectrum or S/N value, so these are regression values of the oracle, not
paper values; the oracle itself is pinned by tests/test_oracle_*.py.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from paper_2302_01293_b200 import synth  # noqa: E402


def main():
    cfg = orc.default_config()
    b = synth.make_batch(1)
    ob = orc.batch(cfg, b.row_ptr, b.t, b.y, b.dy, b.rho, K=3, want_snr=True)
    g = ob["grid"][0]
    t, y, dy = b.star(0)
    lines = ["# oracle results for BASELINE.json configs[0], seed 0 (written by tests/golden/make_golden.py)",
             "# grid: PAPER.md:19,23,35 (DESIGN.md O1); SR: PAPER.md:37 (O4); S/N: PAPER.md:37-42 (O5); peaks: PAPER.md:44 (O6);",
             "# statistics: PAPER.md:53 (O7).  Doubles are printed as C99 hex floats (exact).",
             f"n_points {t.size}",
             f"n_freq {int(g['n_freq'])}",
             f"nb_max {int(g['nb_max'])}"]
    for k in ("t_ref", "baseline", "p_min", "p_max", "c_q", "u0", "h"):
        lines.append(f"grid.{k} {float(g[k]).hex()}")
    lines.append(f"sr.max {float(ob['sr'].max()).hex()}")
    lines.append(f"sr.argmax {int(np.argmax(ob['sr']))}")
    lines.append(f"sr.sum {float(np.sum(ob['sr'])).hex()}")
    lines.append(f"snr.max {float(ob['snr'].max()).hex()}")
    for r, p in enumerate(ob["peaks"][0]):
        st = orc.peak_statistics(t, y, dy, float(p["freq"]), int(p["m"]), int(p["nb"]), float(p["t0"]))
        lines.append(f"peak{r} k={int(p['k'])} m={int(p['m'])} j={int(p['j'])} nb={int(p['nb'])} "
                     f"period={float(p['period']).hex()} t0={float(p['t0']).hex()} snr={float(p['snr']).hex()} "
                     f"n_in={int(st['n_in'])} n_before={int(st['n_before'])} n_after={int(st['n_after'])} "
                     f"n_transits={int(st['n_transits'])}")
    with open(os.path.join(HERE, "config1_oracle.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
