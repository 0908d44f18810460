"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/qlp_bls.h declares; struct layouts match the Python binding.  No compute calls (no GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2302_01293_b200 import build, bls
    build.build()
    return bls.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "qlp_bls.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qlp_bls_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    from paper_2302_01293_b200 import bls
    names = declared_symbols()
    assert {"qlp_bls_create", "qlp_bls_grid", "qlp_bls_spectrum", "qlp_bls_snr", "qlp_bls_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in qlp_bls.h but not exported"
    assert sorted(bls.EXPORTS) == names


def test_struct_layouts(lib):
    from paper_2302_01293_b200 import bls
    assert bls.GRID_DTYPE.itemsize == 72
    assert bls.PEAK_DTYPE.itemsize == 64
    assert bls.STATS_DTYPE.itemsize == 32 and bls.TRAP_DTYPE.itemsize == 72 and bls.PINK_DTYPE.itemsize == 48
    cfg = bls.default_config()
    assert cfg.struct_bytes == C.sizeof(bls.Config) == 88
    # the paper's parameters: PAPER.md:35 (samples_per_peak=2, dlogq=0.1, noverlap=3), :19, :23, :7
    assert (cfg.samples_per_peak, cfg.dlogq, cfg.noverlap) == (2.0, 0.1, 3)
    assert (cfg.qmin_fac, cfg.qmax_fac, cfg.a_over_rstar_min, cfg.sector_days) == (0.5, 2.0, 2.0, 27.4)
    assert (cfg.max_period_days, cfg.max_freq) == (0.0, 0)       # the paper's GPU grid: no caps (O1.10)


def test_strerror_and_bad_args(lib):
    assert lib.qlp_bls_strerror(0) == b"ok"
    assert lib.qlp_bls_strerror(-4) == b"unsupported"
    # NULL arguments are rejected before any CUDA call
    assert lib.qlp_bls_create(None, None) == -1
    from paper_2302_01293_b200 import bls
    cfg = bls.default_config(top_k=99)
    h = C.c_void_p()
    assert lib.qlp_bls_create(C.byref(cfg), C.byref(h)) == -1
    for bad in (dict(max_freq=1), dict(max_freq=-5), dict(max_period_days=-1.0), dict(flags=4), dict(reserved_=1)):
        assert lib.qlp_bls_create(C.byref(bls.default_config(**bad)), C.byref(h)) == -1
    cfg = bls.default_config(a_over_rstar_min=0.5)  # boxes would be wider than the histogram
    assert lib.qlp_bls_create(C.byref(cfg), C.byref(h)) == -1
    assert lib.qlp_bls_destroy(None) == 0


def test_product_has_no_oracle_import():
    """The product path must not import, read or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2302_01293_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "qlp_oracle" not in txt, fn


def test_no_cuda_means_loud_failure(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2302_01293_b200 import bls
    with pytest.raises(bls.QlpBlsError):
        bls.QlpBls()
