"""ctypes wrapper around oracle/qlp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` leg may
import this module.  It imports nothing from the CUDA package except nothing at all: inputs come
in as numpy arrays.  See the header of qlp_oracle.c for what each routine follows in the paper.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qlp_oracle.c")
_LIB = os.path.join(_HERE, "libqlp_oracle.so")
_LIB_SAN = os.path.join(_HERE, "libqlp_oracle_san.so")


class Config(C.Structure):
    _fields_ = [("samples_per_peak", C.c_double), ("dlogq", C.c_double), ("noverlap", C.c_int32),
                ("uniform_freq", C.c_int32), ("qmin_fac", C.c_double), ("qmax_fac", C.c_double),
                ("a_over_rstar_min", C.c_double), ("sector_days", C.c_double),
                ("max_period_days", C.c_double), ("max_freq", C.c_int64)]


GRID_DTYPE = np.dtype([("t_ref", "f8"), ("baseline", "f8"), ("p_min", "f8"), ("p_max", "f8"),
                       ("c_q", "f8"), ("u0", "f8"), ("h", "f8"), ("n_freq", "i8"),
                       ("nb_max", "i4"), ("status", "i4")], align=True)
PEAK_DTYPE = np.dtype([("k", "i8"), ("freq", "f8"), ("period", "f8"), ("t0", "f8"), ("sr", "f8"),
                       ("snr", "f8"), ("q", "f8"), ("depth", "f8"), ("m", "i4"), ("j", "i4"),
                       ("nb", "i4"), ("status", "i4")], align=True)


STATS_DTYPE = np.dtype([("n_in", "i4"), ("n_before", "i4"), ("n_after", "i4"), ("n_transits", "i4"),
                        ("oot_level", "f8"), ("duration", "f8")], align=True)


def default_config(**kw) -> Config:
    """PAPER.md:19 (0.5-2.0 x q_circ), :23 (a = 2 R*), :35 (samples_per_peak=2, dlogq=0.1, noverlap=3), :7 (27.4 d)."""
    c = Config(2.0, 0.1, 3, 0, 0.5, 2.0, 2.0, 27.4, 0.0, 0)
    for k, v in kw.items():
        setattr(c, k, v)
    return c


def sanitized() -> bool:
    """QLP_ORACLE_SANITIZE=1: the same source built with AddressSanitizer + UndefinedBehaviorSanitizer (any report
    aborts).  The process must have libasan preloaded (tests/test_oracle_sanitized.py starts such a child)."""
    return os.environ.get("QLP_ORACLE_SANITIZE", "0") == "1"


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (FP64, no FMA contraction, OpenMP over stars)."""
    if sanitized():
        if force or not os.path.exists(_LIB_SAN) or os.path.getmtime(_LIB_SAN) < os.path.getmtime(_SRC):
            cmd = ["gcc", "-O1", "-g", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
                   "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer",
                   "-std=c11", "-o", _LIB_SAN, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
        return _LIB_SAN
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_cbrt_det.restype = C.c_double
        L.orc_cbrt_det.argtypes = [C.c_double]
        L.orc_sturges.restype = C.c_int32
        L.orc_sturges.argtypes = [C.c_int64]
        assert L.orc_sizeof_grid() == GRID_DTYPE.itemsize
        assert L.orc_sizeof_peak() == PEAK_DTYPE.itemsize
        assert L.orc_sizeof_config() == C.sizeof(Config)
        assert L.orc_sizeof_peak_stats() == STATS_DTYPE.itemsize
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f8(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def cbrt_det(x: float) -> float:
    return lib().orc_cbrt_det(float(x))


def sturges(n: int) -> int:
    return int(lib().orc_sturges(int(n)))


def widths(cfg: Config) -> np.ndarray:
    M = np.zeros(64, dtype=np.int32)
    n = lib().orc_widths(C.byref(cfg), _p(M))
    assert n > 0
    return M[:n].copy()


def grid(cfg: Config, t, rho: float = 1.0) -> np.ndarray:
    """O1 descriptor of one star -> 0-d structured array (GRID_DTYPE)."""
    t = _f8(t)
    g = np.zeros(1, dtype=GRID_DTYPE)
    lib().orc_grid(C.byref(cfg), C.c_int64(t.size), _p(t), C.c_double(rho), _p(g))
    return g[0]


def freqs(cfg: Config, g, k0: int = 0, k1: int | None = None):
    """O1.8: (f_k, nb_k) for k in [k0, k1)."""
    ga = np.array([g], dtype=GRID_DTYPE)
    if k1 is None:
        k1 = int(ga[0]["n_freq"])
    n = max(0, k1 - k0)
    f = np.zeros(n, dtype=np.float64)
    nb = np.zeros(n, dtype=np.int32)
    if n:
        lib().orc_freqs(C.byref(cfg), _p(ga), C.c_int64(k0), C.c_int64(k1), _p(f), _p(nb))
    return f, nb


def prep(t, y, dy, t_ref: float):
    """O2: (tau, w, w*ytilde)."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    n = t.size
    tau, w, wy = np.zeros(n), np.zeros(n), np.zeros(n)
    lib().orc_prep(C.c_int64(n), _p(t), _p(y), _p(dy), C.c_double(t_ref), _p(tau), _p(w), _p(wy))
    return tau, w, wy


def bins(f: float, nb: int, tau) -> np.ndarray:
    """O3: bin index of every point at one frequency."""
    tau = _f8(tau)
    b = np.zeros(tau.size, dtype=np.int32)
    lib().orc_bins(C.c_double(f), C.c_int32(nb), C.c_int64(tau.size), _p(tau), _p(b))
    return b


def sr_one(tau, w, wy, f: float, nb: int, M):
    """O3+O4 at one frequency with arbitrary (nb, M) -> (sr, m, j, r, s)."""
    tau, w, wy = _f8(tau), _f8(w), _f8(wy)
    M = np.ascontiguousarray(M, dtype=np.int32)
    H = np.zeros(2 * nb)
    sr, r, s = C.c_double(), C.c_double(), C.c_double()
    m, j = C.c_int32(), C.c_int32()
    lib().orc_sr_one(C.c_int64(tau.size), _p(tau), _p(w), _p(wy), C.c_double(f), C.c_int32(nb),
                     C.c_int(M.size), _p(M), _p(H), C.c_void_p(H.ctypes.data + 8 * nb),
                     C.byref(sr), C.byref(m), C.byref(j), C.byref(r), C.byref(s))
    return sr.value, m.value, j.value, r.value, s.value


def spectrum_star(cfg: Config, g, t, y, dy):
    """SR(f_k), best (m, j) over the star's own grid."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    ga = np.array([g], dtype=GRID_DTYPE)
    nf = int(ga[0]["n_freq"])
    sr = np.zeros(nf)
    m = np.zeros(nf, dtype=np.int32)
    j = np.zeros(nf, dtype=np.int32)
    rc = lib().orc_spectrum_star(C.byref(cfg), _p(ga), C.c_int64(t.size), _p(t), _p(y), _p(dy),
                                 _p(sr), _p(m), _p(j))
    assert rc == 0
    return sr, m, j


def spectrum_samples(cfg: Config, g, t, y, dy, ks):
    """O3+O4 of one star at the grid indices ks (OpenMP over the samples) -> (sr, m, j)."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    ga = np.array([g], dtype=GRID_DTYPE)
    ks = np.ascontiguousarray(ks, dtype=np.int64)
    sr = np.zeros(ks.size)
    m = np.zeros(ks.size, dtype=np.int32)
    j = np.zeros(ks.size, dtype=np.int32)
    rc = lib().orc_spectrum_samples(C.byref(cfg), _p(ga), C.c_int64(t.size), _p(t), _p(y), _p(dy),
                                    C.c_int64(ks.size), _p(ks), _p(sr), _p(m), _p(j))
    assert rc == 0, rc
    return sr, m, j


def box_values(cfg: Config, g, t, y, dy, ks, ms, js) -> np.ndarray:
    """Value s^2/(r(1-r)) of the given boxes (ms bins from start bin js) at grid indices ks, oracle arithmetic."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    ga = np.array([g], dtype=GRID_DTYPE)
    ks = np.ascontiguousarray(ks, dtype=np.int64)
    ms = np.ascontiguousarray(ms, dtype=np.int32)
    js = np.ascontiguousarray(js, dtype=np.int32)
    val = np.zeros(ks.size)
    rc = lib().orc_box_values(C.byref(cfg), _p(ga), C.c_int64(t.size), _p(t), _p(y), _p(dy),
                              C.c_int64(ks.size), _p(ks), _p(ms), _p(js), _p(val))
    assert rc == 0, rc
    return val


def snr(f, sr):
    """O5 -> (snr, trend, sigma)."""
    f, sr = _f8(f), _f8(sr)
    out, tr = np.zeros(f.size), np.zeros(f.size)
    sig = C.c_double()
    if f.size:
        lib().orc_snr(C.c_int64(f.size), _p(f), _p(sr), _p(out), _p(tr), C.byref(sig))
    return out, tr, sig.value


def peak_indices(snr_arr, K: int) -> np.ndarray:
    s = _f8(snr_arr)
    out = np.zeros(max(K, 1), dtype=np.int64)
    n = lib().orc_peak_indices(C.c_int64(s.size), _p(s), C.c_int(K), _p(out))
    return out[:n].copy()


def peak_record(cfg: Config, g, t, y, dy, k: int, snr_k: float):
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    ga = np.array([g], dtype=GRID_DTYPE)
    p = np.zeros(1, dtype=PEAK_DTYPE)
    lib().orc_peak_record(C.byref(cfg), _p(ga), C.c_int64(t.size), _p(t), _p(y), _p(dy),
                          C.c_int64(k), C.c_double(snr_k), _p(p))
    return p[0]


def peak_statistics(t, y, dy, f: float, m: int, nb: int, t0: float):
    """O7: points in / before / after transit, number of transits, out-of-transit level."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    out = np.zeros(1, dtype=STATS_DTYPE)
    lib().orc_peak_statistics(C.c_int64(t.size), _p(t), _p(y), _p(dy), C.c_double(f), C.c_int32(m), C.c_int32(nb),
                              C.c_double(t0), _p(out))
    return out[0]


TRAP_DTYPE = np.dtype([("t0", "f8"), ("depth", "f8"), ("q", "f8"), ("q_in", "f8"), ("z", "f8"), ("chi2", "f8"),
                       ("chi2_init", "f8"), ("n_fit", "i4"), ("n_eval", "i4"), ("status", "i4"), ("pad_", "i4")],
                      align=True)


def trapezoid_fit(t, y, dy, f: float, m: int, nb: int, t0: float):
    """O8: trapezoid fit (T0, depth, q, q_in, z) of one peak at fixed P = 1/f."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    out = np.zeros(1, dtype=TRAP_DTYPE)
    assert lib().orc_sizeof_trapezoid() == TRAP_DTYPE.itemsize
    lib().orc_trapezoid_fit(C.c_int64(t.size), _p(t), _p(y), _p(dy), C.c_double(f), C.c_int32(m), C.c_int32(nb),
                            C.c_double(t0), _p(out))
    return out[0]


def trapezoid_chi2_at(t, y, dy, f: float, m: int, nb: int, t0: float, c: float, q: float, q_in: float):
    """O8: (chi2, depth, z) of the fit data of a peak at given (c = T0 - t0, q, q_in)."""
    t, y, dy = _f8(t), _f8(y), _f8(dy)
    res = np.zeros(3)
    lib().orc_trapezoid_chi2_at.restype = C.c_int64
    lib().orc_trapezoid_chi2_at(C.c_int64(t.size), _p(t), _p(y), _p(dy), C.c_double(f), C.c_int32(m), C.c_int32(nb),
                                C.c_double(t0), C.c_double(c), C.c_double(q), C.c_double(q_in), _p(res))
    return float(res[0]), float(res[1]), float(res[2])


PINK_DTYPE = np.dtype([("sigma_w", "f8"), ("sigma_r", "f8"), ("depth_eff", "f8"), ("snr_pink", "f8"),
                       ("n_t", "i4"), ("n_transits", "i4"), ("n_bins", "i4"), ("detected", "i4")], align=True)


def pink_noise(t, y, f: float, t0: float, depth: float, q: float, q_in: float, z: float, snr: float):
    """O9: sigma_w, sigma_r on the duration timescale, S/N_pink (Eq. 2), detection flag."""
    t, y = _f8(t), _f8(y)
    out = np.zeros(1, dtype=PINK_DTYPE)
    assert lib().orc_sizeof_pink() == PINK_DTYPE.itemsize
    lib().orc_pink_noise(C.c_int64(t.size), _p(t), _p(y), C.c_double(f), C.c_double(t0), C.c_double(depth),
                         C.c_double(q), C.c_double(q_in), C.c_double(z), C.c_double(snr), _p(out))
    return out[0]


def batch(cfg: Config, row_ptr, t, y, dy, rho, K: int = 3, want_snr: bool = True, threads: int | None = None):
    """Whole path on a CSR batch (OpenMP over stars) -> dict(grid, freq_ptr, sr, m, j, snr, peaks)."""
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    t, y, dy, rho = _f8(t), _f8(y), _f8(dy), _f8(rho)
    S = row_ptr.size - 1
    L = lib()
    if threads:
        omp = C.CDLL("libgomp.so.1")
        omp.omp_set_num_threads(int(threads))
    grids = np.zeros(S, dtype=GRID_DTYPE)
    for s in range(S):
        a, b = int(row_ptr[s]), int(row_ptr[s + 1])
        L.orc_grid(C.byref(cfg), C.c_int64(b - a), C.c_void_p(t.ctypes.data + 8 * a), C.c_double(rho[s]),
                   C.c_void_p(grids.ctypes.data + s * GRID_DTYPE.itemsize))
    freq_ptr = np.zeros(S + 1, dtype=np.int64)
    np.cumsum(grids["n_freq"], out=freq_ptr[1:])
    nf = int(freq_ptr[-1])
    sr = np.zeros(nf)
    m = np.zeros(nf, dtype=np.int32)
    j = np.zeros(nf, dtype=np.int32)
    sn = np.zeros(nf) if want_snr else None
    peaks = np.zeros(S * K, dtype=PEAK_DTYPE) if K > 0 else None
    rc = L.orc_batch(C.byref(cfg), C.c_int64(S), _p(row_ptr), _p(t), _p(y), _p(dy), _p(rho), _p(grids),
                     _p(freq_ptr), _p(sr), _p(m), _p(j), _p(sn) if want_snr else None, C.c_int(K),
                     _p(peaks) if K > 0 else None)
    assert rc == 0
    return dict(grid=grids, freq_ptr=freq_ptr, sr=sr, m=m, j=j, snr=sn,
                peaks=None if peaks is None else peaks.reshape(S, K))
