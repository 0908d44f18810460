"""Thin Python binding of the C ABI in include/qlp_bls.h (argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs inside
``libqlp_bls.so``.  There is no CPU fallback: if the library is missing or a call fails, a
``QlpBlsError`` is raised.  Function names mirror the C entry points.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqlp_bls.so")
LIB_CHECK_PATH = os.path.join(_HERE, "libqlp_bls_check.so")   # bounds-check build (tests only)


class QlpBlsError(RuntimeError):
    pass


class Config(C.Structure):
    """qlp_bls_config (PAPER.md:7, :19, :23, :35 defaults via qlp_bls_default_config)."""
    _fields_ = [("struct_bytes", C.c_uint32), ("device", C.c_int32), ("samples_per_peak", C.c_double),
                ("dlogq", C.c_double), ("noverlap", C.c_int32), ("top_k", C.c_int32),
                ("qmin_fac", C.c_double), ("qmax_fac", C.c_double), ("a_over_rstar_min", C.c_double),
                ("sector_days", C.c_double), ("flags", C.c_uint32), ("reserved_", C.c_uint32),
                ("max_period_days", C.c_double), ("max_freq", C.c_int64)]


GRID_DTYPE = np.dtype([("t_ref", "f8"), ("baseline", "f8"), ("p_min", "f8"), ("p_max", "f8"),
                       ("c_q", "f8"), ("u0", "f8"), ("h", "f8"), ("n_freq", "i8"),
                       ("nb_max", "i4"), ("status", "i4")], align=True)
PEAK_DTYPE = np.dtype([("k", "i8"), ("freq", "f8"), ("period", "f8"), ("t0", "f8"), ("sr", "f4"),
                       ("snr", "f4"), ("q", "f4"), ("depth", "f4"), ("m", "i4"), ("j", "i4"),
                       ("nb", "i4"), ("status", "i4")], align=True)

STATS_DTYPE = np.dtype([("n_in", "i4"), ("n_before", "i4"), ("n_after", "i4"), ("n_transits", "i4"),
                        ("oot_level", "f8"), ("duration", "f8")], align=True)

TRAP_DTYPE = np.dtype([("t0", "f8"), ("depth", "f8"), ("q", "f8"), ("q_in", "f8"), ("z", "f8"), ("chi2", "f8"),
                       ("chi2_init", "f8"), ("n_fit", "i4"), ("n_eval", "i4"), ("status", "i4"), ("pad_", "i4")],
                      align=True)

PINK_DTYPE = np.dtype([("sigma_w", "f8"), ("sigma_r", "f8"), ("depth_eff", "f8"), ("snr_pink", "f8"),
                       ("n_t", "i4"), ("n_transits", "i4"), ("n_bins", "i4"), ("detected", "i4")], align=True)

EXPORTS = ["qlp_bls_peak_stats", "qlp_bls_trapezoid_fit", "qlp_bls_pink_noise", "qlp_bls_vet_host", "qlp_bls_default_config", "qlp_bls_create", "qlp_bls_grid", "qlp_bls_grid_noalloc", "qlp_bls_spectrum", "qlp_bls_snr",
           "qlp_bls_search_host", "qlp_bls_destroy", "qlp_bls_strerror", "qlp_bls_launch_count",
           "qlp_bls_widths", "qlp_bls_fold_timing", "qlp_bls_fold_elapsed_ms", "qlp_bls_fold_phase_clocks", "qlp_bls_fold_class_counters", "qlp_bls_fit_work", "qlp_bls_debug_freqs", "qlp_bls_debug_bins", "qlp_bls_debug_prep",
           "qlp_bls_debug_set_path", "qlp_bls_debug_violations"]

_libs = {}


def load_library(check: bool = False):
    """dlopen libqlp_bls.so (built by paper_2302_01293_b200.build); raises if it is missing.
    check=True: the bounds-check build libqlp_bls_check.so (`python -m paper_2302_01293_b200.build --check`)."""
    path = LIB_CHECK_PATH if check else LIB_PATH
    if path not in _libs:
        if not os.path.exists(path):
            raise QlpBlsError(f"{path} not built: run `python -m paper_2302_01293_b200.build"
                              f"{' --check' if check else ''}` (there is no CPU fallback)")
        L = C.CDLL(path)
        vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
        L.qlp_bls_default_config.argtypes = [C.POINTER(Config)]
        L.qlp_bls_default_config.restype = None
        L.qlp_bls_create.argtypes = [C.POINTER(Config), C.POINTER(vp)]
        L.qlp_bls_grid.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, C.POINTER(i64), C.POINTER(i64), vp]
        L.qlp_bls_grid_noalloc.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp]
        L.qlp_bls_spectrum.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.qlp_bls_snr.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.qlp_bls_peak_stats.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp]
        L.qlp_bls_trapezoid_fit.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp]
        L.qlp_bls_pink_noise.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp]
        L.qlp_bls_search_host.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, C.POINTER(i64), vp]
        L.qlp_bls_vet_host.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, C.POINTER(i64), vp]
        L.qlp_bls_destroy.argtypes = [vp]
        L.qlp_bls_strerror.argtypes = [C.c_int]
        L.qlp_bls_strerror.restype = C.c_char_p
        L.qlp_bls_launch_count.argtypes = [vp]
        L.qlp_bls_launch_count.restype = i64
        L.qlp_bls_widths.argtypes = [vp, vp, i32]
        L.qlp_bls_debug_freqs.argtypes = [vp, vp, i64, i64, i64, vp, vp, vp]
        L.qlp_bls_debug_bins.argtypes = [vp, vp, vp, vp, i64, i64, vp, vp]
        L.qlp_bls_debug_prep.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, vp]
        L.qlp_bls_debug_set_path.argtypes = [vp, i32]
        L.qlp_bls_fold_timing.argtypes = [vp, i32]
        L.qlp_bls_fold_elapsed_ms.argtypes = [vp, C.POINTER(i32), C.POINTER(C.c_double)]
        L.qlp_bls_fold_phase_clocks.argtypes = [vp, vp]
        L.qlp_bls_fold_class_counters.argtypes = [vp, vp]
        L.qlp_bls_fit_work.argtypes = [vp, vp]
        L.qlp_bls_debug_violations.argtypes = [vp, vp, i32]
        _libs[path] = L
    return _libs[path]


def default_config(**kw) -> Config:
    cfg = Config()
    load_library().qlp_bls_default_config(C.byref(cfg))
    uniform = kw.pop("uniform_freq", None)
    for k, v in kw.items():
        setattr(cfg, k, v)
    if uniform is not None:                # flags bit 1: comparison grid with equal steps in frequency (O1.10c)
        cfg.flags = (cfg.flags | 2) if uniform else (cfg.flags & ~2)
    return cfg


def _check(rc: int, what: str):
    if rc != 0:
        msg = load_library().qlp_bls_strerror(rc).decode()
        raise QlpBlsError(f"{what} failed: {msg} ({rc})")


def _ptr(x):
    if x is None:
        return None
    return C.c_void_p(x.data_ptr())


class QlpBls:
    """One qlp_bls_ctx.  Methods take/return torch CUDA tensors; nothing is computed in Python."""

    def __init__(self, cfg: Config | None = None, check: bool = False, **kw):
        import torch
        self.torch = torch
        self.lib = load_library(check)
        if not torch.cuda.is_available():
            raise QlpBlsError("no CUDA device: the QLP BLS path has no CPU fallback")
        self.cfg = cfg if cfg is not None else default_config(**kw)
        self.device = torch.device("cuda", self.cfg.device)
        h = C.c_void_p()
        _check(self.lib.qlp_bls_create(C.byref(self.cfg), C.byref(h)), "qlp_bls_create")
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self.lib.qlp_bls_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    @property
    def top_k(self) -> int:
        return int(self.cfg.top_k)

    def launch_count(self) -> int:
        return int(self.lib.qlp_bls_launch_count(self._h))

    def widths(self) -> np.ndarray:
        m = np.zeros(32, dtype=np.int32)
        n = self.lib.qlp_bls_widths(self._h, m.ctypes.data_as(C.c_void_p), 32)
        return m[:n].copy()

    def fold_timing(self, enable: bool):
        _check(self.lib.qlp_bls_fold_timing(self._h, 1 if enable else 0), "qlp_bls_fold_timing")

    def fold_elapsed_ms(self):
        """-> (number of spectrum calls timed, summed device ms of their fold/scan launches)."""
        n, ms = C.c_int32(), C.c_double()
        _check(self.lib.qlp_bls_fold_elapsed_ms(self._h, C.byref(n), C.byref(ms)), "qlp_bls_fold_elapsed_ms")
        return int(n.value), float(ms.value)

    def fold_phase_clocks(self):
        """-> (set-up, fold, scan) SM clocks of thread 0 summed over all tiles since fold_timing(True)."""
        a = np.zeros(3, dtype=np.uint64)
        _check(self.lib.qlp_bls_fold_phase_clocks(self._h, a.ctypes.data_as(C.c_void_p)), "qlp_bls_fold_phase_clocks")
        return [int(x) for x in a]

    def fold_class_counters(self) -> np.ndarray:
        """-> uint64[9, 5]: per tile class (set-up, fold, scan clocks of thread 0; evaluations; tiles)."""
        a = np.zeros((9, 5), dtype=np.uint64)
        _check(self.lib.qlp_bls_fold_class_counters(self._h, a.ctypes.data_as(C.c_void_p)),
               "qlp_bls_fold_class_counters")
        return a

    def fit_work(self) -> int:
        """(point, sweep) pairs inside a transit that the fit kernels processed since fold_timing(True)."""
        a = np.zeros(2, dtype=np.uint64)
        _check(self.lib.qlp_bls_fit_work(self._h, a.ctypes.data_as(C.c_void_p)), "qlp_bls_fit_work")
        return int(a[0])

    def debug_violations(self, reset: bool = True) -> np.ndarray:
        """Bounds-check build only -> uint64[8] violation counters (fold cell, staging, scan bin, fit slot, ...)."""
        a = np.zeros(8, dtype=np.uint64)
        _check(self.lib.qlp_bls_debug_violations(self._h, a.ctypes.data_as(C.c_void_p), 1 if reset else 0),
               "qlp_bls_debug_violations")
        return a

    def debug_set_path(self, path: int):
        _check(self.lib.qlp_bls_debug_set_path(self._h, path), "qlp_bls_debug_set_path")

    # -- S1
    def grid(self, row_ptr, t, rho, rstar=None):
        """qlp_bls_grid -> (grid uint8[S, 72] tensor, freq_ptr int64[S+1], total_freq, total_bins)."""
        torch = self.torch
        S = int(row_ptr.numel()) - 1
        grid = torch.zeros((max(S, 1), GRID_DTYPE.itemsize), dtype=torch.uint8, device=self.device)[:S]
        freq_ptr = torch.zeros(S + 1, dtype=torch.int64, device=self.device)
        tf, tb = C.c_int64(), C.c_int64()
        _check(self.lib.qlp_bls_grid(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(rho), _ptr(rstar), _ptr(grid),
                                     _ptr(freq_ptr), C.byref(tf), C.byref(tb), self._stream()), "qlp_bls_grid")
        return grid, freq_ptr, int(tf.value), int(tb.value)

    def grid_noalloc(self, row_ptr, t, rho, grid, freq_ptr, totals):
        """qlp_bls_grid_noalloc: S1 into caller-provided device tensors (grid uint8[S, 72], freq_ptr int64[S+1],
        totals int64[2]); the library allocates nothing, copies nothing back and does not synchronise."""
        S = int(row_ptr.numel()) - 1
        _check(self.lib.qlp_bls_grid_noalloc(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(rho), _ptr(grid),
                                             _ptr(freq_ptr), _ptr(totals), self._stream()), "qlp_bls_grid_noalloc")

    # -- S0 + S2 + S3
    def spectrum(self, row_ptr, t, y, dy, grid, freq_ptr, total_freq: int):
        """qlp_bls_spectrum -> (sr float32[total_freq], best uint32-as-int32[total_freq])."""
        torch = self.torch
        S = int(row_ptr.numel()) - 1
        # at least one element each, so that a batch without any frequency still hands over valid pointers
        sr = torch.empty(max(total_freq, 1), dtype=torch.float32, device=self.device)
        best = torch.empty(max(total_freq, 1), dtype=torch.int32, device=self.device)
        _check(self.lib.qlp_bls_spectrum(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(dy), _ptr(grid),
                                         _ptr(freq_ptr), _ptr(sr), _ptr(best), self._stream()), "qlp_bls_spectrum")
        return sr[:total_freq], best[:total_freq]

    def spectrum_into(self, row_ptr, t, y, dy, grid, freq_ptr, sr, best):
        S = int(row_ptr.numel()) - 1
        _check(self.lib.qlp_bls_spectrum(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(dy), _ptr(grid),
                                         _ptr(freq_ptr), _ptr(sr), _ptr(best), self._stream()), "qlp_bls_spectrum")

    # -- S4
    def snr(self, row_ptr, t, y, dy, grid, freq_ptr, sr, best, want_snr: bool = True, peaks=None):
        """qlp_bls_snr -> (snr float32[total_freq] or None, peaks uint8[S*top_k, 64] tensor)."""
        torch = self.torch
        S = int(row_ptr.numel()) - 1
        snr = torch.empty_like(sr) if want_snr else None
        if peaks is None:
            peaks = torch.zeros((max(S * self.top_k, 1), PEAK_DTYPE.itemsize), dtype=torch.uint8,
                                device=self.device)[:S * self.top_k]
        _check(self.lib.qlp_bls_snr(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(dy), _ptr(grid),
                                    _ptr(freq_ptr), _ptr(sr), _ptr(best), _ptr(snr), _ptr(peaks), self._stream()),
               "qlp_bls_snr")
        return snr, peaks

    # -- O7
    def peak_stats(self, row_ptr, t, y, dy, peaks):
        """qlp_bls_peak_stats -> stats uint8[S*top_k, 32] tensor (see stats_to_numpy)."""
        torch = self.torch
        S = int(row_ptr.numel()) - 1
        stats = torch.zeros((max(S * self.top_k, 1), STATS_DTYPE.itemsize), dtype=torch.uint8,
                            device=self.device)[:S * self.top_k]
        _check(self.lib.qlp_bls_peak_stats(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(dy), _ptr(peaks),
                                           _ptr(stats), self._stream()), "qlp_bls_peak_stats")
        return stats

    # -- O8
    def trapezoid_fit(self, row_ptr, t, y, dy, peaks):
        """qlp_bls_trapezoid_fit -> fits uint8[S*top_k, 72] tensor (see fits_to_numpy).  Synchronises once."""
        torch = self.torch
        S = int(row_ptr.numel()) - 1
        fits = torch.zeros((max(S * self.top_k, 1), TRAP_DTYPE.itemsize), dtype=torch.uint8,
                           device=self.device)[:S * self.top_k]
        _check(self.lib.qlp_bls_trapezoid_fit(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(dy), _ptr(peaks),
                                              _ptr(fits), self._stream()), "qlp_bls_trapezoid_fit")
        return fits

    # -- O9
    def pink_noise(self, row_ptr, t, y, peaks, fits):
        """qlp_bls_pink_noise -> pink uint8[S*top_k, 48] tensor (see pink_to_numpy)."""
        torch = self.torch
        S = int(row_ptr.numel()) - 1
        pink = torch.zeros((max(S * self.top_k, 1), PINK_DTYPE.itemsize), dtype=torch.uint8,
                           device=self.device)[:S * self.top_k]
        _check(self.lib.qlp_bls_pink_noise(self._h, S, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(peaks), _ptr(fits),
                                           _ptr(pink), self._stream()), "qlp_bls_pink_noise")
        return pink

    # -- whole path from host (numpy / pinned torch CPU) buffers
    def search_host(self, row_ptr, t, y, dy, rho, want_grid: bool = False, want_stats: bool = False):
        """qlp_bls_search_host on numpy arrays -> (peaks structured [S, top_k], grid or None, total_freq)
        or, with want_stats, (peaks, stats [S, top_k], grid or None, total_freq)."""
        S = int(row_ptr.shape[0]) - 1
        peaks = np.zeros(S * self.top_k, dtype=PEAK_DTYPE)
        stats = np.zeros(S * self.top_k, dtype=STATS_DTYPE) if want_stats else None
        grid = np.zeros(S, dtype=GRID_DTYPE) if want_grid else None
        tf = C.c_int64()

        def hp(a):
            return C.c_void_p(a.ctypes.data)
        _check(self.lib.qlp_bls_search_host(self._h, S, hp(row_ptr), hp(t), hp(y), hp(dy), hp(rho), None, hp(peaks),
                                            hp(stats) if want_stats else None, hp(grid) if want_grid else None,
                                            C.byref(tf), self._stream()),
               "qlp_bls_search_host")
        if want_stats:
            return peaks.reshape(S, self.top_k), stats.reshape(S, self.top_k), grid, int(tf.value)
        return peaks.reshape(S, self.top_k), grid, int(tf.value)

    def vet_host(self, row_ptr, t, y, dy, rho):
        """qlp_bls_vet_host on numpy arrays -> (peaks, stats, fits, pink), structured [S, top_k] each: the search and
        the rows after it from host buffers."""
        S = int(row_ptr.shape[0]) - 1
        n = S * self.top_k
        peaks, stats = np.zeros(n, dtype=PEAK_DTYPE), np.zeros(n, dtype=STATS_DTYPE)
        fits, pink = np.zeros(n, dtype=TRAP_DTYPE), np.zeros(n, dtype=PINK_DTYPE)
        tf = C.c_int64()

        def hp(a):
            return C.c_void_p(a.ctypes.data)
        _check(self.lib.qlp_bls_vet_host(self._h, S, hp(row_ptr), hp(t), hp(y), hp(dy), hp(rho), None, hp(peaks),
                                         hp(stats), hp(fits), hp(pink), None, C.byref(tf), self._stream()),
               "qlp_bls_vet_host")
        shape = (S, self.top_k)
        return peaks.reshape(shape), stats.reshape(shape), fits.reshape(shape), pink.reshape(shape)

    # -- test-only
    def debug_freqs(self, grid, star: int, k0: int, k1: int):
        torch = self.torch
        n = max(k1 - k0, 0)
        f = torch.zeros(max(n, 1), dtype=torch.float64, device=self.device)[:n]
        nb = torch.zeros(max(n, 1), dtype=torch.int32, device=self.device)[:n]
        _check(self.lib.qlp_bls_debug_freqs(self._h, _ptr(grid), star, k0, k1, _ptr(f), _ptr(nb), self._stream()),
               "qlp_bls_debug_freqs")
        return f, nb

    def debug_bins(self, row_ptr, t, grid, star: int, k: int, n_pts: int):
        torch = self.torch
        out = torch.zeros(max(n_pts, 1), dtype=torch.int32, device=self.device)[:n_pts]
        _check(self.lib.qlp_bls_debug_bins(self._h, _ptr(row_ptr), _ptr(t), _ptr(grid), star, k, _ptr(out),
                                           self._stream()), "qlp_bls_debug_bins")
        return out

    def debug_prep(self, row_ptr, t, y, dy, grid, star: int, n_pts: int):
        torch = self.torch
        tau = torch.zeros(max(n_pts, 1), dtype=torch.float64, device=self.device)[:n_pts]
        w = torch.zeros(max(n_pts, 1), dtype=torch.float32, device=self.device)[:n_pts]
        wy = torch.zeros(max(n_pts, 1), dtype=torch.float32, device=self.device)[:n_pts]
        _check(self.lib.qlp_bls_debug_prep(self._h, _ptr(row_ptr), _ptr(t), _ptr(y), _ptr(dy), _ptr(grid), star,
                                           _ptr(tau), _ptr(w), _ptr(wy), self._stream()), "qlp_bls_debug_prep")
        return tau, w, wy


def grid_to_numpy(grid_tensor) -> np.ndarray:
    """Device grid descriptors -> structured numpy array (a D2H copy, for tests and reports)."""
    return np.frombuffer(grid_tensor.cpu().numpy().tobytes(), dtype=GRID_DTYPE).copy()


def peaks_to_numpy(peaks_tensor, top_k: int) -> np.ndarray:
    a = np.frombuffer(peaks_tensor.cpu().numpy().tobytes(), dtype=PEAK_DTYPE).copy()
    return a.reshape(-1, top_k)


def stats_to_numpy(stats_tensor, top_k: int) -> np.ndarray:
    a = np.frombuffer(stats_tensor.cpu().numpy().tobytes(), dtype=STATS_DTYPE).copy()
    return a.reshape(-1, top_k)


def fits_to_numpy(fits_tensor, top_k: int) -> np.ndarray:
    a = np.frombuffer(fits_tensor.cpu().numpy().tobytes(), dtype=TRAP_DTYPE).copy()
    return a.reshape(-1, top_k)


def pink_to_numpy(pink_tensor, top_k: int) -> np.ndarray:
    a = np.frombuffer(pink_tensor.cpu().numpy().tobytes(), dtype=PINK_DTYPE).copy()
    return a.reshape(-1, top_k)


def upload(batch, device="cuda"):
    """Copy a synth.Batch (numpy) to device tensors: (row_ptr, t, y, dy, rho, rstar)."""
    import torch
    dev = torch.device(device)
    f = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).to(dev)
    return (f(batch.row_ptr, np.int64), f(batch.t, np.float64), f(batch.y, np.float64), f(batch.dy, np.float64),
            f(batch.rho, np.float64), f(batch.rstar, np.float64))
