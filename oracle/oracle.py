"""ctypes wrapper around oracle/nsfrb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never touches the CUDA path.  The C file's header
states the definition (O1..O7, S1..S6) and the PAPER.md passages it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nsfrb_oracle.c")
_LIB = os.path.join(_HERE, "libnsfrb_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-pthread", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32p = ctypes.POINTER(ctypes.c_int32)
        i64p = ctypes.POINTER(ctypes.c_int64)
        f64p = ctypes.POINTER(ctypes.c_double)
        f32p = ctypes.POINTER(ctypes.c_float)
        lib.nsfrb_oracle_delays.restype = ctypes.c_int
        lib.nsfrb_oracle_delays.argtypes = [ctypes.c_int, f64p, ctypes.c_double, ctypes.c_int, f64p, i32p]
        lib.nsfrb_oracle_search.restype = ctypes.c_int
        lib.nsfrb_oracle_search.argtypes = [
            f32p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, i32p, ctypes.c_int, i32p, ctypes.c_int,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_int, i64p, ctypes.c_int64, ctypes.c_int,
            f64p, i64p, f64p, f64p, f64p, i64p,
        ]
        lib.nsfrb_oracle_search_norm.restype = ctypes.c_int
        lib.nsfrb_oracle_search_norm.argtypes = lib.nsfrb_oracle_search.argtypes + [f64p]
        lib.nsfrb_oracle_snr_at.restype = ctypes.c_double
        lib.nsfrb_oracle_snr_at.argtypes = [
            f32p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, i32p, ctypes.c_int, i32p, ctypes.c_int,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
        ]
        lib.nsfrb_oracle_bin.restype = ctypes.c_int
        lib.nsfrb_oracle_bin.argtypes = [f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int64, ctypes.c_int, f32p]
        lib.nsfrb_oracle_cells_per_pixel.restype = ctypes.c_int64
        lib.nsfrb_oracle_cells_per_pixel.argtypes = [ctypes.c_int, ctypes.c_int, i32p, ctypes.c_int, i32p, ctypes.c_int]
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def delays(freqs_GHz, tsamp_s, dm_list) -> np.ndarray:
    """O1: int32 delay table [ndm][nchan]."""
    f = np.ascontiguousarray(freqs_GHz, dtype=np.float64)
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    out = np.empty((dm.size, f.size), dtype=np.int32)
    rc = _load().nsfrb_oracle_delays(f.size, _p(f, ctypes.c_double), float(tsamp_s), dm.size,
                                     _p(dm, ctypes.c_double), _p(out, ctypes.c_int32))
    if rc != 0:
        raise ValueError(f"nsfrb_oracle_delays failed: {rc}")
    return out


@dataclass
class OracleResult:
    snr: np.ndarray          # [n_sel] float64
    argmax: np.ndarray       # [n_sel][3] int64 (dm_idx, width_idx, t)
    pixels: np.ndarray       # [n_sel] int64
    mu: np.ndarray | None = None      # [n_sel][ndm]
    sigma: np.ndarray | None = None   # [n_sel][ndm]
    best: np.ndarray | None = None    # [n_sel][ndm][nw] max_t S(k,j,t)
    best_t: np.ndarray | None = None  # [n_sel][ndm][nw]

    def candidates(self, threshold: float):
        """O7: set of (pixel, dm_idx, width_idx, t) with snr > threshold (strict)."""
        sel = np.nonzero(self.snr > threshold)[0]
        return {(int(self.pixels[i]), int(self.argmax[i, 0]), int(self.argmax[i, 1]), int(self.argmax[i, 2]))
                for i in sel}


def search(cube, delay_table, widths, *, pixels=None, raw_end_min=0, t_offset=0,
           brute=False, nthreads=1, details=False, sigma_norm=None) -> OracleResult:
    """O2..O6 (+S5/S6) for the selected pixels of cube[nchan][nt][npix] (float32).
    sigma_norm [n_sel][ndm] (float64), if given, replaces sigma_k in O5 (reading R30: running standard deviation)."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    if cube.ndim != 3:
        raise ValueError("cube must be [nchan][nt][npix]")
    nchan, nt, npix = cube.shape
    d = np.ascontiguousarray(delay_table, dtype=np.int32)
    if d.ndim != 2 or d.shape[1] != nchan:
        raise ValueError("delay table must be [ndm][nchan]")
    ndm = d.shape[0]
    w = np.ascontiguousarray(widths, dtype=np.int32)
    nw = w.size
    if pixels is None:
        pix = None
        sel = np.arange(npix, dtype=np.int64)
    else:
        sel = np.ascontiguousarray(pixels, dtype=np.int64)
        pix = sel
    n_sel = sel.size
    snr = np.empty(n_sel, dtype=np.float64)
    arg = np.empty((n_sel, 3), dtype=np.int64)
    mu = sigma = best = best_t = None
    if details:
        mu = np.empty((n_sel, ndm), dtype=np.float64)
        sigma = np.empty((n_sel, ndm), dtype=np.float64)
        best = np.empty((n_sel, ndm, nw), dtype=np.float64)
        best_t = np.empty((n_sel, ndm, nw), dtype=np.int64)
    sn = None
    if sigma_norm is not None:
        sn = np.ascontiguousarray(sigma_norm, dtype=np.float64)
        if sn.shape != (n_sel, ndm):
            raise ValueError("sigma_norm must be [n_sel][ndm]")
    rc = _load().nsfrb_oracle_search_norm(
        _p(cube, ctypes.c_float), npix, nchan, nt, _p(d, ctypes.c_int32), ndm, _p(w, ctypes.c_int32), nw,
        int(raw_end_min), int(t_offset), int(bool(brute)), _p(pix, ctypes.c_int64), n_sel, int(nthreads),
        _p(snr, ctypes.c_double), _p(arg, ctypes.c_int64), _p(mu, ctypes.c_double), _p(sigma, ctypes.c_double),
        _p(best, ctypes.c_double), _p(best_t, ctypes.c_int64), _p(sn, ctypes.c_double))
    if rc != 0:
        raise ValueError(f"nsfrb_oracle_search failed: {rc}")
    return OracleResult(snr, arg, sel, mu, sigma, best, best_t)


def snr_at(cube, delay_table, widths, p, k, j, t, *, raw_end_min=0, t_offset=0) -> float:
    """S(k,j,t) of one cell (NaN if the cell is not defined)."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    nchan, nt, npix = cube.shape
    d = np.ascontiguousarray(delay_table, dtype=np.int32)
    w = np.ascontiguousarray(widths, dtype=np.int32)
    return float(_load().nsfrb_oracle_snr_at(
        _p(cube, ctypes.c_float), npix, nchan, nt, _p(d, ctypes.c_int32), d.shape[0], _p(w, ctypes.c_int32),
        w.size, int(raw_end_min), int(t_offset), int(p), int(k), int(j), int(t)))


def cells_per_pixel(delay_table, widths, nt) -> int:
    """Exact cell count per pixel of one offline call: sum_k sum_j max(0, T_k - w_j + 1)."""
    d = np.ascontiguousarray(delay_table, dtype=np.int32)
    w = np.ascontiguousarray(widths, dtype=np.int32)
    return int(_load().nsfrb_oracle_cells_per_pixel(d.shape[1], int(nt), _p(d, ctypes.c_int32), d.shape[0],
                                                    _p(w, ctypes.c_int32), w.size))


def bin_time(cube, factor: int) -> np.ndarray:
    """NEXT 2 / reading R24: sum of `factor` consecutive samples, floor(nt/factor) outputs."""
    a = np.ascontiguousarray(cube, dtype=np.float32)
    nchan, nt, npix = a.shape
    out = np.empty((nchan, nt // int(factor), npix), dtype=np.float32)
    if out.size:
        rc = _load().nsfrb_oracle_bin(_p(a, ctypes.c_float), nchan, nt, npix, int(factor), _p(out, ctypes.c_float))
        if rc != 0:
            raise ValueError("nsfrb_oracle_bin: bad arguments")
    return out


def median_subtract(cube):
    """NEXT 1 (first part) / reading R29: "Data is first median subtracted in each pixel".  For every
    (channel, pixel) series of the nt samples: median = the middle element of the sorted series (the mean of the two
    middle ones for even nt, in float64, rounded once to float32); out = cube - median in float32.
    Returns (out [nchan][nt][npix] float32, median [nchan][npix] float32)."""
    a = np.ascontiguousarray(cube, dtype=np.float32)
    nchan, nt, npix = a.shape
    if nt < 1:
        raise ValueError("nt must be >= 1")
    s = np.sort(a.astype(np.float64), axis=1)
    med = (0.5 * (s[:, (nt - 1) // 2, :] + s[:, nt // 2, :])).astype(np.float32)
    return a - med[:, None, :], med


class StreamOracle:
    """S1..S6: the streaming definition, by re-running the offline definition on the
    chronological ring contents after every push (no incremental state)."""

    def __init__(self, nchan, npix, ring_len, delay_table, widths):
        self.nchan, self.npix, self.L = int(nchan), int(npix), int(ring_len)
        self.d = np.ascontiguousarray(delay_table, dtype=np.int32)
        self.w = np.ascontiguousarray(widths, dtype=np.int32)
        self.hist = np.zeros((self.nchan, 0, self.npix), dtype=np.float32)  # chronological, <= L samples
        self.n = 0  # S1: absolute count of samples received

    def push(self, chunk, **kw) -> OracleResult:
        chunk = np.ascontiguousarray(chunk, dtype=np.float32)
        assert chunk.shape[0] == self.nchan and chunk.shape[2] == self.npix
        n_prev = self.n
        self.n += chunk.shape[1]                                   # S2
        self.hist = np.concatenate([self.hist, chunk], axis=1)[:, -self.L:, :]
        lo = max(0, self.n - self.L)                               # S1
        return search(self.hist, self.d, self.w, raw_end_min=n_prev - lo, t_offset=lo, **kw)  # S3..S6


def running_variance(var_prev, sigma_now, alpha: float):
    """Reading R30 ("normalized by the running standard deviation", L180 "the running standard deviation
    accumulated during" the survey): per (pixel, DM trial) an exponentially weighted variance carried across pushes,
        v_0 = sigma_0^2,   v_n = (1 - alpha) v_{n-1} + alpha sigma_n^2,
    sigma_n = this push's own sigma_k (O3).  A trial with no valid sample yet (sigma NaN) keeps its previous state."""
    s2 = np.asarray(sigma_now, dtype=np.float64) ** 2
    if var_prev is None:
        return s2.copy()
    v = (1.0 - alpha) * var_prev + alpha * s2
    v = np.where(np.isnan(var_prev), s2, v)        # first defined sigma starts the recursion
    return np.where(np.isnan(s2), var_prev, v)


class RunningStreamOracle(StreamOracle):
    """S1..S6 with O5 normalised by the running standard deviation (reading R30): every push first evaluates the
    offline definition for this push's own sigma_k, updates the running variance, then evaluates the definition again
    with sigma_norm = sqrt(v_n).  No incremental shortcut."""

    def __init__(self, nchan, npix, ring_len, delay_table, widths, alpha):
        super().__init__(nchan, npix, ring_len, delay_table, widths)
        self.alpha = float(alpha)
        self.var = None            # [npix][ndm] float64

    def push(self, chunk, **kw) -> OracleResult:
        kw.pop("details", None)
        inst = super().push(chunk, details=True, **kw)
        self.var = running_variance(self.var, inst.sigma, self.alpha)
        n_prev = self.n - np.asarray(chunk).shape[1]
        lo = max(0, self.n - self.L)
        return search(self.hist, self.d, self.w, raw_end_min=n_prev - lo, t_offset=lo, details=True,
                      sigma_norm=np.sqrt(self.var), **kw)
