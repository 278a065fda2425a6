"""Thin ctypes binding over the C-ABI library libnsfrb.so (include/nsfrb.h).

Argument marshalling only: every step of the search runs in the library's CUDA kernels.
PyTorch supplies device memory and streams.  There is no CPU fallback: loading fails loudly
if the library has not been built (python -m paper_2510_18136_b200.build).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnsfrb.so")

NSFRB_OK, NSFRB_EINVAL, NSFRB_ENOMEM, NSFRB_ECUDA, NSFRB_ESTATE = 0, -1, -2, -3, -4


class NsfrbError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"nsfrb error {code}: {msg}")
        self.code = code


class nsfrb_cand(ctypes.Structure):
    _fields_ = [("pixel", ctypes.c_int32), ("dm_idx", ctypes.c_int32), ("width_idx", ctypes.c_int32),
                ("t", ctypes.c_int32), ("snr", ctypes.c_float)]


class nsfrb_plan_info(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in (
        "npix", "nchan", "nt", "ndm", "nwidth", "ndm_unique", "dmax", "wmax", "n_groups", "n_width_batches",
        "series_per_cta", "block_len", "ring_len", "search_threads")] + [
        (n, ctypes.c_int64) for n in ("search_smem_bytes", "workspace_bytes", "cells_per_pixel", "shift_adds_per_pixel")]


CAND_DTYPE = np.dtype([("pixel", "<i4"), ("dm_idx", "<i4"), ("width_idx", "<i4"), ("t", "<i4"), ("snr", "<f4")])
assert CAND_DTYPE.itemsize == ctypes.sizeof(nsfrb_cand) == 20

# every symbol include/nsfrb.h declares
EXPORTS = ("nsfrb_plan_create", "nsfrb_search", "nsfrb_stream_push", "nsfrb_stream_reset", "nsfrb_search_host",
           "nsfrb_stream_push_host", "nsfrb_plan_destroy", "nsfrb_plan_get_delays", "nsfrb_plan_get_info",
           "nsfrb_plan_last_launches", "nsfrb_stream_mode", "nsfrb_plan_set_profiling", "nsfrb_plan_get_kernel_ms", "nsfrb_last_error",
           "nsfrb_version", "nsfrb_jit_stream_kernel", "nsfrb_bin_time", "nsfrb_jit_search_kernel", "nsfrb_stream_set_cubes",
           "nsfrb_psf_mask", "nsfrb_cluster", "nsfrb_median_subtract",
           "nsfrb_stream_push_host_async", "nsfrb_stream_wait", "nsfrb_stream_set_running_sigma",
           "nsfrb_peaks_count", "nsfrb_peaks_name", "nsfrb_measure_peaks", "nsfrb_plan_prepare", "nsfrb_cluster_static",
           "nsfrb_imager_create", "nsfrb_imager_image", "nsfrb_imager_get_table", "nsfrb_imager_destroy")

_lib = None


def lib() -> ctypes.CDLL:
    """Load libnsfrb.so; raises if it is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2510_18136_b200.build` (needs nvcc); "
                              "there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32p, f64p = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_double)
        L.nsfrb_plan_create.restype = ctypes.c_int
        L.nsfrb_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                        f64p, ctypes.c_double, f64p, ctypes.c_int, i32p, ctypes.c_int, ctypes.c_float]
        out = [vp, vp, vp, ctypes.c_uint32, vp]
        L.nsfrb_search.restype = ctypes.c_int
        L.nsfrb_search.argtypes = [vp, vp, vp] + out
        L.nsfrb_stream_push.restype = ctypes.c_int
        L.nsfrb_stream_push.argtypes = [vp, vp, ctypes.c_int, vp] + out
        L.nsfrb_search_host.restype = ctypes.c_int
        L.nsfrb_search_host.argtypes = [vp, vp, vp] + out
        L.nsfrb_stream_push_host.restype = ctypes.c_int
        L.nsfrb_stream_push_host.argtypes = [vp, vp, ctypes.c_int, vp] + out
        L.nsfrb_stream_set_cubes.restype = ctypes.c_int
        L.nsfrb_stream_set_cubes.argtypes = [vp, vp, vp]
        L.nsfrb_stream_reset.restype = ctypes.c_int
        L.nsfrb_stream_reset.argtypes = [vp]
        L.nsfrb_plan_destroy.restype = ctypes.c_int
        L.nsfrb_plan_destroy.argtypes = [vp]
        L.nsfrb_plan_get_delays.restype = ctypes.c_int
        L.nsfrb_plan_get_delays.argtypes = [vp, i32p]
        L.nsfrb_plan_get_info.restype = ctypes.c_int
        L.nsfrb_plan_get_info.argtypes = [vp, ctypes.POINTER(nsfrb_plan_info)]
        L.nsfrb_plan_last_launches.restype = ctypes.c_int
        L.nsfrb_plan_last_launches.argtypes = [vp]
        L.nsfrb_stream_mode.restype = ctypes.c_int
        L.nsfrb_stream_mode.argtypes = [vp]
        L.nsfrb_plan_set_profiling.restype = ctypes.c_int
        L.nsfrb_plan_set_profiling.argtypes = [vp, ctypes.c_int]
        L.nsfrb_plan_get_kernel_ms.restype = ctypes.c_int
        L.nsfrb_plan_get_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
        L.nsfrb_jit_stream_kernel.restype = ctypes.c_int
        L.nsfrb_jit_stream_kernel.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, f64p, ctypes.c_double,
                                              f64p, ctypes.c_int, i32p, ctypes.c_int, ctypes.c_int, ctypes.c_char_p,
                                              ctypes.c_int, vp, ctypes.c_size_t, ctypes.POINTER(ctypes.c_size_t)]
        L.nsfrb_jit_search_kernel.restype = ctypes.c_int
        L.nsfrb_jit_search_kernel.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, f64p, ctypes.c_double,
                                              f64p, ctypes.c_int, i32p, ctypes.c_int, ctypes.c_int, vp, ctypes.c_size_t,
                                              ctypes.POINTER(ctypes.c_size_t)]
        L.nsfrb_bin_time.restype = ctypes.c_int
        L.nsfrb_bin_time.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int64, ctypes.c_int, vp, vp]
        L.nsfrb_stream_push_host_async.restype = ctypes.c_int
        L.nsfrb_stream_push_host_async.argtypes = [vp, vp, ctypes.c_int, vp, vp, vp, ctypes.c_uint32, vp]
        L.nsfrb_stream_set_running_sigma.restype = ctypes.c_int
        L.nsfrb_stream_set_running_sigma.argtypes = [vp, ctypes.c_double, vp, vp]
        L.nsfrb_stream_wait.restype = ctypes.c_int
        L.nsfrb_stream_wait.argtypes = [vp]
        L.nsfrb_median_subtract.restype = ctypes.c_int
        L.nsfrb_median_subtract.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int64, vp, vp, vp]
        L.nsfrb_psf_mask.restype = ctypes.c_int
        L.nsfrb_psf_mask.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_double, vp, vp, vp]
        L.nsfrb_cluster.restype = ctypes.c_int
        L.nsfrb_cluster.argtypes = [vp, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, vp]
        L.nsfrb_cluster_static.restype = ctypes.c_int
        L.nsfrb_cluster_static.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_float, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int,
                                           ctypes.c_int, vp, vp, vp, vp, vp]
        L.nsfrb_imager_create.restype = ctypes.c_int
        L.nsfrb_imager_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, ctypes.c_double, f64p, ctypes.c_int, f64p, ctypes.c_int,
                                          ctypes.c_double, ctypes.c_double, ctypes.c_double]
        L.nsfrb_imager_image.restype = ctypes.c_int
        L.nsfrb_imager_image.argtypes = [vp, vp, ctypes.c_int, vp, vp]
        L.nsfrb_imager_get_table.restype = ctypes.c_int
        L.nsfrb_imager_get_table.argtypes = [vp, i32p, f64p]
        L.nsfrb_imager_destroy.restype = ctypes.c_int
        L.nsfrb_imager_destroy.argtypes = [vp]
        L.nsfrb_plan_prepare.restype = ctypes.c_int
        L.nsfrb_plan_prepare.argtypes = [vp, ctypes.c_int, ctypes.c_int]
        L.nsfrb_peaks_count.restype = ctypes.c_int
        L.nsfrb_peaks_count.argtypes = []
        L.nsfrb_peaks_name.restype = ctypes.c_char_p
        L.nsfrb_peaks_name.argtypes = [ctypes.c_int]
        L.nsfrb_measure_peaks.restype = ctypes.c_int
        L.nsfrb_measure_peaks.argtypes = [ctypes.c_int, f64p, f64p, vp]
        L.nsfrb_last_error.restype = ctypes.c_char_p
        L.nsfrb_version.restype = ctypes.c_char_p
        _lib = L
    return _lib


def last_error() -> str:
    return lib().nsfrb_last_error().decode()


def _check(rc: int):
    if rc != 0:
        raise NsfrbError(rc, last_error())


@dataclass
class SearchResult:
    snr_map: torch.Tensor   # [npix] float32
    argmax: torch.Tensor    # [3][npix] int32: dm_idx | width_idx | t
    cands: torch.Tensor     # [capacity*20] uint8 (raw nsfrb_cand records)
    ncands: torch.Tensor    # [1] int32 view of the uint32 counter

    def candidates(self) -> np.ndarray:
        """Structured array of the stored candidates (synchronises)."""
        n = int(self.ncands.cpu().numpy().view(np.uint32)[0])
        cap = self.cands.numel() // CAND_DTYPE.itemsize
        raw = self.cands[: min(n, cap) * CAND_DTYPE.itemsize].cpu().numpy()
        return raw.view(CAND_DTYPE).copy()

    def n_found(self) -> int:
        return int(self.ncands.cpu().numpy().view(np.uint32)[0])


def jit_stream_kernel(nx, ny, nchan, nt, freqs_GHz, tsamp_s, dm_list, width_list, chunk_nt, variant="", cubin=False) -> bytes:
    """nsfrb_jit_stream_kernel: CUDA source (or sm_100a cubin) of the plan-specialised real-time kernel.
    Needs no GPU."""
    f = np.ascontiguousarray(freqs_GHz, dtype=np.float64)
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    w = np.ascontiguousarray(width_list, dtype=np.int32)
    f64p, i32p = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    args = (int(nx), int(ny), int(nchan), int(nt), f.ctypes.data_as(f64p), float(tsamp_s), dm.ctypes.data_as(f64p), dm.size,
            w.ctypes.data_as(i32p), w.size, int(chunk_nt), variant.encode(), int(bool(cubin)))
    need = ctypes.c_size_t(0)
    _check(lib().nsfrb_jit_stream_kernel(*args, None, 0, ctypes.byref(need)))
    buf = ctypes.create_string_buffer(need.value)
    _check(lib().nsfrb_jit_stream_kernel(*args, buf, need.value, ctypes.byref(need)))
    return buf.raw[: need.value]


def jit_search_kernel(nx, ny, nchan, nt, freqs_GHz, tsamp_s, dm_list, width_list, cubin=False) -> bytes:
    """nsfrb_jit_search_kernel: CUDA source (or sm_100a cubin) of the plan-specialised offline kernel.  Needs no GPU."""
    f = np.ascontiguousarray(freqs_GHz, dtype=np.float64)
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    w = np.ascontiguousarray(width_list, dtype=np.int32)
    f64p, i32p = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    args = (int(nx), int(ny), int(nchan), int(nt), f.ctypes.data_as(f64p), float(tsamp_s), dm.ctypes.data_as(f64p), dm.size,
            w.ctypes.data_as(i32p), w.size, int(bool(cubin)))
    need = ctypes.c_size_t(0)
    _check(lib().nsfrb_jit_search_kernel(*args, None, 0, ctypes.byref(need)))
    buf = ctypes.create_string_buffer(need.value)
    _check(lib().nsfrb_jit_search_kernel(*args, buf, need.value, ctypes.byref(need)))
    return buf.raw[: need.value]


def measure_peaks(iters: int = 2000) -> dict:
    """nsfrb_measure_peaks: {test name: (operations or words per second, per SM clock per SM)} of the current device."""
    L = lib()
    n = L.nsfrb_peaks_count()
    a, b = (ctypes.c_double * n)(), (ctypes.c_double * n)()
    _check(L.nsfrb_measure_peaks(int(iters), a, b, int(torch.cuda.current_stream().cuda_stream)))
    return {L.nsfrb_peaks_name(i).decode(): (float(a[i]), float(b[i])) for i in range(n)}


def bin_time(cube: torch.Tensor, factor: int, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """nsfrb_bin_time on a device cube [nchan][nt][npix] float32 -> [nchan][nt // factor][npix] (asynchronous)."""
    if not cube.is_cuda or cube.dtype != torch.float32 or not cube.is_contiguous() or cube.dim() != 3:
        raise ValueError("expected a contiguous float32 CUDA tensor [nchan][nt][npix]")
    nchan, nt, npix = cube.shape
    if out is None:
        out = torch.empty((nchan, nt // int(factor) if factor >= 1 else 0, npix), dtype=torch.float32, device=cube.device)
    if factor >= 1 and nt // int(factor) == 0:
        return out  # nothing left to compute
    s = torch.cuda.current_stream() if stream is None else stream
    _check(lib().nsfrb_bin_time(cube.data_ptr(), nchan, nt, npix, int(factor), out.data_ptr(), int(s.cuda_stream)))
    return out


def median_subtract(cube: torch.Tensor, out: torch.Tensor | None = None, want_median: bool = True, stream=None):
    """nsfrb_median_subtract on a device cube [nchan][nt][npix] float32 -> (out, median [nchan][npix] or None);
    out=cube works in place (asynchronous)."""
    if not cube.is_cuda or cube.dtype != torch.float32 or not cube.is_contiguous() or cube.dim() != 3:
        raise ValueError("expected a contiguous float32 CUDA tensor [nchan][nt][npix]")
    nchan, nt, npix = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    elif out.shape != cube.shape or out.dtype != cube.dtype or not out.is_contiguous() or out.device != cube.device:
        raise ValueError("out must match the cube")
    med = torch.empty((nchan, npix), dtype=torch.float32, device=cube.device) if want_median else None
    s = torch.cuda.current_stream() if stream is None else stream
    _check(lib().nsfrb_median_subtract(cube.data_ptr(), nchan, nt, npix, out.data_ptr(),
                                       med.data_ptr() if med is not None else None, int(s.cuda_stream)))
    return out, med


def psf_mask(psf: torch.Tensor, percentile: float = 90.0, stream=None):
    """nsfrb_psf_mask on a device PSF [mh][mw] float32 -> (mask uint8 [mh][mw], value float64 [1]) (asynchronous)."""
    if not psf.is_cuda or psf.dtype != torch.float32 or not psf.is_contiguous() or psf.dim() != 2:
        raise ValueError("expected a contiguous float32 CUDA tensor [mh][mw]")
    mask = torch.empty(psf.shape, dtype=torch.uint8, device=psf.device)
    value = torch.empty(1, dtype=torch.float64, device=psf.device)
    s = torch.cuda.current_stream() if stream is None else stream
    _check(lib().nsfrb_psf_mask(psf.data_ptr(), psf.shape[0], psf.shape[1], float(percentile), mask.data_ptr(),
                                value.data_ptr(), int(s.cuda_stream)))
    return mask, value


@dataclass
class ClusterResult:
    top: torch.Tensor       # [topn*20] uint8 (raw nsfrb_cand records, rank order)
    wsnr: torch.Tensor      # [topn] float64
    members: torch.Tensor   # [topn] int32
    result: torch.Tensor    # [2] int32: n_found, best

    def to_host(self) -> dict:
        """Synchronises; the found candidates only."""
        n, best = (int(v) for v in self.result.cpu())
        cands = self.top.cpu().numpy().view(CAND_DTYPE)[:n].copy()
        return dict(cands=cands, pixels=[int(p) for p in cands["pixel"]], wsnr=self.wsnr.cpu().numpy()[:n].tolist(),
                    members=self.members.cpu().numpy()[:n].tolist(), best=best)


def alloc_cluster_result(topn: int, device="cuda") -> ClusterResult:
    """Output buffers of nsfrb_cluster / nsfrb_cluster_static for `topn` candidates (reusable from call to call)."""
    n = max(int(topn), 1)
    return ClusterResult(torch.empty(n * CAND_DTYPE.itemsize, dtype=torch.uint8, device=device),
                         torch.empty(n, dtype=torch.float64, device=device),
                         torch.empty(n, dtype=torch.int32, device=device), torch.empty(2, dtype=torch.int32, device=device))


def cluster_static(snr_map: torch.Tensor, argmax: torch.Tensor, nx: int, ny: int, threshold: float, psf: torch.Tensor,
                   mask: torch.Tensor, topn: int = 10, out: ClusterResult | None = None, stream=None) -> ClusterResult:
    """nsfrb_cluster_static: nsfrb_cluster without a plan and without any device allocation inside the library (its
    workspace is a fixed array in the library's device image).  Pass `out` (alloc_cluster_result) to reuse the output
    buffers; calls must not overlap on the GPU (they share the workspace)."""
    res = out if out is not None else alloc_cluster_result(topn, snr_map.device)
    s = torch.cuda.current_stream() if stream is None else stream
    _check(lib().nsfrb_cluster_static(int(nx), int(ny), float(threshold), snr_map.data_ptr(), argmax.data_ptr(),
                                      psf.data_ptr(), mask.data_ptr(), psf.shape[0], psf.shape[1], int(topn),
                                      res.top.data_ptr(), res.wsnr.data_ptr(), res.members.data_ptr(), res.result.data_ptr(),
                                      int(s.cuda_stream)))
    return res


class Imager:
    """nsfrb_imager_create / nsfrb_imager_image / nsfrb_imager_destroy (NEXT 4: visibilities -> images)."""

    def __init__(self, n, pixel_rad, uv_m, freqs_GHz, bmin_m=20.0, bmax_m=485.0, robust=-2.0):
        uv = np.ascontiguousarray(uv_m, dtype=np.float64)
        f = np.ascontiguousarray(freqs_GHz, dtype=np.float64)
        self.n, self.nbase, self.nchan = int(n), uv.shape[0], f.size
        self._h = ctypes.c_void_p()
        f64p = ctypes.POINTER(ctypes.c_double)
        _check(lib().nsfrb_imager_create(ctypes.byref(self._h), self.n, float(pixel_rad), uv.ctypes.data_as(f64p), self.nbase,
                                         f.ctypes.data_as(f64p), self.nchan, float(bmin_m), float(bmax_m), float(robust)))

    def table(self):
        cells = np.zeros((self.nchan, self.nbase, 2), dtype=np.int32)
        w = np.zeros((self.nchan, self.nbase), dtype=np.float64)
        _check(lib().nsfrb_imager_get_table(self._h, cells.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                                            w.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
        return cells, w

    def image(self, vis: torch.Tensor, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
        """vis: CUDA complex64 [nt][nchan][nbase][2] -> float32 [nt][n*n] (asynchronous)."""
        if not (vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous() and vis.dim() == 4
                and tuple(vis.shape[1:]) == (self.nchan, self.nbase, 2)):
            raise ValueError("vis must be a contiguous complex64 CUDA tensor [nt][nchan][nbase][2]")
        nt = vis.shape[0]
        if out is None:
            out = torch.empty((nt, self.n * self.n), dtype=torch.float32, device=vis.device)
        s = torch.cuda.current_stream() if stream is None else stream
        _check(lib().nsfrb_imager_image(self._h, vis.data_ptr(), nt, out.data_ptr(), int(s.cuda_stream)))
        return out

    def close(self):
        if self._h:
            lib().nsfrb_imager_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


class Plan:
    """nsfrb_plan_create / nsfrb_search / nsfrb_stream_push / nsfrb_plan_destroy."""

    def __init__(self, nx, ny, nchan, nt, freqs_GHz, tsamp_s, dm_list, width_list, threshold, cand_capacity=4096):
        f = np.ascontiguousarray(freqs_GHz, dtype=np.float64)
        dm = np.ascontiguousarray(dm_list, dtype=np.float64)
        w = np.ascontiguousarray(width_list, dtype=np.int32)
        if f.size != nchan:
            raise ValueError("len(freqs_GHz) != nchan")
        self._h = ctypes.c_void_p()
        self.nx, self.ny, self.npix, self.nchan, self.nt = int(nx), int(ny), int(nx) * int(ny), int(nchan), int(nt)
        self.ndm, self.nwidth = dm.size, w.size
        self.cand_capacity = int(cand_capacity)
        _check(lib().nsfrb_plan_create(
            ctypes.byref(self._h), int(nx), int(ny), int(nchan), int(nt),
            f.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), float(tsamp_s),
            dm.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), dm.size,
            w.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), w.size, float(threshold)))
        self.device = torch.device("cuda", torch.cuda.current_device())

    @classmethod
    def for_workload(cls, wl, **kw) -> "Plan":
        return cls(wl.nx, wl.ny, wl.nchan, wl.nt, wl.freqs_GHz, wl.tsamp_s, wl.dm_list, wl.width_list, wl.threshold, **kw)

    # -- plan facts
    def delays(self) -> np.ndarray:
        out = np.empty((self.ndm, self.nchan), dtype=np.int32)
        _check(lib().nsfrb_plan_get_delays(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))))
        return out

    def info(self) -> dict:
        s = nsfrb_plan_info()
        _check(lib().nsfrb_plan_get_info(self._h, ctypes.byref(s)))
        return {n: int(getattr(s, n)) for n, _ in s._fields_}

    def prepare(self, stream_chunk_nt: int | None = None):
        """nsfrb_plan_prepare: compile the plan's kernel and allocate its workspaces now (offline search by default, the
        real-time path for pushes of stream_chunk_nt samples otherwise)."""
        if stream_chunk_nt is None:
            _check(lib().nsfrb_plan_prepare(self._h, 0, 0))
        else:
            _check(lib().nsfrb_plan_prepare(self._h, 1, int(stream_chunk_nt)))
        return self

    def last_launches(self) -> int:
        return int(lib().nsfrb_plan_last_launches(self._h))

    def stream_mode(self) -> int:
        """nsfrb_stream_mode: 0 no streaming state yet, 1 raw ring, 2 + dedispersed history, 3 + its block sums."""
        return int(lib().nsfrb_stream_mode(self._h))

    def set_profiling(self, on: bool = True):
        _check(lib().nsfrb_plan_set_profiling(self._h, int(on)))

    def kernel_ms(self) -> dict:
        """Device milliseconds of the last call's kernels (needs set_profiling(True)); synchronises."""
        a = (ctypes.c_float * 4)()
        _check(lib().nsfrb_plan_get_kernel_ms(self._h, a))
        return {"layout": a[0], "search": a[1], "finalize": a[2], "compact": a[3]}

    # -- outputs
    def alloc_outputs(self) -> SearchResult:
        dev = self.device
        return SearchResult(
            torch.empty(self.npix, dtype=torch.float32, device=dev),
            torch.empty((3, self.npix), dtype=torch.int32, device=dev),
            torch.empty(max(self.cand_capacity, 1) * CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev),
            torch.zeros(1, dtype=torch.int32, device=dev))

    @staticmethod
    def _stream_handle(stream) -> int:
        s = torch.cuda.current_stream() if stream is None else stream
        return int(s.cuda_stream)

    def search(self, cube: torch.Tensor, out: SearchResult | None = None, stream=None) -> SearchResult:
        """nsfrb_search on a device cube [nchan][nt][npix] float32 (asynchronous on `stream`)."""
        self._check_dev(cube, (self.nchan, self.nt, self.npix))
        out = out or self.alloc_outputs()
        _check(lib().nsfrb_search(self._h, cube.data_ptr(), self._stream_handle(stream), out.snr_map.data_ptr(),
                                  out.argmax.data_ptr(), out.cands.data_ptr(), self.cand_capacity,
                                  out.ncands.data_ptr()))
        return out

    def stream_push(self, chunk: torch.Tensor, out: SearchResult | None = None, stream=None) -> SearchResult:
        """nsfrb_stream_push of a device chunk [nchan][chunk_nt][npix] float32."""
        if chunk.dim() != 3:
            raise ValueError("chunk must be [nchan][chunk_nt][npix]")
        self._check_dev(chunk, (self.nchan, chunk.shape[1], self.npix))
        out = out or self.alloc_outputs()
        _check(lib().nsfrb_stream_push(self._h, chunk.data_ptr(), int(chunk.shape[1]), self._stream_handle(stream),
                                       out.snr_map.data_ptr(), out.argmax.data_ptr(), out.cands.data_ptr(),
                                       self.cand_capacity, out.ncands.data_ptr()))
        return out

    def stream_set_cubes(self, snr_cube: torch.Tensor | None, toa_cube: torch.Tensor | None):
        """nsfrb_stream_set_cubes: per-(dm, width, pixel) peak S/N [ndm][nwidth][npix] float32 and window start (int32)
        written by every later push; None, None switches them off.  The tensors must stay alive."""
        if snr_cube is None and toa_cube is None:
            _check(lib().nsfrb_stream_set_cubes(self._h, None, None))
            self._cubes = None
            return
        shape = (self.ndm, self.nwidth, self.npix)
        for t, dt in ((snr_cube, torch.float32), (toa_cube, torch.int32)):
            if t is None or not t.is_cuda or t.dtype != dt or not t.is_contiguous() or tuple(t.shape) != shape:
                raise ValueError(f"cubes must be contiguous CUDA tensors of shape {shape} (float32 / int32)")
        _check(lib().nsfrb_stream_set_cubes(self._h, snr_cube.data_ptr(), toa_cube.data_ptr()))
        self._cubes = (snr_cube, toa_cube)

    def stream_reset(self):
        _check(lib().nsfrb_stream_reset(self._h))

    def stream_set_running_sigma(self, alpha: float, snr_map_run: torch.Tensor | None, argmax_run: torch.Tensor | None):
        """nsfrb_stream_set_running_sigma: every later push also writes the maps normalised by the running standard
        deviation (float32 [npix], int32 [3][npix]); None, None switches the mode off.  The tensors must stay alive."""
        if snr_map_run is None and argmax_run is None:
            _check(lib().nsfrb_stream_set_running_sigma(self._h, float(alpha), None, None))
            self._running = None
            return
        ok = (snr_map_run is not None and argmax_run is not None and snr_map_run.is_cuda and argmax_run.is_cuda
              and snr_map_run.dtype == torch.float32 and argmax_run.dtype == torch.int32
              and snr_map_run.is_contiguous() and argmax_run.is_contiguous()
              and snr_map_run.numel() == self.npix and tuple(argmax_run.shape) == (3, self.npix))
        if not ok:
            raise ValueError("expected contiguous CUDA tensors float32 [npix] and int32 [3][npix]")
        _check(lib().nsfrb_stream_set_running_sigma(self._h, float(alpha), snr_map_run.data_ptr(), argmax_run.data_ptr()))
        self._running = (snr_map_run, argmax_run)

    def cluster(self, snr_map: torch.Tensor, argmax: torch.Tensor, psf: torch.Tensor, mask: torch.Tensor, topn: int = 10,
                stream=None) -> ClusterResult:
        """nsfrb_cluster: the topn best candidates of (snr_map, argmax) and their PSF-mask weighted mean S/N."""
        if not (snr_map.is_cuda and snr_map.dtype == torch.float32 and snr_map.is_contiguous()
                and snr_map.numel() == self.npix):
            raise ValueError("snr_map must be a contiguous float32 CUDA tensor of npix elements")
        if not (argmax.is_cuda and argmax.dtype == torch.int32 and argmax.is_contiguous()
                and tuple(argmax.shape) == (3, self.npix)):
            raise ValueError("argmax must be a contiguous int32 CUDA tensor [3][npix]")
        if not (psf.is_cuda and psf.dtype == torch.float32 and psf.is_contiguous() and psf.dim() == 2
                and mask.is_cuda and mask.dtype == torch.uint8 and mask.is_contiguous() and mask.shape == psf.shape):
            raise ValueError("psf / mask must be contiguous CUDA tensors [mh][mw] (float32 / uint8)")
        n = max(int(topn), 1)
        dev = self.device
        res = ClusterResult(torch.empty(n * CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev),
                            torch.empty(n, dtype=torch.float64, device=dev),
                            torch.empty(n, dtype=torch.int32, device=dev), torch.empty(2, dtype=torch.int32, device=dev))
        s = torch.cuda.current_stream() if stream is None else stream
        _check(lib().nsfrb_cluster(self._h, snr_map.data_ptr(), argmax.data_ptr(), psf.data_ptr(), mask.data_ptr(),
                                   psf.shape[0], psf.shape[1], int(topn), res.top.data_ptr(), res.wsnr.data_ptr(),
                                   res.members.data_ptr(), res.result.data_ptr(), int(s.cuda_stream)))
        return res

    # -- host-buffer variants (H2D, search, D2H, synchronise) used for the end-to-end number
    def _host_out(self):
        pin = torch.cuda.is_available()
        return (torch.empty(self.npix, dtype=torch.float32, pin_memory=pin),
                torch.empty((3, self.npix), dtype=torch.int32, pin_memory=pin),
                torch.empty(max(self.cand_capacity, 1) * CAND_DTYPE.itemsize, dtype=torch.uint8, pin_memory=pin),
                torch.zeros(1, dtype=torch.int32, pin_memory=pin))

    def search_host(self, cube_host: torch.Tensor, out=None, stream=None):
        self._check_host(cube_host, (self.nchan, self.nt, self.npix))
        out = out or self._host_out()
        _check(lib().nsfrb_search_host(self._h, cube_host.data_ptr(), self._stream_handle(stream), out[0].data_ptr(),
                                       out[1].data_ptr(), out[2].data_ptr(), self.cand_capacity, out[3].data_ptr()))
        return out

    def stream_push_host(self, chunk_host: torch.Tensor, out=None, stream=None):
        self._check_host(chunk_host, (self.nchan, chunk_host.shape[1], self.npix))
        out = out or self._host_out()
        _check(lib().nsfrb_stream_push_host(self._h, chunk_host.data_ptr(), int(chunk_host.shape[1]),
                                            self._stream_handle(stream), out[0].data_ptr(), out[1].data_ptr(),
                                            out[2].data_ptr(), self.cand_capacity, out[3].data_ptr()))
        return out

    def stream_push_host_async(self, chunk_host: torch.Tensor, out):
        """nsfrb_stream_push_host_async: returns at once; `out` (from _host_out(), pinned) is valid after stream_wait()
        or after the second following call.  Keep chunk_host and out alive and untouched until then."""
        self._check_host(chunk_host, (self.nchan, chunk_host.shape[1], self.npix))
        _check(lib().nsfrb_stream_push_host_async(self._h, chunk_host.data_ptr(), int(chunk_host.shape[1]),
                                                  out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(),
                                                  self.cand_capacity, out[3].data_ptr()))
        return out

    def stream_wait(self):
        _check(lib().nsfrb_stream_wait(self._h))

    # -- checks / lifetime
    def _check_dev(self, t, shape):
        if not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
            raise ValueError(f"expected contiguous float32 CUDA tensor of shape {shape}, got {tuple(t.shape)} {t.dtype} {t.device}")

    def _check_host(self, t, shape):
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
            raise ValueError(f"expected contiguous float32 host tensor of shape {shape}")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().nsfrb_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()
