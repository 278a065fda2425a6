"""Seeded synthetic workloads shaped like the paper's (BASELINE.json configs C1..C5).

This module holds NONE of the method's arithmetic: no delay formula, no dedispersion,
no S/N.  It serves both the oracle (tests) and the CUDA path (tests, bench), which is why
every function that has to place a dispersed pulse takes the integer delay vector(s) as an
ARGUMENT -- the caller obtains them from its own side (oracle.delays() in tests,
nsfrb_plan_get_delays() in bench.py).

The paper measures on DSA-110 images that are not public; these cubes take the paper's
shapes (16 sub-bands over 1.28-1.53 GHz, 134.2 ms sampling, 25-sample chunks, boxcar
injections at trial DMs/widths) and stand in for them.
Recipe: DESIGN.md "Input recipe"; conventions: SURVEY.md sec. 8(d).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np
import torch

TSAMP_S = 0.1342  # PAPER.md:L48 (134 ms sampling), BASELINE.json configs


def log_widths(n: int, wmax: int = 1200) -> np.ndarray:
    """'n log-spaced widths 1..wmax' as a strictly increasing integer list (reading R12):
    w_i = floor(wmax^(i/(n-1)) + 0.5), then w_i = max(w_i, w_{i-1}+1)."""
    out = []
    for i in range(n):
        w = int(np.floor(float(wmax) ** (i / (n - 1)) + 0.5))
        if out and w <= out[-1]:
            w = out[-1] + 1
        out.append(w)
    return np.asarray(out, dtype=np.int32)


def subband_centres(nchan: int, lo: float = 1.28, hi: float = 1.53) -> np.ndarray:
    """Centres of nchan equal sub-bands of [lo, hi] GHz (16 sub-bands)."""
    return lo + (np.arange(nchan, dtype=np.float64) + 0.5) * (hi - lo) / nchan


@dataclass(frozen=True)
class Workload:
    name: str
    nx: int
    ny: int
    nchan: int
    nt: int                      # cube length, or ring length L when streaming
    freqs_GHz: np.ndarray
    dm_list: np.ndarray
    width_list: np.ndarray
    threshold: float
    seed: int
    tsamp_s: float = TSAMP_S
    n_pulses: int = 0
    s0_range: tuple = (8.0, 40.0)
    streaming: bool = False
    chunk_nt: int = 25
    pulses_per_100_chunks: int = 5
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def npix(self) -> int:
        return self.nx * self.ny

    def scaled(self, nx: int, ny: int, nt: int | None = None, n_pulses: int | None = None) -> "Workload":
        """Same grid/recipe on fewer pixels (and optionally a shorter cube) for parity tests."""
        return replace(self, nx=nx, ny=ny, nt=self.nt if nt is None else nt,
                       n_pulses=self.n_pulses if n_pulses is None else n_pulses,
                       name=f"{self.name}[{nx}x{ny}x{self.nt if nt is None else nt}]")


def config(name: str) -> Workload:
    """The five BASELINE.json configs (full size)."""
    name = name.lower()
    if name == "c1":
        return Workload("c1", 32, 32, 8, 64, np.linspace(1.311, 1.499, 8), np.linspace(0.0, 1400.0, 8),
                        np.asarray([1, 2, 4, 8], dtype=np.int32), 6.0, seed=0, n_pulses=1,
                        note="tiny correctness cube; one pulse at (x,y)=(11,20), DM 500, w 4, t0 30, A 1.5")
    if name == "c2":
        return Workload("c2", 256, 256, 16, 1536, subband_centres(16), np.linspace(0.0, 2000.0, 16),
                        log_widths(20), 8.0, seed=2, streaming=True, chunk_nt=25, s0_range=(8.0, 40.0),
                        note="real-time: 1536-sample ring, 25-sample pushes, per-pixel sigma U(0.5,2)")
    if name == "c3":
        return Workload("c3", 301, 301, 16, 4096, subband_centres(16), np.linspace(0.0, 3000.0, 32),
                        log_widths(24), 8.0, seed=3, n_pulses=50, s0_range=(8.0, 40.0),
                        note="offline full cube; 20 constant point sources; ~10 of 50 pulses are periodic trains")
    if name == "c4":
        return Workload("c4", 1024, 1024, 16, 512, subband_centres(16), np.linspace(0.0, 1500.0, 64),
                        np.asarray([1, 2, 3, 5, 8, 13, 21, 34, 55, 89, 144, 233], dtype=np.int32), 8.0,
                        seed=4, n_pulses=200, s0_range=(8.0, 40.0),
                        note="survey mosaic, ~34 GB cube; per-channel gain U(0.8,1.2)")
    if name == "c5":
        return Workload("c5", 128, 128, 64, 8192, subband_centres(64), np.linspace(0.0, 5000.0, 256),
                        log_widths(32), 6.0, seed=5, n_pulses=100, s0_range=(6.0, 100.0),
                        note="DM/width stress; RFI-like spikes in channels 13 and 41")
    if name == "paper":
        # the grid the paper itself runs in real time: 301x301 px, 16 sub-bands, 16 DM trials
        # 171-4000 pc/cm^3, log2 widths 1-16 samples, 25-sample chunks, 8.5 sigma; the ring length is ours (as C2)
        return Workload("paper", 301, 301, 16, 1536, subband_centres(16), np.linspace(171.0, 4000.0, 16),
                        np.asarray([1, 2, 4, 8, 16], dtype=np.int32), 8.5, seed=12, streaming=True, chunk_nt=25,
                        s0_range=(8.0, 40.0), note="the paper's own real-time grid: 16 DM x 5 log2 widths, 301x301 px")
    raise ValueError(f"unknown config {name!r}")


# --------------------------------------------------------------------------------------
# noise / sky / RFI  (no method arithmetic)
# --------------------------------------------------------------------------------------
def _gen(device, seed):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def pixel_sigma(wl: Workload, device="cpu") -> torch.Tensor:
    """C2: per-pixel noise sigma ~ U(0.5, 2), fixed per pixel; 1 elsewhere."""
    if wl.name.startswith("c2"):
        rng = np.random.default_rng(wl.seed + 7000)
        return torch.from_numpy(rng.uniform(0.5, 2.0, wl.npix).astype(np.float32)).to(device)
    return torch.ones(wl.npix, dtype=torch.float32, device=device)


def make_cube(wl: Workload, device="cpu") -> torch.Tensor:
    """Noise (+ sky term, gains, RFI) cube [nchan][nt][npix] float32, no pulses yet.
    Filled one channel slab at a time so the 34 GB configs never need a second copy."""
    dev = torch.device(device)
    base = wl.name.split("[")[0]
    if base == "c1":
        # NumPy stream so it can be reproduced on any machine
        a = np.random.default_rng(0).standard_normal((wl.nchan, wl.nt, wl.npix)).astype(np.float32)
        return torch.from_numpy(a).to(dev)
    cube = torch.empty((wl.nchan, wl.nt, wl.npix), dtype=torch.float32, device=dev)
    g = _gen(dev, wl.seed)
    rng = np.random.default_rng(wl.seed + 500)
    gains = rng.uniform(0.8, 1.2, wl.nchan) if base == "c4" else np.ones(wl.nchan)
    sig = pixel_sigma(wl, dev)
    for c in range(wl.nchan):
        cube[c].normal_(0.0, 1.0, generator=g)
        if base == "c2":
            cube[c].mul_(sig[None, :])
        if base == "c4":
            cube[c].mul_(float(gains[c]))
    if base == "c3":
        # 20 single-pixel sources, constant flux U(0.2,3) sigma in every channel and sample
        n_src = min(20, wl.npix)
        src_p = rng.choice(wl.npix, n_src, replace=False)
        flux = rng.uniform(0.2, 3.0, n_src).astype(np.float32)
        cube[:, :, torch.as_tensor(src_p, device=dev)] += torch.as_tensor(flux, device=dev)[None, None, :]
    if base == "c5":
        # zero-DM RFI: +10 on a Bernoulli(0.01) set of samples, same samples for all pixels
        for c in (13, 41):
            if c < wl.nchan:
                hit = np.nonzero(rng.random(wl.nt) < 0.01)[0]
                if hit.size:
                    cube[c, torch.as_tensor(hit, device=dev), :] += 10.0
    return cube


# --------------------------------------------------------------------------------------
# injections: boxcar in time, same amplitude per channel, at TRIAL DMs/widths
# --------------------------------------------------------------------------------------
@dataclass
class Pulse:
    pixel: int
    dm_idx: int
    width_idx: int
    t0: int          # start sample in the reference-frequency frame (absolute index when streaming)
    width: int
    s0: float        # nominal S0 = A*w*nchan/(sigma*sqrt(w*nchan))
    amp: float       # per-channel amplitude A
    train_period: int = 0   # >0: repeated every train_period samples over the whole cube


def injection_table(wl: Workload, delay_table: np.ndarray) -> list[Pulse]:
    """Seeded pulse list for an offline cube.  `delay_table` is the caller's int32 [ndm][nchan]
    table (needed only to keep each pulse inside its trial's valid range)."""
    base = wl.name.split("[")[0]
    d = np.asarray(delay_table)
    if base == "c1":
        # BASELINE.json config 1: pixel (x,y)=(11,20) => p = 20*nx+11 (reading R23)
        return [Pulse(pixel=20 * wl.nx + 11, dm_idx=-1, width_idx=2, t0=30, width=4, s0=float("nan"), amp=1.5)]
    rng = np.random.default_rng(1000 + int(base[1:]))
    n = min(wl.n_pulses, wl.npix)
    pix = rng.choice(wl.npix, n, replace=False)
    sig = pixel_sigma(wl).numpy()
    out = []
    for i in range(n):
        k = int(rng.integers(0, len(wl.dm_list)))
        T_k = wl.nt - int(d[k].max())
        ok = [j for j, w in enumerate(wl.width_list) if w <= T_k]
        j = int(ok[int(rng.integers(0, len(ok)))])
        w = int(wl.width_list[j])
        period = 0
        if base == "c3" and i < max(1, n // 5):
            # periodic train: period 75..373 samples (10-50 s), duty cycle <= 10 %
            period = int(rng.integers(75, 374))
            okw = [jj for jj, ww in enumerate(wl.width_list) if ww <= period // 10 and ww <= T_k]
            j = int(okw[int(rng.integers(0, len(okw)))])
            w = int(wl.width_list[j])
        t0 = int(rng.integers(0, T_k - w + 1)) if not period else int(rng.integers(0, min(period, T_k - w + 1)))
        s0 = float(rng.uniform(*wl.s0_range))
        amp = s0 * float(sig[pix[i]]) / np.sqrt(w * wl.nchan)
        out.append(Pulse(int(pix[i]), k, j, t0, w, s0, float(amp), period))
    return out


def inject(cube: torch.Tensor, pulses: list[Pulse], delay_table: np.ndarray, *, extra_delays=None) -> None:
    """Add the pulses in place: I[c][t0 + d[c] .. + w)[pixel] += A for every channel.
    delay_table[k] is the trial's delay vector; a pulse with dm_idx < 0 uses extra_delays (C1's DM 500)."""
    nchan, nt, _ = cube.shape
    for pu in pulses:
        dvec = np.asarray(extra_delays if pu.dm_idx < 0 else delay_table[pu.dm_idx])
        starts = [pu.t0] if not pu.train_period else list(range(pu.t0, nt, pu.train_period))
        for c in range(nchan):
            for s in starts:
                a, b = s + int(dvec[c]), s + int(dvec[c]) + pu.width
                a, b = max(a, 0), min(b, nt)
                if b > a:
                    cube[c, a:b, pu.pixel] += pu.amp


# --------------------------------------------------------------------------------------
# streaming (C2): chunks with pulses placed on the absolute time axis
# --------------------------------------------------------------------------------------
def stream_pulses(wl: Workload, delay_table: np.ndarray, n_chunks: int) -> list[Pulse]:
    """pulses_per_100_chunks seeded pulses per 100 chunks, random trial DM/width, S0 in s0_range."""
    d = np.asarray(delay_table)
    rng = np.random.default_rng(1000 + 2)
    n = max(1, (n_chunks * wl.pulses_per_100_chunks) // 100)
    n = min(n, wl.npix)
    pix = rng.choice(wl.npix, n, replace=False)
    sig = pixel_sigma(wl).numpy()
    total = n_chunks * wl.chunk_nt
    out = []
    for i in range(n):
        k = int(rng.integers(0, len(wl.dm_list)))
        ok = [j for j, w in enumerate(wl.width_list) if w + int(d[k].max()) < min(wl.nt, total)]
        j = int(ok[int(rng.integers(0, len(ok)))])
        w = int(wl.width_list[j])
        t0 = int(rng.integers(0, max(1, total - w - int(d[k].max()))))
        s0 = float(rng.uniform(*wl.s0_range))
        out.append(Pulse(int(pix[i]), k, j, t0, w, s0, float(s0 * sig[pix[i]] / np.sqrt(w * wl.nchan))))
    return out


class ChunkSource:
    """Seeded generator of [nchan][chunk_nt][npix] chunks: noise * sigma_p + the parts of
    each pulse that fall inside the chunk."""

    def __init__(self, wl: Workload, delay_table: np.ndarray, n_chunks: int, device="cpu"):
        self.wl, self.dev = wl, torch.device(device)
        self.d = np.asarray(delay_table)
        self.pulses = stream_pulses(wl, delay_table, n_chunks)
        self.sig = pixel_sigma(wl, self.dev)
        self.g = _gen(self.dev, wl.seed)
        self.n = 0

    def next(self, out: torch.Tensor | None = None) -> torch.Tensor:
        wl = self.wl
        if out is None:
            out = torch.empty((wl.nchan, wl.chunk_nt, wl.npix), dtype=torch.float32, device=self.dev)
        out.normal_(0.0, 1.0, generator=self.g)
        out.mul_(self.sig[None, None, :])
        a0, a1 = self.n, self.n + wl.chunk_nt
        for pu in self.pulses:
            dv = self.d[pu.dm_idx]
            if pu.t0 + int(dv.max()) + pu.width <= a0 or pu.t0 >= a1:
                continue
            for c in range(wl.nchan):
                a, b = max(pu.t0 + int(dv[c]), a0), min(pu.t0 + int(dv[c]) + pu.width, a1)
                if b > a:
                    out[c, a - a0:b - a0, pu.pixel] += pu.amp
        self.n = a1
        return out


# ---- inputs of the post-search candidate selection (nsfrb_psf_mask / nsfrb_cluster) -------------------

def synthetic_psf(size: int = 301, seed: int = 0, n_ant: int = 24) -> np.ndarray:
    """A simulated dirty beam [size][size] float32, peak 1 at [size//2][size//2] (stands in for the paper's
    "simulated PSF", L94; the DSA-110 one is not public).  Antennas on a mostly east-west line with a few
    north-south outriggers (L46: the array is east-west dominated), one frequency: the beam is the mean over
    baselines of cos(2 pi (u x + v y)), so it has a narrow main lobe, a north-south elongation and sidelobes."""
    rng = np.random.default_rng(1000 + seed)
    ew = np.sort(rng.uniform(-1.0, 1.0, n_ant))
    ns = np.where(rng.random(n_ant) < 0.25, rng.uniform(-0.5, 0.5, n_ant), rng.normal(0.0, 0.01, n_ant))
    i, j = np.triu_indices(n_ant, 1)
    u = (ew[i] - ew[j]) * 0.12                     # cycles per pixel at the longest baseline ~ 0.24
    v = (ns[i] - ns[j]) * 0.12
    r = np.arange(size) - size // 2
    px = np.exp(2j * np.pi * np.outer(u, r))       # [nbl][size]
    py = np.exp(2j * np.pi * np.outer(v, r))
    beam = np.real(np.einsum("by,bx->yx", py, px)) / u.size
    return np.ascontiguousarray(beam, dtype=np.float32)


def synthetic_snr_map(nx: int, ny: int, psf: np.ndarray, seed: int = 0, *, peak: float = 25.0, n_side: int = 6,
                      n_spurious: int = 3, background: float = 4.5):
    """A per-pixel peak-S/N map [ny][nx] float32 shaped like one with a bright source: noise-only pixels around
    `background` (the maximum of many trials), one source of S/N `peak`, `n_side` copies at the strongest PSF
    sidelobe offsets scaled by the PSF there, and `n_spurious` unrelated threshold crossings.  Returns
    (map, (x0, y0))."""
    rng = np.random.default_rng(2000 + seed)
    m = (background + 0.45 * rng.gumbel(size=(ny, nx))).astype(np.float32)
    x0, y0 = int(rng.integers(nx // 4, 3 * nx // 4)), int(rng.integers(ny // 4, 3 * ny // 4))
    mh, mw = psf.shape
    side = psf.astype(np.float64).copy()
    cy, cx = mh // 2, mw // 2
    side[max(0, cy - 3):cy + 4, max(0, cx - 3):cx + 4] = -np.inf      # not the main lobe itself
    placed = 0
    for flat in np.argsort(-side, axis=None):
        if placed == n_side:
            break
        dy, dx = int(flat // mw) - cy, int(flat % mw) - cx
        x, y = x0 + dx, y0 + dy
        if 0 <= x < nx and 0 <= y < ny:
            m[y, x] = np.float32(peak * float(psf[cy + dy, cx + dx]) + rng.normal(0.0, 0.5))
            side[max(0, cy + dy - 2):cy + dy + 3, max(0, cx + dx - 2):cx + dx + 3] = -np.inf
            placed += 1
    m[y0, x0] = np.float32(peak)
    for _ in range(n_spurious):
        m[int(rng.integers(ny)), int(rng.integers(nx))] = np.float32(rng.uniform(7.0, 12.0))
    return m, (x0, y0)


# ----------------------------------------------------------------------------- NEXT 4: synthetic visibilities (imaging)
IMG_N = 175                                   # 175 x 175-pixel UV grid / image
IMG_PIXEL_RAD = 10.3 / 206264.80624709636     # L55: 10.3 arcsec pixels
IMG_NANT, IMG_NCORE = 97, 82                  # Fig. 1 (L65): 97 antennas -> 4656 baselines (L48); L55: 82-antenna core


def imaging_array(seed: int = 0) -> np.ndarray:
    """Seeded stand-in for the DSA-110 layout (the real antenna positions are not in the paper): 82 core antennas on a
    mostly east-west line about 400 m long with a short north-south arm and metre-scale jitter (all core baselines < 485 m),
    plus 15 outriggers 0.6-2.5 km away (their baselines are cut by b_max).  Returns uv_m [4656][2] float64 = (east, north)
    separations in metres of every antenna pair i < j (W-term neglected, L55)."""
    rng = np.random.default_rng(9000 + seed)
    ew = np.stack([np.linspace(-200.0, 200.0, 62) + rng.uniform(-2.0, 2.0, 62), rng.uniform(-3.0, 3.0, 62)], axis=1)
    ns = np.stack([rng.uniform(-3.0, 3.0, 20) + 40.0, np.linspace(15.0, 230.0, 20) + rng.uniform(-2.0, 2.0, 20)], axis=1)
    ang = rng.uniform(0.0, 2.0 * np.pi, IMG_NANT - IMG_NCORE)
    rad = rng.uniform(600.0, 2500.0, IMG_NANT - IMG_NCORE)
    out = np.stack([rad * np.cos(ang), rad * np.sin(ang)], axis=1)
    pos = np.concatenate([ew, ns, out], axis=0)
    i, j = np.triu_indices(IMG_NANT, k=1)
    return (pos[j] - pos[i]).astype(np.float64)


def imaging_freqs(subband: int = 8, nchan: int = 8) -> np.ndarray:
    """Centres of the 8 x 1.46 MHz channels of one 11.7 MHz sub-band of the 187.5 MHz band centred on 1.4 GHz (L48)."""
    lo = 1.4 - 0.09375 + subband * 0.01171875
    return lo + (np.arange(nchan) + 0.5) * (0.01171875 / nchan)


def imaging_visibilities(uv_m: np.ndarray, freqs_GHz, nt: int, sources, noise: float = 0.0, seed: int = 0) -> np.ndarray:
    """vis [nt][nchan][nbase][2 pol] complex64: point sources (l_rad, m_rad, flux[, t_on, t_off]) with half the flux in each
    polarisation, V = S exp(-2 pi i (u l + v m)) with u, v in wavelengths, plus complex Gaussian noise of rms `noise` per
    polarisation.  (The paper images fringe-stopped, calibrated visibilities, L48-L55; these stand in for them.)"""
    rng = np.random.default_rng(9100 + seed)
    f = np.asarray(freqs_GHz, dtype=np.float64)
    uvl = uv_m[None, :, :] * (f[:, None, None] * 1.0e9 / 299792458.0)          # [nchan][nbase][2] wavelengths
    vis = np.zeros((nt, len(f), uv_m.shape[0], 2), dtype=np.complex128)
    for src in sources:
        l, m, flux = src[0], src[1], src[2]
        t_on, t_off = (src[3], src[4]) if len(src) >= 5 else (0, nt)
        ph = np.exp(-2j * np.pi * (uvl[:, :, 0] * l + uvl[:, :, 1] * m)) * (0.5 * flux)
        vis[t_on:t_off] += ph[None, :, :, None]
    if noise > 0.0:
        vis += noise * (rng.standard_normal(vis.shape) + 1j * rng.standard_normal(vis.shape)) / np.sqrt(2.0)
    return vis.astype(np.complex64)
