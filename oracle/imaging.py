"""Oracle for the upstream imaging step -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares nothing with
the CUDA path (no tables, no helpers, no imports either way).  Plain numpy, float64 / complex128, written in the order of the paper:

  PAPER.md:L55  "grids visibilities with baseline lengths b > b_min = 20 m from the dense 82-antenna 'core'
                 (b < b_max = 485 m) to a 175 x 175-pixel UV-grid.  The core is assumed to be coplanar, so the W-term is
                 neglected ...  The two visibility polarizations are summed, then approximately uniform weighting (Briggs
                 robustness parameter R = -2; D. S. Briggs 1995) is applied to accumulate visibilities, and a 2-dimensional
                 inverse-FFT is applied to form the final image"
  PAPER.md:L61  (fn. 10) "np.fft.ifft2 ... The visibility grid is first shifted using np.fft.ifftshift to properly order the
                 zero-frequency component; np.fft.ifftshift is then applied to the resulting image."
  PAPER.md:L67  "Each of the 8 channels are imaged individually, then summed together to form a single image for each 134 ms
                 time sample."

Where the paper is silent the readings I1..I6 of DESIGN.md apply (nearest-cell gridding, Hermitian copy, Briggs' formula,
normalisation to unit point-source response, real part).  Pins: tests/test_imaging_pins.py.
"""
from __future__ import annotations

import numpy as np

C_M_PER_S = 299792458.0


def select_baselines(uv_m: np.ndarray, bmin_m: float = 20.0, bmax_m: float = 485.0) -> np.ndarray:
    """L55: indices of the baselines with bmin < b < bmax, b = sqrt(u^2 + v^2) in metres (W-term neglected)."""
    uv_m = np.asarray(uv_m, dtype=np.float64)
    b = np.sqrt(uv_m[:, 0] * uv_m[:, 0] + uv_m[:, 1] * uv_m[:, 1])
    return np.nonzero((b > bmin_m) & (b < bmax_m))[0]


def uv_cells(uv_m: np.ndarray, freq_GHz: float, n: int, pixel_rad: float) -> np.ndarray:
    """Reading I1: nearest UV cell of every baseline at one channel.  u in wavelengths = u_m * f / c; the grid spacing that
    makes an n-pixel image of pixel size `pixel_rad` is du = 1 / (n * pixel_rad); cell = floor(u / du + 0.5).
    Returns int64 [nb][2] = (fu, fv), the signed offsets from the grid centre n // 2."""
    uv_m = np.asarray(uv_m, dtype=np.float64)
    scale = (freq_GHz * 1.0e9 / C_M_PER_S) * (n * pixel_rad)      # metres -> cells
    return np.floor(uv_m * scale + 0.5).astype(np.int64)


def briggs_weights(cells: np.ndarray, n: int, robust: float = -2.0) -> np.ndarray:
    """Reading I3 (D. S. Briggs 1995, the form every imager implements): with natural weights w_i = 1 and W_k the sum of the
    natural weights gridded into cell k (every visibility counted at its cell and at the Hermitian one),
        f^2 = (5 * 10^-R)^2 / (sum_k W_k^2 / sum_i w_i),       w'_i = w_i / (1 + W_k(i) f^2).
    R = -2 is 'approximately uniform' (w' ~ 1 / W_k).  Returns float64 [nb]; baselines whose cell falls outside the grid get 0."""
    c = n // 2
    W = np.zeros((n, n), dtype=np.float64)
    inside = np.zeros(len(cells), dtype=bool)
    for i, (fu, fv) in enumerate(cells):
        if 0 <= c + fu < n and 0 <= c - fu < n and 0 <= c + fv < n and 0 <= c - fv < n:
            inside[i] = True
            W[c + fv, c + fu] += 1.0
            W[c - fv, c - fu] += 1.0
    nvis = 2.0 * inside.sum()
    out = np.zeros(len(cells), dtype=np.float64)
    if nvis == 0:
        return out
    f2 = (5.0 * 10.0 ** (-robust)) ** 2 / (np.sum(W * W) / nvis)
    for i, (fu, fv) in enumerate(cells):
        if inside[i]:
            out[i] = 1.0 / (1.0 + W[c + fv, c + fu] * f2)
    return out


def grid_channel(vis: np.ndarray, cells: np.ndarray, weights: np.ndarray, n: int) -> np.ndarray:
    """Readings I1, I2: vis [nb][2 pol] complex -> the n x n UV grid of one channel and time sample.  The two polarisations
    are summed (L55); every visibility is accumulated with its weight at its nearest cell and its complex conjugate at the
    Hermitian cell, so the image is real."""
    c = n // 2
    G = np.zeros((n, n), dtype=np.complex128)
    for i, (fu, fv) in enumerate(cells):
        if weights[i] == 0.0:
            continue
        v = complex(vis[i, 0]) + complex(vis[i, 1])
        G[c + fv, c + fu] += weights[i] * v
        G[c - fv, c - fu] += weights[i] * np.conj(v)
    return G


def image_channel(G: np.ndarray) -> np.ndarray:
    """L61 (fn. 10), literally: ifftshift the grid, np.fft.ifft2, ifftshift the image.  Complex n x n."""
    return np.fft.ifftshift(np.fft.ifft2(np.fft.ifftshift(G)))


def image(vis: np.ndarray, uv_m: np.ndarray, freqs_GHz, n: int = 175, pixel_rad: float = 10.3 / 206264.80624709636,
          bmin_m: float = 20.0, bmax_m: float = 485.0, robust: float = -2.0) -> np.ndarray:
    """vis [nt][nchan][nbase][2 pol] complex -> images [nt][n][n] float64 (L55, L61, L67).
    Per time sample: every channel is gridded (its own cells and Briggs weights) and imaged individually, normalised so that
    a unit point source at the phase centre has value 1 at the centre pixel (reading I4: times n^2 / sum of the weights
    of both Hermitian halves), the real part taken (I5: the grid is Hermitian, the imaginary part is rounding), and the
    channel images are summed (L67)."""
    vis = np.asarray(vis)
    nt, nchan = vis.shape[0], vis.shape[1]
    sel = select_baselines(uv_m, bmin_m, bmax_m)
    uv_sel = np.asarray(uv_m, dtype=np.float64)[sel]
    out = np.zeros((nt, n, n), dtype=np.float64)
    for ch in range(nchan):
        cells = uv_cells(uv_sel, float(freqs_GHz[ch]), n, pixel_rad)
        w = briggs_weights(cells, n, robust)
        wsum = 2.0 * w.sum()
        if wsum == 0.0:
            continue
        for t in range(nt):
            G = grid_channel(vis[t, ch][sel], cells, w, n)
            out[t] += (image_channel(G) * (n * n / wsum)).real
    return out


def phase_centre_pixel(n: int) -> int:
    """Where the paper's route puts the phase centre (direction l = m = 0): np.fft.ifftshift of the image moves ifft2's
    index 0 to index n - n // 2, i.e. pixel 88 of 175 -- one past the centre pixel for odd n (fftshift would give n // 2;
    fn. 10 says ifftshift, and the oracle follows it)."""
    return (n - n // 2) % n


def direct_image(vis_tc: np.ndarray, cells: np.ndarray, weights: np.ndarray, n: int) -> np.ndarray:
    """Brute force for tiny n (a pin, not a route): the definition of the inverse DFT written out,
        I[y][x] = (1 / n^2) sum_i w_i ( V_i e^{+2 pi i (fu (x - x0) + fv (y - x0)) / n} + conj(V_i) e^{-2 pi i (...)/n} ),
    x0 = phase_centre_pixel(n).  (Frequency 0 sits at grid index n // 2: the first ifftshift moves it to index 0.)"""
    c = phase_centre_pixel(n)
    out = np.zeros((n, n), dtype=np.complex128)
    for y in range(n):
        for x in range(n):
            acc = 0.0 + 0.0j
            for i, (fu, fv) in enumerate(cells):
                if weights[i] == 0.0:
                    continue
                v = complex(vis_tc[i, 0]) + complex(vis_tc[i, 1])
                ph = np.exp(2j * np.pi * (fu * (x - c) + fv * (y - c)) / n)
                acc += weights[i] * (v * ph + np.conj(v) * np.conj(ph))
            out[y, x] = acc / (n * n)
    return out
