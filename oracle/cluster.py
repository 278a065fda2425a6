"""Oracle for the post-search candidate selection (second part) -- TEST INFRASTRUCTURE,
NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import it.

PAPER.md:L94: "Standard post-processing is limited to the 10 highest S/N candidates ... the PSF is thresholded at
the 90th percentile to make a binary mask, which is centered on each candidate in turn.  This candidate is treated
as the central PSF lobe, and any other candidates within the binary mask are identified as possible sidelobes.  The
weighted mean S/N is computed over the central and sidelobe candidate S/Ns.  After repeating with each candidate,
the maximum S/N is identified and its central lobe candidate's width, DM, position, and TOA are taken as the final,
most-likely candidate."

Plain numpy / Python loops in float64, written in the order of that passage.  The weights of the weighted mean
are a reading (R28): PARITY UNPINNED to the paper for them (no worked example is printed); everything else is pinned
in tests/test_cluster_pins.py.  Readings (R25..R28):
  R25  percentile = linear interpolation between order statistics at rank q/100*(n-1); mask = psf > that value.
  R26  candidates = per-pixel peaks with snr > threshold (O7, strict); the N highest, equal S/N -> smaller pixel.
  R27  the mask is centred by putting PSF element [mh//2][mw//2] on the central candidate; a candidate outside the
       PSF array is outside the mask; the central candidate is always a member.
  R28  weights of the "weighted mean S/N" (not stated in the paper) = the PSF value at the member's offset from the
       central candidate (so the central lobe weighs psf[mh//2][mw//2]); the final candidate is the centre with the
       largest weighted mean, equal means -> the higher-ranked (higher S/N) centre.
"""
from __future__ import annotations

import numpy as np


def percentile_value(values, q: float) -> float:
    """R25: q-th percentile of `values` by sorting and interpolating linearly between the two neighbouring order
    statistics (written out; pinned against numpy's routine in tests/test_cluster_pins.py)."""
    v = np.sort(np.asarray(values, dtype=np.float64).ravel())
    n = v.size
    if n == 0:
        raise ValueError("empty PSF")
    r = float(q) / 100.0 * (n - 1)
    lo = int(np.floor(r))
    lo = min(max(lo, 0), n - 1)
    hi = min(lo + 1, n - 1)
    frac = r - lo
    return float(v[lo] + frac * (v[hi] - v[lo]))


def psf_mask(psf, q: float = 90.0):
    """L94 "the PSF is thresholded at the 90th percentile to make a binary mask" -> (mask uint8 [mh][mw], value)."""
    psf = np.asarray(psf, dtype=np.float32)
    thr = percentile_value(psf, q)
    return (psf.astype(np.float64) > thr).astype(np.uint8), thr


def top_n(snr_map, threshold: float, n: int):
    """R26: pixel indices of the n highest per-pixel peaks with snr > threshold, best first."""
    s = np.asarray(snr_map, dtype=np.float32).ravel()
    cand = [(float(s[p]), p) for p in range(s.size) if s[p] > np.float32(threshold)]   # NaN and -inf fail the test
    cand.sort(key=lambda sp: (-sp[0], sp[1]))
    return [p for _, p in cand[:n]]


def cluster(snr_map, nx: int, ny: int, threshold: float, n: int, psf, mask):
    """L94 step by step.  Returns dict(pixels=[...], wsnr=[...], members=[...], best=index or -1)."""
    psf = np.asarray(psf, dtype=np.float32)
    mask = np.asarray(mask)
    mh, mw = psf.shape
    cy, cx = mh // 2, mw // 2                                       # R27
    s = np.asarray(snr_map, dtype=np.float32).ravel()
    assert s.size == nx * ny
    pix = top_n(s, threshold, n)
    wsnr, members = [], []
    for pi in pix:                                                  # "centered on each candidate in turn"
        xi, yi = pi % nx, pi // nx
        num = 0.0
        den = 0.0
        cnt = 0
        for pj in pix:                                              # rank order
            xj, yj = pj % nx, pj // nx
            mx, my = cx + (xj - xi), cy + (yj - yi)
            inside = 0 <= mx < mw and 0 <= my < mh
            if pj == pi:
                w = float(psf[cy, cx])                              # the central lobe
            elif inside and mask[my, mx]:
                w = float(psf[my, mx])                              # a possible sidelobe
            else:
                continue
            num = num + w * float(s[pj])
            den = den + w
            cnt += 1
        wsnr.append(num / den)
        members.append(cnt)
    best = -1
    for i in range(len(pix)):                                       # "the maximum S/N is identified"
        if best < 0 or wsnr[i] > wsnr[best]:
            best = i
    return dict(pixels=pix, wsnr=wsnr, members=members, best=best)
