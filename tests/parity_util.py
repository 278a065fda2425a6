"""P-rule of SURVEY.md sec. 8(c): element-by-element comparison of the CUDA path with the oracle.

tol(s) = 1e-4 + 1e-4*|s|  (BASELINE.json north_star: "within 1e-4 relative / 1e-4 absolute on
float32 S/N values"; "bit-exactly on delays, arg-max indices and candidate sets wherever the
winning S/N margin exceeds the tolerance").
 (i)   |snr_gpu - snr_orc| <= tol
 (ii)  argmax_gpu == argmax_orc, or the oracle adjudicates: S_orc(argmax_gpu) >= snr_orc - 2*tol and
       the reported dm index is the lowest one among trials with an identical delay vector
 (iii) candidate sets equal after removing pixels with |snr_orc - threshold| <= tol
"""
from __future__ import annotations

import numpy as np

from oracle import oracle


def tol(s):
    return 1e-4 + 1e-4 * np.abs(s)


def check(cube_sel: np.ndarray, delays: np.ndarray, widths, gpu_snr: np.ndarray, gpu_arg: np.ndarray,
          threshold: float, *, raw_end_min=0, t_offset=0, nthreads=8, max_adjudicated_frac=0.10, label=""):
    """cube_sel: [nchan][nt][n] float32 (the pixels compared); gpu_snr [n]; gpu_arg [n][3].
    Returns a dict of counts; raises AssertionError with a readable message on any violation."""
    cube_sel = np.ascontiguousarray(cube_sel, dtype=np.float32)
    n = cube_sel.shape[2]
    assert gpu_snr.shape == (n,) and gpu_arg.shape == (n, 3), (gpu_snr.shape, gpu_arg.shape)
    r = oracle.search(cube_sel, delays, widths, raw_end_min=raw_end_min, t_offset=t_offset, nthreads=nthreads)
    # lowest index among identical delay vectors
    canon = np.arange(delays.shape[0])
    for k in range(delays.shape[0]):
        for k2 in range(k):
            if np.array_equal(delays[k], delays[k2]):
                canon[k] = k2
                break
    exact = adjud = undefined = 0
    worst = 0.0
    for i in range(n):
        so, sg = r.snr[i], float(gpu_snr[i])
        if np.isneginf(so):
            assert np.isneginf(sg) and tuple(gpu_arg[i]) == (-1, -1, -1), f"{label} px{i}: oracle has no cell, gpu {sg} {gpu_arg[i]}"
            undefined += 1
            continue
        t = tol(so)
        assert abs(sg - so) <= t, f"{label} px{i}: snr gpu {sg!r} vs oracle {so!r} (|d|={abs(sg-so):.3e} > tol {t:.3e}); arg gpu {gpu_arg[i]} orc {r.argmax[i]}"
        worst = max(worst, abs(sg - so) / t)
        if tuple(int(v) for v in gpu_arg[i]) == tuple(int(v) for v in r.argmax[i]):
            exact += 1
            continue
        k, j, tt = (int(v) for v in gpu_arg[i])
        assert 0 <= k < delays.shape[0] and 0 <= j < len(widths), f"{label} px{i}: bad argmax {gpu_arg[i]}"
        assert canon[k] == k, f"{label} px{i}: dm_idx {k} is a duplicate of {canon[k]} (lowest index must be reported)"
        s_at = oracle.snr_at(cube_sel, delays, widths, i, k, j, tt, raw_end_min=raw_end_min, t_offset=t_offset)
        assert not np.isnan(s_at), f"{label} px{i}: gpu argmax {gpu_arg[i]} is not a defined cell (oracle {r.argmax[i]})"
        assert s_at >= so - 2 * t, (f"{label} px{i}: gpu argmax {gpu_arg[i]} has oracle S/N {s_at!r}, "
                                    f"oracle max {so!r} at {r.argmax[i]} (margin {so - s_at:.3e} > 2 tol)")
        adjud += 1
    defined = max(n - undefined, 1)
    assert adjud / defined <= max_adjudicated_frac, f"{label}: {adjud}/{defined} arg-max needed adjudication"
    return {"n": n, "exact": exact, "adjudicated": adjud, "undefined": undefined, "worst_tol_frac": worst,
            "oracle": r}


def check_candidates(oracle_res, pixel_ids, gpu_cands, gpu_n_found, threshold, capacity, all_pixels_checked=True,
                     gpu_snr_all=None):
    """(iii): candidate sets equal after removing pixels within tol of the threshold.
    oracle_res covers `pixel_ids` (global pixel numbers); gpu_cands is the structured array."""
    so = oracle_res.snr
    near = np.abs(so - threshold) <= tol(so)
    expect = {int(pixel_ids[i]) for i in np.nonzero((so > threshold) & ~near)[0]}
    fuzzy = {int(pixel_ids[i]) for i in np.nonzero(near)[0]}
    got = {int(c["pixel"]) for c in gpu_cands}
    inside = set(int(p) for p in pixel_ids)
    got_in = got & inside
    if gpu_n_found <= capacity:
        assert expect <= got_in, f"missing candidates: {sorted(expect - got_in)[:10]}"
    assert got_in <= (expect | fuzzy), f"spurious candidates: {sorted(got_in - expect - fuzzy)[:10]}"
    if all_pixels_checked and gpu_n_found <= capacity:
        assert len(got) == len(gpu_cands), "duplicate pixels in the candidate list"
        assert len(expect) <= gpu_n_found <= len(expect) + len(fuzzy)
    # every stored record repeats the maps
    return {"expected": len(expect), "near_threshold": len(fuzzy), "found": int(gpu_n_found)}
