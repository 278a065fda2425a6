"""-m "not gpu": pins of oracle/cluster.py (top-N selection + PSF-mask sidelobe clustering) against
things other than itself: numpy's percentile routine, closed forms, hand-worked examples, brute force, invariants."""
import itertools

import numpy as np
import pytest

from oracle import cluster as C
from paper_2510_18136_b200 import workloads as W


# ---- percentile / mask ------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n,q", [(1, 90.0), (2, 90.0), (10, 90.0), (11, 90.0), (1000, 90.0), (77, 37.5), (64, 0.0),
                                 (64, 100.0)])
def test_percentile_matches_numpy_routine(n, q):
    v = np.random.default_rng(n).normal(size=n).astype(np.float32)
    assert C.percentile_value(v, q) == pytest.approx(float(np.percentile(v.astype(np.float64), q)), rel=0, abs=1e-15)


def test_percentile_closed_forms():
    # 0..10: rank 0.9*10 = 9 exactly -> 9; 0..9: rank 8.1 -> 8.1
    assert C.percentile_value(np.arange(11.0), 90.0) == 9.0
    assert C.percentile_value(np.arange(10.0)[::-1], 90.0) == pytest.approx(8.1, abs=1e-12)
    assert C.percentile_value(np.full(7, 3.5), 90.0) == 3.5


def test_mask_is_strict_and_keeps_a_tenth():
    psf = np.arange(100, dtype=np.float32).reshape(10, 10)       # percentile 90 -> rank 89.1 -> 89.1
    mask, thr = C.psf_mask(psf, 90.0)
    assert thr == pytest.approx(89.1, abs=1e-12)
    assert mask.sum() == 10 and mask.ravel()[90:].all() and not mask.ravel()[:90].any()
    psf = np.arange(11, dtype=np.float32).reshape(1, 11)         # value 9 sits exactly on the percentile: excluded
    mask, thr = C.psf_mask(psf, 90.0)
    assert thr == 9.0 and mask.ravel().tolist() == [0] * 10 + [1]
    big = W.synthetic_psf(101, 3)
    mask, _ = C.psf_mask(big, 90.0)
    assert abs(mask.mean() - 0.1) < 1e-3 and mask[50, 50] == 1


# ---- top-N --------------------------------------------------------------------------------------------------------

def test_top_n_matches_stable_sort_and_breaks_ties_by_pixel():
    rng = np.random.default_rng(5)
    s = rng.integers(0, 12, size=500).astype(np.float32)         # many exact ties
    s[17] = np.nan
    s[18] = -np.inf
    thr = 6.0
    order = np.argsort(-np.where(np.isnan(s), -np.inf, s), kind="stable")
    want = [int(p) for p in order if s[p] > thr][:10]
    assert C.top_n(s, thr, 10) == want
    assert C.top_n(s, 100.0, 10) == []
    assert C.top_n(s, thr, 3) == want[:3]
    assert C.top_n(np.asarray([7, 9, 9, 6, 6.0001], np.float32), 6.0, 10) == [1, 2, 0, 4]   # strict threshold


# ---- clustering: hand-worked examples and invariants -------------------------------------------------------------

def _cross_psf():
    """5x5 PSF: centre 1, the four neighbours at distance 2 along x are 0.5, everything else 0."""
    psf = np.zeros((5, 5), np.float32)
    psf[2, 2] = 1.0
    psf[2, 0] = psf[2, 4] = 0.5
    mask = (psf > 0.25).astype(np.uint8)
    return psf, mask


def test_hand_worked_example():
    psf, mask = _cross_psf()
    nx, ny = 8, 4
    s = np.zeros((ny, nx), np.float32)
    s[1, 3] = 10.0      # A
    s[1, 5] = 8.0       # B: 2 to the right of A -> inside A's mask (weight .5), and A inside B's
    s[3, 3] = 9.0       # C: 2 below A -> psf 0 there: not a member
    r = C.cluster(s, nx, ny, 6.0, 10, psf, mask)
    assert r["pixels"] == [1 * nx + 3, 3 * nx + 3, 1 * nx + 5]          # A (10), C (9), B (8)
    # A: (1*10 + .5*8)/1.5 = 9.3333; C: 9; B: (1*8 + .5*10)/1.5 = 8.6667
    assert r["wsnr"] == pytest.approx([14.0 / 1.5, 9.0, 13.0 / 1.5], abs=1e-12)
    assert r["members"] == [2, 1, 2]
    assert r["best"] == 0


def test_sidelobe_group_can_beat_a_brighter_loner():
    psf, mask = _cross_psf()
    nx, ny = 12, 3
    s = np.zeros((ny, nx), np.float32)
    s[0, 0] = 10.0                      # alone
    s[2, 6] = 9.9
    s[2, 8] = 10.5                      # its neighbour is brighter: centre 9.9 -> (9.9 + .5*10.5)/1.5 = 10.1
    r = C.cluster(s, nx, ny, 6.0, 10, psf, mask)
    assert r["pixels"] == [2 * nx + 8, 0, 2 * nx + 6]
    assert r["wsnr"] == pytest.approx([(10.5 + 0.5 * 9.9) / 1.5, 10.0, (9.9 + 0.5 * 10.5) / 1.5], abs=1e-6)
    assert r["best"] == 0               # 10.3 > 10.1 > 10


def test_degenerate_cases():
    psf, mask = _cross_psf()
    s = np.full((4, 4), 3.0, np.float32)
    r = C.cluster(s, 4, 4, 6.0, 10, psf, mask)
    assert r == dict(pixels=[], wsnr=[], members=[], best=-1)
    s[2, 1] = 7.0
    r = C.cluster(s, 4, 4, 6.0, 10, psf, mask)
    assert r["pixels"] == [9] and r["wsnr"] == [7.0] and r["members"] == [1] and r["best"] == 0
    # delta PSF: nobody has sidelobes, the result is the top-1
    d = np.zeros((3, 3), np.float32)
    d[1, 1] = 1.0
    s = np.random.default_rng(0).uniform(6.5, 20, size=(6, 6)).astype(np.float32)
    r = C.cluster(s, 6, 6, 6.0, 10, d, (d > 0).astype(np.uint8))
    assert r["best"] == 0 and r["members"] == [1] * 10
    assert r["wsnr"] == [float(s.ravel()[p]) for p in r["pixels"]]
    # all candidates equal: every weighted mean is that value, the first (smallest pixel) wins
    s = np.zeros((3, 9), np.float32)
    s[1, 2] = s[1, 4] = s[1, 6] = 8.0
    r = C.cluster(s, 9, 3, 6.0, 10, psf, mask)
    assert r["wsnr"] == pytest.approx([8.0] * 3, abs=1e-12) and r["members"] == [2, 3, 2] and r["best"] == 0


def test_translation_invariance_and_membership_symmetry():
    psf = W.synthetic_psf(41, 1)
    mask, _ = C.psf_mask(psf, 90.0)
    assert (mask == mask[::-1, ::-1]).all()          # a real beam is point-symmetric -> membership is mutual
    nx = ny = 96
    rng = np.random.default_rng(2)
    pts = [(30 + int(dx), 30 + int(dy)) for dx, dy in rng.integers(-12, 13, size=(9, 2))]
    pts = list(dict.fromkeys(pts))
    vals = rng.uniform(7, 20, size=len(pts)).astype(np.float32)

    def run(ox, oy):
        s = np.zeros((ny, nx), np.float32)
        for (x, y), v in zip(pts, vals):
            s[y + oy, x + ox] = v
        return C.cluster(s, nx, ny, 6.0, 10, psf, mask)

    a, b = run(0, 0), run(17, 31)
    assert a["wsnr"] == pytest.approx(b["wsnr"], abs=1e-12) and a["members"] == b["members"] and a["best"] == b["best"]
    # brute force of the membership count from the definition
    pix = a["pixels"]
    for i, pi in enumerate(pix):
        cnt = 0
        for pj in pix:
            dx, dy = pj % nx - pi % nx, pj // nx - pi // nx
            if pj == pi or (abs(dx) <= 20 and abs(dy) <= 20 and mask[20 + dy, 20 + dx]):
                cnt += 1
        assert cnt == a["members"][i]


def test_weighted_mean_is_bounded_by_member_snrs_and_recovers_the_source():
    psf = W.synthetic_psf(301, 0)
    mask, _ = C.psf_mask(psf, 90.0)
    for seed in range(4):
        m, (x0, y0) = W.synthetic_snr_map(301, 301, psf, seed)
        r = C.cluster(m, 301, 301, 6.0, 10, psf, mask)
        s = m.ravel()
        assert len(r["pixels"]) == 10 and r["pixels"][0] == y0 * 301 + x0
        assert all(s[a] >= s[b] for a, b in itertools.pairwise(r["pixels"]))
        lo, hi = float(s[r["pixels"][-1]]), float(s[r["pixels"][0]])
        assert all(lo - 1e-9 <= w <= hi + 1e-9 for w in r["wsnr"])
        assert r["pixels"][r["best"]] == y0 * 301 + x0     # the injected source is the most likely candidate
