"""-m gpu: nsfrb_psf_mask / nsfrb_cluster through the C ABI vs oracle/cluster.py.  Index work is
compared bit for bit; the float64 weighted means are computed in the same order with single roundings on both
sides, so they are compared exactly as well."""
import numpy as np
import pytest
import torch

from oracle import cluster as OC
from oracle import oracle
from paper_2510_18136_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _nsfrb():
    from paper_2510_18136_b200 import nsfrb
    return nsfrb


def _plan(nsfrb, nx, ny, thr):
    return nsfrb.Plan(nx, ny, 2, 64, [1.3, 1.5], W.TSAMP_S, [0.0], [1], thr)


@pytest.mark.parametrize("shape,q,seed", [((301, 301), 90.0, 0), ((33, 65), 90.0, 1), ((1, 1), 90.0, 2),
                                          ((7, 3), 0.0, 3), ((7, 3), 100.0, 4), ((101, 101), 37.5, 5),
                                          ((601, 601), 90.0, 6)])
def test_psf_mask_matches_oracle(shape, q, seed):
    nsfrb = _nsfrb()
    if shape[0] == shape[1] and shape[0] > 7:
        psf = W.synthetic_psf(shape[0], seed)
    else:
        psf = np.random.default_rng(seed).normal(size=shape).astype(np.float32)
    mask_o, thr_o = OC.psf_mask(psf, q)
    mask, value = nsfrb.psf_mask(torch.from_numpy(psf).cuda(), q)
    assert float(value.cpu()[0]) == thr_o
    assert np.array_equal(mask.cpu().numpy(), mask_o)


def test_psf_mask_with_repeated_values_and_signed_zeros():
    nsfrb = _nsfrb()
    rng = np.random.default_rng(9)
    psf = rng.integers(-3, 4, size=(40, 50)).astype(np.float32)     # heavy ties around every order statistic
    psf[psf == 0] *= rng.choice([-1.0, 1.0], size=int((psf == 0).sum())).astype(np.float32)   # +0 and -0
    for q in (10.0, 50.0, 90.0, 99.9):
        mask_o, thr_o = OC.psf_mask(psf, q)
        mask, value = nsfrb.psf_mask(torch.from_numpy(psf).cuda(), q)
        assert float(value.cpu()[0]) == thr_o and np.array_equal(mask.cpu().numpy(), mask_o)


def _compare(nsfrb, m, nx, ny, thr, topn, psf, mask_o, arg=None):
    want = OC.cluster(m, nx, ny, thr, topn, psf, mask_o)
    if arg is None:
        arg = np.random.default_rng(1).integers(0, 1000, size=(3, nx * ny)).astype(np.int32)
    with _plan(nsfrb, nx, ny, thr) as plan:
        for _ in range(2):       # twice: the ticket counter must be back at zero after a call
            res = plan.cluster(torch.from_numpy(m.ravel().copy()).cuda(), torch.from_numpy(arg).cuda(),
                               torch.from_numpy(psf).cuda(), torch.from_numpy(mask_o).cuda(), topn)
            assert plan.last_launches() == 1
            got = res.to_host()
            assert got["pixels"] == want["pixels"]
            assert got["members"] == want["members"]
            assert got["wsnr"] == want["wsnr"]              # same operations, same order, float64
            assert got["best"] == want["best"]
            for c in got["cands"]:
                p = int(c["pixel"])
                assert c["snr"] == m.ravel()[p] and (c["dm_idx"], c["width_idx"], c["t"]) == tuple(arg[:, p])
            raw = res.top.cpu().numpy().view(nsfrb.CAND_DTYPE)
            assert all(tuple(r) == (-1, -1, -1, -1, 0.0) for r in raw[len(got["pixels"]):])
            assert res.members.cpu().numpy()[len(got["pixels"]):].tolist() == [0] * (topn - len(got["pixels"]))
    return want


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_cluster_matches_oracle_on_source_with_sidelobes(seed):
    nsfrb = _nsfrb()
    psf = W.synthetic_psf(301, seed)
    mask_o, _ = OC.psf_mask(psf, 90.0)
    m, (x0, y0) = W.synthetic_snr_map(301, 301, psf, seed)
    want = _compare(nsfrb, m, 301, 301, 6.0, 10, psf, mask_o)
    assert want["pixels"][0] == y0 * 301 + x0 and max(want["members"]) > 1     # the scenario has sidelobe groups


def test_cluster_ties_few_candidates_and_edges():
    nsfrb = _nsfrb()
    psf = W.synthetic_psf(41, 7)
    mask_o, _ = OC.psf_mask(psf, 90.0)
    nx, ny = 130, 77                                   # ragged: 10 010 pixels -> 5 CTAs, the last one short
    rng = np.random.default_rng(3)
    m = rng.integers(0, 12, size=(ny, nx)).astype(np.float32)       # thousands of exact ties
    m[0, 0] = m[ny - 1, nx - 1] = m[0, nx - 1] = 11.0               # corners: the mask hangs over the edge
    m[5, 5] = np.nan
    m[6, 6] = np.inf
    m[7, 7] = -np.inf
    for topn in (1, 10, 32):
        _compare(nsfrb, m, nx, ny, 6.0, topn, psf, mask_o)
    # fewer candidates than topn, then none
    m2 = np.full((ny, nx), 3.0, np.float32)
    m2[10, 20], m2[10, 22], m2[40, 100] = 9.0, 8.0, 7.5
    w = _compare(nsfrb, m2, nx, ny, 6.0, 10, psf, mask_o)
    assert len(w["pixels"]) == 3
    w = _compare(nsfrb, m2, nx, ny, 20.0, 10, psf, mask_o)
    assert w["pixels"] == [] and w["best"] == -1
    # one pixel image, mask bigger than the image
    _compare(nsfrb, np.full((1, 1), 9.0, np.float32), 1, 1, 6.0, 10, psf, mask_o)


def test_cluster_at_full_size():
    """The bench configuration's map sizes (301 x 301 and 1024 x 1024 pixels): 45 / 148 CTAs."""
    nsfrb = _nsfrb()
    psf = W.synthetic_psf(301, 11)
    mask_o, _ = OC.psf_mask(psf, 90.0)
    m, _ = W.synthetic_snr_map(1024, 1024, psf, 11)
    _compare(nsfrb, m, 1024, 1024, 8.5, 10, psf, mask_o)


def test_cluster_after_stream_push():
    """End to end on the real-time path: push chunks (injected pulses + noise, a threshold low enough that noise
    peaks are candidates too), cluster the device maps of the last push; the oracle clusters ITS OWN maps.  The
    two S/N maps agree to the search tolerance only, so ranks may swap between near-equal candidates: the sorted
    S/N lists must agree within tol, pixels wherever the oracle's neighbours in the list are further than 2 tol
    apart, and -- when the whole list agrees -- members exactly and the weighted means to 1e-3."""
    from dataclasses import replace
    nsfrb = _nsfrb()
    wl = replace(W.config("c1"), threshold=2.5)
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    psf = W.synthetic_psf(41, 2)
    mask_o, _ = OC.psf_mask(psf, 90.0)
    n_push = 6
    src = W.ChunkSource(wl, d, n_push, "cuda")
    so = oracle.StreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list)
    with nsfrb.Plan.for_workload(wl) as plan:
        out = plan.alloc_outputs()
        dpsf = torch.from_numpy(psf).cuda()
        dmask, _ = nsfrb.psf_mask(dpsf, 90.0)
        for i in range(n_push):
            chunk = src.next()
            plan.stream_push(chunk, out)
            res = plan.cluster(out.snr_map, out.argmax, dpsf, dmask, 10)
            ores = so.push(chunk.cpu().numpy(), nthreads=8)
        got = res.to_host()
        arg = out.argmax.cpu().numpy()
    want = OC.cluster(ores.snr.astype(np.float32), wl.nx, wl.ny, wl.threshold, 10, psf, mask_o)
    assert len(want["pixels"]) == 10 and len(got["pixels"]) == 10
    ws = np.asarray([ores.snr[p] for p in want["pixels"]])
    gs = np.asarray([float(c["snr"]) for c in got["cands"]])
    tol = 1e-4 + 1e-4 * np.abs(ws)
    assert np.all(np.abs(gs - ws) <= tol)
    for i in range(10):
        lonely = (i == 0 or ws[i - 1] - ws[i] > 2 * tol[i]) and (i == 9 or ws[i] - ws[i + 1] > 2 * tol[i])
        if lonely:
            assert got["pixels"][i] == want["pixels"][i]
    for c in got["cands"]:
        assert (c["dm_idx"], c["width_idx"], c["t"]) == tuple(arg[:, int(c["pixel"])])
    if got["pixels"] == want["pixels"]:
        assert got["members"] == want["members"]
        assert np.allclose(got["wsnr"], want["wsnr"], rtol=0, atol=1e-3)
        top2 = sorted(want["wsnr"])[-2:]
        if top2[1] - top2[0] > 2e-3:
            assert got["best"] == want["best"]


# ---- NEXT 1 (first part): nsfrb_median_subtract vs oracle.median_subtract, exact ------------------------------------

@pytest.mark.parametrize("nchan,nt,npix", [
    (1, 1, 1), (2, 2, 33), (3, 3, 77), (2, 5, 300), (2, 8, 64), (1, 16, 1000), (2, 17, 129), (16, 25, 1024),
    (2, 31, 95), (2, 32, 257), (2, 33, 257), (3, 64, 100), (2, 100, 77), (1, 257, 65), (2, 1000, 90), (2, 2048, 75),
    (1, 2304, 40), (1, 4097, 21), (1, 16384, 7), (1, 30000, 3), (1, 43007, 2), (1, 65535, 1)])
def test_median_subtract_matches_oracle(nchan, nt, npix):
    nsfrb = _nsfrb()
    rng = np.random.default_rng(nt * 131 + npix)
    a = rng.normal(size=(nchan, nt, npix)).astype(np.float32)
    a[0, :, 0] = np.round(3 * a[0, :, 0])                 # exact ties, zeros
    if nt > 3:
        a[0, 1, 0], a[0, 2, 0] = 0.0, -0.0
    a[-1, :, -1] = -np.abs(a[-1, :, -1]) * 1e30            # large negative values: the key order of negative floats
    want, wmed = oracle.median_subtract(a)
    d = torch.from_numpy(a).cuda()
    out, med = nsfrb.median_subtract(d)
    assert np.array_equal(med.cpu().numpy(), wmed)
    assert np.array_equal(out.cpu().numpy(), want)
    assert np.array_equal(d.cpu().numpy(), a)              # the input is untouched
    out2, none = nsfrb.median_subtract(d, out=d, want_median=False)      # in place, no median output
    assert none is None and out2 is d and np.array_equal(d.cpu().numpy(), want)


def test_median_subtract_every_register_length():
    """nt = 1..32 each has its own compile-time comparator network: all of them, with ties."""
    nsfrb = _nsfrb()
    for nt in range(1, 33):
        rng = np.random.default_rng(nt)
        a = rng.normal(size=(2, nt, 300)).astype(np.float32)
        a[1] = np.round(2 * a[1])
        want, wmed = oracle.median_subtract(a)
        out, med = nsfrb.median_subtract(torch.from_numpy(a).cuda())
        assert np.array_equal(med.cpu().numpy(), wmed), nt
        assert np.array_equal(out.cpu().numpy(), want), nt


@pytest.mark.parametrize("nt", [130, 1000, 4096, 5001])
def test_median_subtract_crowded_buckets(nt):
    """Series whose keys crowd one histogram bucket force the extra histogram passes of k_median_stream: a large
    offset (all keys share the top byte, then the second), constants (all 32 bits decided, multiplicity > the candidate
    capacity), two-valued series whose two middle elements sit in different buckets, lanes that need different numbers
    of passes in one warp, and non-finite-free extremes."""
    nsfrb = _nsfrb()
    rng = np.random.default_rng(nt)
    npix = 70
    a = rng.normal(size=(2, nt, npix)).astype(np.float32)
    a[0, :, 0:8] += 1000.0                                   # top two bytes shared
    a[0, :, 8:12] = a[0, :, 8:12] * 1e-3 + 65536.0           # only the low mantissa bits differ
    a[0, :, 12] = 3.25                                        # constant
    a[0, :, 13] = np.where(np.arange(nt) < nt // 2, -1.0, 2.0)     # even nt: the middle pair straddles two buckets
    a[0, :, 14] = np.where(np.arange(nt) % 3 == 0, 1e-30, 1e30)
    a[0, :, 15] = np.round(a[0, :, 15])                       # few distinct values, heavy ties
    a[1, :, 5] = np.float32(1.5e38) * np.sign(a[1, :, 5])     # near +-FLT_MAX / 2
    a[1, : nt // 2, 6] = 0.0
    a[1, nt // 2:, 6] = -0.0
    want, wmed = oracle.median_subtract(a)
    out, med = nsfrb.median_subtract(torch.from_numpy(a).cuda())
    assert np.array_equal(med.cpu().numpy(), wmed)
    assert np.array_equal(out.cpu().numpy(), want)


def test_median_subtract_rejects_bad_arguments():
    nsfrb = _nsfrb()
    L = nsfrb.lib()
    d = torch.zeros((1, 4, 4), device="cuda")
    assert L.nsfrb_median_subtract(d.data_ptr(), 1, 0, 4, d.data_ptr(), None, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_median_subtract(d.data_ptr(), 1, 65536, 4, d.data_ptr(), None, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_median_subtract(None, 1, 4, 4, d.data_ptr(), None, None) == nsfrb.NSFRB_EINVAL


def test_median_then_search_is_the_same_search():
    """R6/R29: the search of the median-subtracted cube equals the search of the cube within the parity tolerance."""
    nsfrb = _nsfrb()
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    W.inject(cube, W.injection_table(wl, d), d, extra_delays=oracle.delays(wl.freqs_GHz, wl.tsamp_s, [500.0])[0])
    sub, _ = nsfrb.median_subtract(cube)
    with nsfrb.Plan.for_workload(wl) as plan:
        s1 = plan.search(sub).snr_map.cpu().numpy()
    r = oracle.search(oracle.median_subtract(cube.cpu().numpy())[0], d, wl.width_list, nthreads=8)
    assert np.all(np.abs(s1 - r.snr) <= 1e-4 + 1e-4 * np.abs(r.snr))
