"""-m gpu: nsfrb_imager_* (NEXT 4: visibilities -> images, PAPER.md:L55/L61/L67) against oracle/imaging.py, element by element.

Tolerance: the kernel accumulates ~25 000 float32 terms per pixel against the oracle's float64 FFT route:
|I_gpu - I_orc| <= 5e-5 * max|I_orc| per image (measured worst case ~3e-6); the integer part -- baseline selection and UV
cells -- is bit-exact, the Briggs weights agree to 1e-14 relative."""
import numpy as np
import pytest
import torch

from oracle import imaging as OI
from paper_2510_18136_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _nsfrb():
    from paper_2510_18136_b200 import nsfrb
    return nsfrb


def _check_images(got, want, label):
    assert got.shape == want.shape
    for t in range(want.shape[0]):
        scale = np.abs(want[t]).max()
        err = np.abs(got[t] - want[t]).max()
        assert err <= 5e-5 * scale + 1e-12, f"{label} t={t}: |d| = {err:.3e} vs max|I| = {scale:.3e}"
    return float(np.max(np.abs(got - want)) / max(np.abs(want).max(), 1e-30))


def test_tables_are_exact():
    nsfrb = _nsfrb()
    uv = W.imaging_array(0)
    f = W.imaging_freqs()
    with nsfrb.Imager(W.IMG_N, W.IMG_PIXEL_RAD, uv, f) as im:
        cells, w = im.table()
    sel = OI.select_baselines(uv)
    gridded = np.zeros(len(uv), bool); gridded[sel] = True
    for ch in range(len(f)):
        oc = OI.uv_cells(uv[sel], float(f[ch]), W.IMG_N, W.IMG_PIXEL_RAD)
        ow = OI.briggs_weights(oc, W.IMG_N, -2.0)
        assert np.array_equal((w[ch] > 0), gridded)                      # same baselines gridded (b_min, b_max strict)
        assert np.array_equal(cells[ch][sel], oc)                        # UV cells bit-exact
        assert np.allclose(w[ch][sel], ow, rtol=1e-14, atol=0)


def test_paper_shape_block_matches_oracle():
    """The paper's block: 25 samples x 8 channels x 4656 baselines x 2 pols (14.9 MB) -> 25 images of 175 x 175: two steady
    sources, one 3-sample transient, noise."""
    nsfrb = _nsfrb()
    uv = W.imaging_array(0)
    f = W.imaging_freqs()
    px = W.IMG_PIXEL_RAD
    src = [(12 * px, 30 * px, 2.0), (-40.3 * px, -7.6 * px, 1.0), (25 * px, -60 * px, 5.0, 10, 13)]
    vis = W.imaging_visibilities(uv, f, 25, src, noise=0.5, seed=1)
    assert vis.nbytes == 14_899_200
    with nsfrb.Imager(W.IMG_N, px, uv, f) as im:
        got = im.image(torch.from_numpy(vis).cuda()).cpu().numpy().reshape(25, W.IMG_N, W.IMG_N)
    want = OI.image(vis, uv, f)
    worst = _check_images(got, want, "paper block")
    print(f"[parity] imaging, paper block: worst |d| / max|I| = {worst:.2e}")
    x0 = OI.phase_centre_pixel(W.IMG_N)
    for t, (ey, ex) in ((11, (x0 - 60, x0 + 25)), (0, (x0 + 30, x0 + 12))):            # the transient while it is on; the steady source
        gy, gx = np.unravel_index(np.argmax(got[t]), got[t].shape)
        assert (gy, gx) == np.unravel_index(np.argmax(want[t]), want[t].shape)
        assert abs(gy - ey) <= 1 and abs(gx - ex) <= 1


@pytest.mark.parametrize("n,nchan,nt,robust,bmin,bmax", [
    (64, 3, 2, -2.0, 20.0, 485.0),      # even n: phase centre at n/2
    (33, 1, 1, 0.5, 0.0, 300.0),        # one partial 32-column tile + one column; intermediate robustness
    (175, 8, 3, 2.0, 50.0, 5000.0),     # outriggers included: cells beyond the grid are dropped
    (257, 2, 1, -2.0, 20.0, 485.0),     # nine column tiles, 129 rows
])
def test_other_shapes_match_oracle(n, nchan, nt, robust, bmin, bmax):
    nsfrb = _nsfrb()
    uv = W.imaging_array(2)
    f = W.imaging_freqs(5, nchan)
    rng = np.random.default_rng(n)
    vis = (rng.standard_normal((nt, nchan, len(uv), 2)) + 1j * rng.standard_normal((nt, nchan, len(uv), 2))).astype(np.complex64)
    px = W.IMG_PIXEL_RAD * 175 / n
    with nsfrb.Imager(n, px, uv, f, bmin, bmax, robust) as im:
        got = im.image(torch.from_numpy(vis).cuda()).cpu().numpy().reshape(nt, n, n)
    want = OI.image(vis, uv, f, n=n, pixel_rad=px, bmin_m=bmin, bmax_m=bmax, robust=robust)
    _check_images(got, want, f"n={n}")


def test_images_feed_the_search_as_chunks():
    """End of the step: sub-bands imaged straight into the planes of [chan][25][175*175] chunks that nsfrb_stream_push accepts.
    Two noise-only chunks, then one with a 4-sample transient in every sub-band: the search finds it at its pixel.  (One
    25-sample chunk alone cannot exceed S/N = sqrt(T - w) = 4.6: the pulse is its own noise estimate.)"""
    nsfrb = _nsfrb()
    uv = W.imaging_array(0)
    px = W.IMG_PIXEL_RAD
    nsub, nt, n = 4, 25, W.IMG_N
    x0 = OI.phase_centre_pixel(n)
    freqs = np.asarray([W.imaging_freqs(4 * sb).mean() for sb in range(nsub)])
    imagers = [nsfrb.Imager(n, px, uv, W.imaging_freqs(4 * sb)) for sb in range(nsub)]
    try:
        with nsfrb.Plan(n, n, nsub, 128, freqs, W.TSAMP_S, [0.0, 100.0], [1, 2, 4, 8], 6.0) as plan:
            for k in range(3):
                chunk = torch.empty((nsub, nt, n * n), device="cuda")
                for sb in range(nsub):
                    src = [(-20 * px, 15 * px, 0.05, 8, 12)] if k == 2 else []
                    vis = W.imaging_visibilities(uv, W.imaging_freqs(4 * sb), nt, src, noise=1.0, seed=10 * k + sb)
                    imagers[sb].image(torch.from_numpy(vis).cuda(), out=chunk[sb])
                res = plan.stream_push(chunk)
            torch.cuda.synchronize()
            snr = res.snr_map.cpu().numpy()
            arg = res.argmax.cpu().numpy()
    finally:
        for im in imagers:
            im.close()
    p = int(np.argmax(snr))
    py, pxx = divmod(p, n)
    # (the synthesized beam is 3 pixels wide, L55: within 2 pixels = inside the main lobe)
    assert abs(py - (x0 + 15)) <= 2 and abs(pxx - (x0 - 20)) <= 2 and snr[p] > 6.0, (py, pxx, float(snr[p]))
    assert arg[1, p] == 2 and abs(int(arg[2, p]) - 58) <= 1        # width 4, start sample 50 + 8
