"""CPU pins of oracle/imaging.py: what the paper and the mathematics fix, chosen so that a
plausible mistake (fftshift for ifftshift, u/v transposed, a wrong sign, a dropped Hermitian half, mean for sum of the
polarisations, natural for uniform weights) fails one of them."""
import numpy as np
import pytest

from oracle import imaging as I
from paper_2510_18136_b200 import workloads as W


def test_paper_buffer_arithmetic():
    # PAPER.md:L48 N_base = 4656 from Fig. 1's 97 antennas; L55 "14.9 MB buffer"; L67 "buffered (6.125 MB)"
    assert W.IMG_NANT * (W.IMG_NANT - 1) // 2 == 4656 == W.imaging_array(0).shape[0]
    assert 4656 * 8 * 25 * 2 * 8 == 14_899_200          # baselines x channels x samples x pols x complex64
    assert 175 * 175 * 25 * 8 == 6_125_000               # image block of one node, float64
    assert W.IMG_N == 175 and abs(W.IMG_PIXEL_RAD * 206264.80624709636 - 10.3) < 1e-12


def test_uv_cell_hand_value():
    # u = 100 m at 1.4 GHz = 466.99 wavelengths; 175 pixels of 10.3 arcsec = 8.7388e-3 rad  =>  4.081 cells -> 4; -100 m -> -4
    cells = I.uv_cells(np.asarray([[100.0, -100.0], [12.0, 0.0]]), 1.4, 175, W.IMG_PIXEL_RAD)
    assert cells.tolist() == [[4, -4], [0, 0]]
    x = 100.0 * 1.4e9 / 299792458.0 * 175 * W.IMG_PIXEL_RAD
    assert abs(x - 4.081) < 1e-3
    assert I.uv_cells(np.asarray([[61.27, 0.0]]), 1.4, 175, W.IMG_PIXEL_RAD)[0, 0] == 3   # 2.5004 cells rounds up (floor(x + 0.5))


def test_baseline_selection_is_strict_and_in_metres():
    uv = np.asarray([[20.0, 0.0], [0.0, 20.0001], [485.0, 0.0], [300.0, 380.0], [3.0, 4.0], [-484.9, 0.0], [12.0, 16.0]])
    assert I.select_baselines(uv).tolist() == [1, 3, 5]     # b = 20 and 485 are out (L55: b > b_min, b < b_max); |(300,380)| = 484.05


def test_briggs_hand_worked_example():
    # three visibilities: two in cell A, one in cell B.  With the Hermitian copies sum_k W_k^2 = 2*4 + 2*1 = 10, sum_i w_i = 6,
    # f^2 = (5e2)^2 / (10/6) = 150000  =>  w'_A = 1/300001, w'_B = 1/150001
    cells = np.asarray([[2, 1], [2, 1], [-3, 0]])
    w = I.briggs_weights(cells, 9, -2.0)
    assert np.allclose(w, [1 / 300001.0, 1 / 300001.0, 1 / 150001.0], rtol=1e-14)
    # R = -2 is "approximately uniform" (w' W = const to 1e-5), a large positive R is natural weighting, outside the grid -> 0
    assert abs(w[0] * 2 / (w[2] * 1) - 1.0) < 1e-5
    assert np.allclose(I.briggs_weights(cells, 9, 8.0), 1.0, rtol=1e-6)
    assert I.briggs_weights(np.asarray([[5, 0], [1, 1]]), 9, -2.0)[0] == 0.0


@pytest.mark.parametrize("n", [7, 8, 9])
def test_route_equals_the_dft_written_out(n):
    """fn. 10's route (ifftshift -> np.fft.ifft2 -> ifftshift) against the inverse DFT as a triple loop, asymmetric cells
    (u != v, no symmetry to hide a transposition), on both parities of n: frequency 0 at grid index n // 2, phase centre at
    pixel n - n // 2 (one past the centre pixel for odd n: what ifftshift, as opposed to fftshift, does)."""
    rng = np.random.default_rng(n)
    nb = 9
    cells = np.stack([rng.integers(-(n // 2) + 1, n // 2, nb), rng.integers(-(n // 2) + 1, n // 2, nb)], axis=1)
    cells[0] = (2, -1)
    w = rng.uniform(0.5, 2.0, nb)
    vis = rng.standard_normal((nb, 2)) + 1j * rng.standard_normal((nb, 2))
    a = I.image_channel(I.grid_channel(vis, cells, w, n))
    b = I.direct_image(vis, cells, w, n)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max()
    assert np.abs(a.imag).max() <= 1e-13 * np.abs(a.real).max()          # Hermitian grid -> real image
    assert I.phase_centre_pixel(7) == 4 and I.phase_centre_pixel(8) == 4 and I.phase_centre_pixel(175) == 88
    # a single visibility of value 1 in one polarisation: 2 cos(2 pi (fu dx + fv dy)/n) / n^2 -- a closed form with its sign
    one = np.zeros((1, 2), complex)
    one[0, 0] = 1.0
    img = I.image_channel(I.grid_channel(one, np.asarray([[2, -1]]), np.ones(1), n)).real
    x0 = I.phase_centre_pixel(n)
    for (dy, dx) in ((0, 0), (1, 0), (0, 1), (2, -1)):
        want = 2.0 * np.cos(2 * np.pi * (2 * dx - 1 * dy) / n) / (n * n)
        assert abs(img[(x0 + dy) % n, (x0 + dx) % n] - want) < 1e-15


def test_point_source_position_flux_and_orientation():
    """A unit source at the phase centre has value nchan at pixel (88, 88) (every channel normalised to 1, L67 sums them); a
    source at (l, m) = (+10, -20) pixels shows up at x = 88 + 10, y = 88 - 20: x runs with u / l, y with v / m."""
    uv = W.imaging_array(0)
    f = W.imaging_freqs()
    x0 = I.phase_centre_pixel(W.IMG_N)
    img = I.image(W.imaging_visibilities(uv, f, 1, [(0.0, 0.0, 1.0)]), uv, f)[0]
    assert abs(img[x0, x0] - len(f)) < 1e-9 and np.unravel_index(np.argmax(img), img.shape) == (x0, x0)
    src = [(10 * W.IMG_PIXEL_RAD, -20 * W.IMG_PIXEL_RAD, 3.0)]
    img = I.image(W.imaging_visibilities(uv, f, 1, src), uv, f)[0]
    assert np.unravel_index(np.argmax(img), img.shape) == (x0 - 20, x0 + 10)
    assert 0.9 * 3.0 * len(f) < img.max() <= 3.0 * len(f) + 1e-9          # nearest-cell gridding loses a few per cent off-centre


def test_polarisations_are_summed_channels_are_summed_and_the_map_is_linear():
    uv = W.imaging_array(1)
    f = W.imaging_freqs(3)
    rng = np.random.default_rng(5)
    v = (rng.standard_normal((2, 8, 4656, 2)) + 1j * rng.standard_normal((2, 8, 4656, 2))).astype(np.complex64)
    full = I.image(v, uv, f)
    # L55 "The two visibility polarizations are summed": (a, b) == (a + b, 0) == (b, a)
    v2 = v.astype(np.complex128); v2[..., 0] = v2[..., 0] + v2[..., 1]; v2[..., 1] = 0
    assert np.allclose(I.image(v2, uv, f), full, rtol=0, atol=1e-11)
    assert np.allclose(I.image(v[..., ::-1], uv, f), full, rtol=0, atol=1e-12)
    # L67 "Each of the 8 channels are imaged individually, then summed"
    parts = sum(I.image(v[:, c:c + 1], uv, f[c:c + 1]) for c in range(8))
    assert np.allclose(parts, full, rtol=0, atol=1e-10)
    assert np.allclose(I.image(2.5 * v.astype(np.complex128), uv, f), 2.5 * full, rtol=1e-12, atol=1e-10)
    # baselines outside (20 m, 485 m) do not matter (L55): zeroing them changes nothing
    sel = I.select_baselines(uv)
    cut = np.ones(4656, bool); cut[sel] = False
    v3 = v.copy(); v3[:, :, cut, :] = 0
    assert np.array_equal(I.image(v3, uv, f), full) and cut.sum() > 1000
