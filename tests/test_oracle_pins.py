"""Pins for the oracle (-m "not gpu"): what the paper and the mathematics fix, checked with
code that does not share the oracle's formulas (exact rationals, numpy slicing / convolve,
closed forms, pure-Python brute force).  SURVEY.md sec. 8(c) "What pins the oracle"."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle
from paper_2510_18136_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append(line.split())
    return out


# ---------------------------------------------------------------- O1: delay table
def test_delay_hand_value():
    # 4.15 ms * DM * (nu_min^-2 - nu_max^-2); DM 1000, 1.28 vs 1.53 GHz, 0.1342 s
    x = 4.15e-3 * 1000 * (1 / 1.28**2 - 1 / 1.53**2) / 0.1342
    assert abs(x - 5.6642) < 1e-3
    d = oracle.delays([1.28, 1.53], 0.1342, [1000.0])
    assert d.tolist() == [[6, 0]]
    # any channel order, reference is the highest frequency (R2)
    assert oracle.delays([1.53, 1.28], 0.1342, [1000.0]).tolist() == [[0, 6]]


def test_c1_delay_table_golden():
    rows = np.asarray(_rows("c1_delay_table.txt"), dtype=np.int32)
    wl = W.config("c1")
    assert np.array_equal(oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list), rows[:8])
    assert np.array_equal(oracle.delays(wl.freqs_GHz, wl.tsamp_s, [500.0])[0], rows[8])


def test_c2_dmax_golden():
    wl = W.config("c2")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    assert d.max(axis=1).tolist() == [int(v) for v in _rows("c2_dmax.txt")[0]]


def test_delays_against_exact_rationals():
    # independent arithmetic: exact fractions of the decimal inputs, floor(x + 1/2)
    rng = np.random.default_rng(11)
    for _ in range(20):
        nchan = int(rng.integers(2, 9))
        f = [round(float(v), 4) for v in rng.uniform(1.2, 1.6, nchan)]
        dm = [round(float(v), 1) for v in rng.uniform(0, 5000, 6)]
        ts = 0.1342
        got = oracle.delays(f, ts, dm)
        F = [Fraction(str(v)) for v in f]
        fref = max(F)
        for k, m in enumerate(dm):
            for c in range(nchan):
                x = Fraction("0.00415") * Fraction(str(m)) * (1 / F[c] ** 2 - 1 / fref**2) / Fraction(str(ts))
                if abs((x % 1) - Fraction(1, 2)) < Fraction(1, 10**9):
                    continue  # float64 may legitimately differ at an exact .5 tie
                assert got[k, c] == math.floor(x + Fraction(1, 2)), (f, m, c)


def test_table_reuse_identity():
    # PAPER.md:L98 footnote 12: x5 DM range at x5 coarser sampling uses the same shifts
    for name in ("c1", "c2", "c3", "c4", "c5"):
        wl = W.config(name)
        a = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
        b = oracle.delays(wl.freqs_GHz, 5 * wl.tsamp_s, 5 * wl.dm_list)
        assert np.array_equal(a, b), name


def test_single_sample_at_10s():
    # at 10.05 s sampling the delay for DM <~ 20000 is "contained to a single sample"
    d = oracle.delays([1.30625, 1.49375], 10.05, [20000.0])
    assert d.max() == 1


def test_cell_counts_and_distinct_vectors_golden():
    for name, cells, distinct in _rows("cell_counts.txt"):
        wl = W.config(name)
        d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
        n = oracle.cells_per_pixel(d, wl.width_list, wl.nt) * wl.npix
        assert abs(n / float(cells) - 1) < 6e-4, (name, n)
        if int(distinct):
            assert len(np.unique(d, axis=0)) == int(distinct)
    # closed form on a case with no edge loss: nt=10, no delay, widths 1,2 -> 10 + 9
    assert oracle.cells_per_pixel(np.zeros((1, 3), np.int32), [1, 2], 10) == 19


def test_width_lists_golden():
    rows = _rows("width_lists.txt")
    for n, row in zip((20, 24, 32), rows):
        assert W.log_widths(n).tolist() == [int(v) for v in row]


# ---------------------------------------------------------------- helpers (independent code)
def _np_series(cube, dvec, p):
    """Dedispersed series by numpy slicing (no loops over t)."""
    nchan, nt, _ = cube.shape
    T = nt - int(max(dvec))
    return sum(cube[c, dvec[c]:dvec[c] + T, p].astype(np.float64) for c in range(nchan))


def _py_search_pixel(cube, d, widths, p, raw_end_min=0):
    """Pure-Python brute force of O2..O6 with direct O(w) sums; tiny cubes only."""
    nchan, nt, _ = cube.shape
    best, arg = -math.inf, (-1, -1, -1)
    for k in range(d.shape[0]):
        dmax = int(d[k].max())
        T = nt - dmax
        if T < 1:
            continue
        D = [math.fsum(float(cube[c, t + d[k, c], p]) for c in range(nchan)) for t in range(T)]
        mu = math.fsum(D) / T
        var = math.fsum((x - mu) ** 2 for x in D) / T
        sig = math.sqrt(var)
        for j, w in enumerate(widths):
            for t in range(0, T - w + 1):
                if t + w - 1 + dmax < raw_end_min:
                    continue
                B = math.fsum(D[u] - mu for u in range(t, t + w))
                S = 0.0 if sig == 0 else B / (sig * math.sqrt(w))
                if S > best:
                    best, arg = S, (k, j, t)
    return best, arg


def _small_problem(seed=0, nchan=5, nt=48, npix=6, ndm=4, dm_hi=900.0, widths=(1, 2, 3, 7)):
    rng = np.random.default_rng(seed)
    cube = rng.standard_normal((nchan, nt, npix)).astype(np.float32)
    f = np.linspace(1.29, 1.52, nchan)
    d = oracle.delays(f, 0.1342, np.linspace(0, dm_hi, ndm))
    return cube, f, d, np.asarray(widths, dtype=np.int32)


# ---------------------------------------------------------------- O2..O6
def test_dm0_is_plain_channel_sum():
    cube, f, d, w = _small_problem(1)
    assert d[0].max() == 0
    r = oracle.search(cube, d, w, details=True)
    for p in range(cube.shape[2]):
        s = cube[:, :, p].astype(np.float64).sum(axis=0)
        assert abs(r.mu[p, 0] - s.mean()) < 1e-12
        assert abs(r.sigma[p, 0] - s.std()) < 1e-12  # population std (ddof=0)


def test_width1_is_normalised_series():
    cube, f, d, w = _small_problem(2)
    r = oracle.search(cube, d, w, details=True)
    j1 = int(np.nonzero(w == 1)[0][0])
    for p in range(cube.shape[2]):
        for k in range(d.shape[0]):
            D = _np_series(cube, d[k], p)
            z = (D - D.mean()) / D.std()
            assert abs(r.best[p, k, j1] - z.max()) < 1e-10
            assert r.best_t[p, k, j1] == int(z.argmax())


def test_boxcar_equals_numpy_convolve():
    cube, f, d, w = _small_problem(3, nt=80, widths=(1, 2, 5, 11, 30))
    r = oracle.search(cube, d, w, details=True)
    for p in range(cube.shape[2]):
        for k in range(d.shape[0]):
            D = _np_series(cube, d[k], p)
            for j, ww in enumerate(w):
                b = np.convolve(D - D.mean(), np.ones(ww), "valid") / (D.std() * math.sqrt(ww))
                assert len(b) == len(D) - ww + 1
                assert abs(r.best[p, k, j] - b.max()) < 1e-10
                assert r.best_t[p, k, j] == int(b.argmax())  # first maximum
        # O6: overall max and lexicographic arg-max
        flat = r.best[p].ravel()
        assert abs(r.snr[p] - flat.max()) == 0
        kk, jj = np.unravel_index(int(flat.argmax()), r.best[p].shape)
        assert (r.argmax[p, 0], r.argmax[p, 1], r.argmax[p, 2]) == (kk, jj, r.best_t[p, kk, jj])


def test_prefix_vs_direct_sum_and_python_bruteforce():
    cube, f, d, w = _small_problem(4, nchan=4, nt=40, npix=4)
    a = oracle.search(cube, d, w, details=True)
    b = oracle.search(cube, d, w, brute=True, details=True)
    assert np.allclose(a.snr, b.snr, rtol=0, atol=1e-11)
    assert np.array_equal(a.argmax, b.argmax)
    assert np.allclose(a.best, b.best, rtol=0, atol=1e-11)
    for p in range(cube.shape[2]):
        s, arg = _py_search_pixel(cube, d, w, p)
        assert abs(a.snr[p] - s) < 1e-11
        assert tuple(a.argmax[p]) == arg
        assert abs(oracle.snr_at(cube, d, w, p, *arg) - s) < 1e-11


def test_snr_at_matches_details_and_undefined_cells():
    cube, f, d, w = _small_problem(5)
    r = oracle.search(cube, d, w, details=True)
    p, k, j = 2, 3, 2
    assert abs(oracle.snr_at(cube, d, w, p, k, j, int(r.best_t[p, k, j])) - r.best[p, k, j]) < 1e-11
    T = cube.shape[1] - d[k].max()
    assert math.isnan(oracle.snr_at(cube, d, w, p, k, j, T - w[j] + 1))
    assert not math.isnan(oracle.snr_at(cube, d, w, p, k, j, T - w[j]))


def test_noise_free_pulse_closed_form():
    # cube = 0 except one boxcar on a trial's delays: S = sqrt(T_k - w) at the matched cell, any A
    nchan, nt, npix = 8, 64, 3
    f = np.linspace(1.311, 1.499, nchan)
    d = oracle.delays(f, 0.1342, [0.0, 400.0, 600.0, 1400.0])
    w = np.asarray([1, 2, 4, 8], np.int32)
    for A in (0.3, 1.5, 40.0):
        for k, j, t0 in ((2, 2, 30), (3, 3, 5), (0, 0, 63), (1, 1, 0)):
            cube = np.zeros((nchan, nt, npix), np.float32)
            for c in range(nchan):
                cube[c, t0 + d[k, c]:t0 + d[k, c] + w[j], 1] = A
            r = oracle.search(cube, d, w)
            T_k = nt - d[k].max()
            assert abs(r.snr[1] - math.sqrt(T_k - w[j])) < 1e-6 * math.sqrt(T_k)
            assert tuple(r.argmax[1]) == (k, j, t0)
            # e.g. T_k = 61, w = 4 -> sqrt(57) = 7.5498
    # empty pixels of the same cube: sigma = 0 -> S = 0 at the first cell (O5, O6)
    assert r.snr[0] == 0.0 and tuple(r.argmax[0]) == (0, 0, 0)


def test_injected_pulse_in_noise_closed_form():
    # E[S] ~= S0 q / sqrt(1 + S0^2 q / T_k), q = 1 - w/T_k  (self-contamination)
    nchan, nt = 8, 512
    f = np.linspace(1.311, 1.499, nchan)
    d = oracle.delays(f, 0.1342, [0.0, 600.0])
    w = np.asarray([1, 4, 16], np.int32)
    k, j, t0, A = 1, 1, 200, 1.5
    T_k = nt - d[k].max()
    S0 = A * w[j] * nchan / math.sqrt(w[j] * nchan)
    q = 1 - w[j] / T_k
    expect = S0 * q / math.sqrt(1 + S0 * S0 * q / T_k)
    got = []
    rng = np.random.default_rng(5)
    cube = rng.standard_normal((nchan, nt, 64)).astype(np.float32)
    for c in range(nchan):
        cube[c, t0 + d[k, c]:t0 + d[k, c] + w[j], :] += A
    for p in range(64):
        got.append(oracle.snr_at(cube, d, w, p, k, j, t0))
    got = np.asarray(got)
    assert abs(got.mean() - expect) < 0.4, (got.mean(), expect)     # scatter ~1 / sqrt(64)
    assert 0.6 < got.std() < 1.4
    assert expect < S0 - 0.3  # the bias is real: BASELINE's S0 only holds when S0^2 << T_k
    r = oracle.search(cube, d, w)
    assert (r.argmax[:, 0] == k).mean() > 0.9 and (np.abs(r.argmax[:, 2] - t0) <= 2).mean() > 0.9


def test_offset_scale_permutation_invariance():
    cube, f, d, w = _small_problem(6)
    r0 = oracle.search(cube, d, w)
    rng = np.random.default_rng(0)
    off = rng.uniform(-3, 3, (cube.shape[0], 1, cube.shape[2]))
    r1 = oracle.search((cube.astype(np.float64) * 1.0 + off).astype(np.float32), d, w)
    assert np.allclose(r0.snr, r1.snr, atol=2e-5) and (r0.argmax == r1.argmax).mean() > 0.8
    r2 = oracle.search(cube * np.float32(4.0), d, w)  # exact power-of-two scale
    assert np.allclose(r0.snr, r2.snr, atol=1e-12) and np.array_equal(r0.argmax, r2.argmax)
    perm = rng.permutation(cube.shape[0])
    d3 = oracle.delays(f[perm], 0.1342, np.linspace(0, 900.0, 4))
    r3 = oracle.search(cube[perm], d3, w)
    assert np.allclose(r0.snr, r3.snr, atol=1e-10) and np.array_equal(r0.argmax, r3.argmax)


def test_duplicate_dm_never_changes_result():
    cube, f, d, w = _small_problem(7)
    r0 = oracle.search(cube, d, w)
    d2 = np.concatenate([d, d[1:2], d[0:1]], axis=0)
    r1 = oracle.search(cube, d2, w)
    assert np.array_equal(r0.snr, r1.snr) and np.array_equal(r0.argmax, r1.argmax)
    # a duplicate placed FIRST takes over the index (lowest k wins exact ties, R17)
    d3 = np.concatenate([d[3:4], d], axis=0)
    r2 = oracle.search(cube, d3, w)
    moved = r0.argmax[:, 0] == 3
    assert np.array_equal(r2.argmax[moved, 0], np.zeros(moved.sum(), np.int64))
    assert np.array_equal(r2.argmax[~moved, 0], r0.argmax[~moved, 0] + 1)


def test_time_shift_equivariance():
    # exactly true only if mu, sigma are unchanged: content confined to an interior interval
    nchan, nt, npix, m = 5, 96, 4, 7
    f = np.linspace(1.29, 1.52, nchan)
    d = oracle.delays(f, 0.1342, np.linspace(0, 900.0, 4))
    w = np.asarray([1, 2, 5], np.int32)
    rng = np.random.default_rng(8)
    a = np.zeros((nchan, nt, npix), np.float32)
    lo, hi = 20, 60
    a[:, lo:hi, :] = rng.standard_normal((nchan, hi - lo, npix)).astype(np.float32)
    b = np.zeros_like(a)
    b[:, lo + m:hi + m, :] = a[:, lo:hi, :]
    ra, rb = oracle.search(a, d, w), oracle.search(b, d, w)
    assert np.allclose(ra.snr, rb.snr, atol=1e-12)
    assert np.array_equal(ra.argmax[:, :2], rb.argmax[:, :2])
    assert np.array_equal(ra.argmax[:, 2] + m, rb.argmax[:, 2])


def test_degenerate_outputs():
    nchan, nt, npix = 3, 16, 2
    d = np.zeros((2, nchan), np.int32)
    d[1] = [5, 2, 0]
    # constant pixel: sigma = 0 -> every S = 0 -> first cell wins
    cube = np.full((nchan, nt, npix), 2.0, np.float32)
    r = oracle.search(cube, d, [1, 3])
    assert np.all(r.snr == 0.0) and np.all(r.argmax == 0)
    # widths all longer than every series: no cell defined
    r = oracle.search(cube, d, [17, 40])
    assert np.all(np.isneginf(r.snr)) and np.all(r.argmax == -1)
    # width fits DM 0 (T=16) but not DM 1 (T=11): skipped, not an error
    cube2 = np.random.default_rng(0).standard_normal((nchan, nt, npix)).astype(np.float32)
    r = oracle.search(cube2, d, [12], details=True)
    assert np.all(r.argmax[:, 0] == 0) and np.all(np.isneginf(r.best[:, 1, 0]))
    # strict threshold (R16)
    assert len(r.candidates(float(r.snr.max()))) == 0
    assert len(r.candidates(float(np.nextafter(r.snr.max(), -np.inf)))) == 1


# ---------------------------------------------------------------- S1..S6
def test_streaming_rules_against_python_bruteforce():
    nchan, npix, L, C = 4, 3, 40, 5
    f = np.linspace(1.29, 1.52, nchan)
    d = oracle.delays(f, 0.1342, [0.0, 500.0, 1100.0])
    w = np.asarray([1, 3, 8, 30], np.int32)
    rng = np.random.default_rng(9)
    so = oracle.StreamOracle(nchan, npix, L, d, w)
    full = np.zeros((nchan, 0, npix), np.float32)
    for push in range(14):
        chunk = rng.standard_normal((nchan, C, npix)).astype(np.float32)
        full = np.concatenate([full, chunk], axis=1)
        r = so.push(chunk, details=True)
        n, n_prev = full.shape[1], full.shape[1] - C
        lo = max(0, n - L)
        ring = full[:, lo:n, :]
        for p in range(npix):
            s, arg = _py_search_pixel(ring, d, w, p, raw_end_min=n_prev - lo)
            if arg[0] < 0:
                assert np.isneginf(r.snr[p]) and tuple(r.argmax[p]) == (-1, -1, -1)
            else:
                assert abs(r.snr[p] - s) < 1e-11
                assert tuple(r.argmax[p]) == (arg[0], arg[1], arg[2] + lo)  # absolute t (S6)
        # S5: in steady state exactly C windows per (k, j)
        if n >= L + C:
            for k in range(d.shape[0]):
                dmax = int(d[k].max())
                T_k = L - dmax
                for j, ww in enumerate(w):
                    cnt = sum(1 for t in range(T_k - ww + 1) if t + ww - 1 + dmax >= n_prev - lo)
                    assert cnt == C


def test_streaming_push_equals_offline_on_ring():
    nchan, npix, L, C = 4, 5, 64, 8
    f = np.linspace(1.29, 1.52, nchan)
    d = oracle.delays(f, 0.1342, [0.0, 700.0])
    w = np.asarray([1, 4, 16], np.int32)
    rng = np.random.default_rng(10)
    so = oracle.StreamOracle(nchan, npix, L, d, w)
    data = rng.standard_normal((nchan, 12 * C, npix)).astype(np.float32)
    for i in range(12):
        r = so.push(data[:, i * C:(i + 1) * C, :])
    lo = 12 * C - L
    off = oracle.search(data[:, lo:, :], d, w, raw_end_min=L - C, t_offset=lo)
    assert np.array_equal(off.snr, r.snr) and np.array_equal(off.argmax, r.argmax)
    # without the S5 restriction the offline result can only be >=
    assert np.all(oracle.search(data[:, lo:, :], d, w).snr >= r.snr)


# ---------------------------------------------------------------- BASELINE config 1 as specified
def test_config1_as_literally_specified():
    exp = {}
    for row in _rows("c1_oracle_expected.txt"):
        exp[row[0]] = row[1:]
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl)
    W.inject(cube, W.injection_table(wl, d), d, extra_delays=oracle.delays(wl.freqs_GHz, wl.tsamp_s, [500.0])[0])
    r = oracle.search(cube.numpy(), d, wl.width_list)
    p = int(exp["pulse_pixel"][0])
    assert p == 20 * 32 + 11
    assert abs(r.snr[p] - float(exp["pulse_pixel"][2])) < 1e-9
    assert r.argmax[p].tolist() == [int(v) for v in exp["pulse_pixel"][4:7]]
    # 5.728 at (0, 2, 31), pulse pixel is the map maximum, no candidate above 6
    assert abs(r.snr[p] - 5.728) < 1e-3 and int(r.snr.argmax()) == p
    assert len(r.candidates(wl.threshold)) == 0 and len(r.candidates(5.0)) == 1
    # nominal S0 = 1.5*4*8/sqrt(32) = 8.49 is NOT what a 64-sample series can return
    assert abs(1.5 * 4 * 8 / math.sqrt(32) - 8.485) < 1e-3


def test_multithreaded_oracle_is_identical():
    cube, f, d, w = _small_problem(12, npix=37)
    a = oracle.search(cube, d, w, nthreads=1)
    b = oracle.search(cube, d, w, nthreads=5)
    assert np.array_equal(a.snr, b.snr) and np.array_equal(a.argmax, b.argmax)
    sel = np.asarray([5, 0, 36, 5])
    c = oracle.search(cube, d, w, pixels=sel, nthreads=3)
    assert np.array_equal(c.snr, a.snr[sel]) and np.array_equal(c.argmax, a.argmax[sel])


# ----------------------------------------------------------------------------- NEXT 2: time binning (R24)
def test_bin_time_pins():
    """oracle.bin_time against what the definition fixes (reading R24): a constant cube bins to
    factor x constant, factor 1 is the identity, trailing samples are dropped, it equals a reshape-sum (library
    routine), it composes (x5 then x15 == x75, the paper's two binned timescales) and conserves the total."""
    rng = np.random.default_rng(77)
    a = rng.standard_normal((3, 157, 5)).astype(np.float32)
    assert np.array_equal(oracle.bin_time(a, 1), a)
    assert np.array_equal(oracle.bin_time(np.full((2, 10, 3), 1.5, np.float32), 5), np.full((2, 2, 3), 7.5, np.float32))
    b5 = oracle.bin_time(a, 5)
    assert b5.shape == (3, 31, 5)                      # floor(157/5); samples 155, 156 dropped
    ref = a[:, :155, :].astype(np.float64).reshape(3, 31, 5, 5).sum(axis=2)
    assert np.allclose(b5, ref, rtol=0, atol=1e-6)
    assert np.array_equal(b5, ref.astype(np.float32))  # one rounding of the float64 sum
    x = rng.integers(-8, 9, size=(2, 150, 4)).astype(np.float32)   # integers: every sum is exact in float32
    assert np.array_equal(oracle.bin_time(oracle.bin_time(x, 5), 15), oracle.bin_time(x, 75))
    assert oracle.bin_time(x, 75).sum() == x.sum()
    assert oracle.bin_time(a, 200).shape == (3, 0, 5)  # factor > nt: nothing left


def test_binned_search_reuses_the_delay_table():
    """Footnote 12: searching the x5-binned cube at 5x the DMs uses the same integer shifts, so a
    pulse injected at trial k of the fine grid with 5x the delays and 5x the width is recovered at the same (k, j)."""
    f = np.linspace(1.311, 1.499, 8)
    dms = np.linspace(0.0, 1400.0, 8)
    d1 = oracle.delays(f, 0.1342, dms)
    d5 = oracle.delays(f, 5 * 0.1342, 5 * dms)
    assert np.array_equal(d1, d5)
    nt, k, w, t0 = 1200, 5, 4, 100                    # in binned units; the cube is built at the fine sampling
    cube = np.zeros((8, nt, 1), np.float32)
    for c in range(8):
        s = 5 * (t0 + d5[k][c])
        cube[c, s:s + 5 * w, 0] = 1.0
    r = oracle.search(oracle.bin_time(cube, 5), d5, [1, 2, 4, 8, 16])
    assert tuple(r.argmax[0]) == (k, 2, t0)
    Tk = nt // 5 - d5[k].max()
    assert abs(r.snr[0] - np.sqrt(Tk - w)) < 1e-9      # noise-free closed form, as in the unbinned pin


def test_per_trial_width_maxima_are_consistent():
    """The oracle's [ndm][nw] cubes (details=True; PAPER.md:L94 keeps S/N and TOA for all widths and DMs): their maximum
    is the map, the arg of the maximum is the arg-max, and the prefix and brute-force routines agree on them."""
    rng = np.random.default_rng(94)
    cube = rng.standard_normal((4, 90, 6)).astype(np.float32)
    d = np.asarray([[0, 0, 0, 0], [3, 2, 1, 0], [7, 5, 2, 0]], dtype=np.int32)
    w = [1, 4, 13, 200]
    a = oracle.search(cube, d, w, details=True)
    b = oracle.search(cube, d, w, details=True, brute=True)
    assert np.allclose(a.best[:, :, :3], b.best[:, :, :3], rtol=0, atol=1e-12) and np.array_equal(a.best_t, b.best_t)
    assert np.all(np.isneginf(a.best[:, :, 3])) and np.all(a.best_t[:, :, 3] == -1)      # width 200 > 90 samples
    flat = a.best.reshape(6, -1)
    assert np.array_equal(flat.max(axis=1), a.snr)
    k, j = np.unravel_index(flat.argmax(axis=1), (3, 4))
    assert np.array_equal(np.stack([k, j, a.best_t[np.arange(6), k, j]], axis=1), a.argmax)
    # a width-1 maximum is the largest normalised sample of the dedispersed series (DM 0 row)
    D0 = cube.astype(np.float64).sum(axis=0)
    z = (D0 - D0.mean(axis=0)) / D0.std(axis=0)
    assert np.allclose(a.best[:, 0, 0], z.max(axis=0), rtol=0, atol=1e-12) and np.array_equal(a.best_t[:, 0, 0], z.argmax(axis=0))


# ---- NEXT 1 (first part): per-(channel, pixel) median subtraction (reading R29) ------------------------

@pytest.mark.parametrize("nt", [1, 2, 3, 24, 25, 64, 101])
def test_median_matches_numpy_routine_and_rank_definition(nt):
    rng = np.random.default_rng(nt)
    a = rng.normal(size=(3, nt, 7)).astype(np.float32)
    a[0, :, 0] = np.round(a[0, :, 0])                    # ties
    out, med = oracle.median_subtract(a)
    assert np.array_equal(med, np.median(a.astype(np.float64), axis=1).astype(np.float32))
    assert np.array_equal(out, a - med[:, None, :]) and out.dtype == np.float32
    # the definition by counting: at least half of the samples are <= m and at least half are >= m
    for c in range(3):
        for p in range(7):
            x, m = a[c, :, p].astype(np.float64), float(med[c, p])
            lo, hi = np.sort(x)[(nt - 1) // 2], np.sort(x)[nt // 2]
            assert lo <= m <= hi or np.isclose(m, 0.5 * (lo + hi), rtol=1e-7, atol=0)
            assert 2 * np.sum(x <= hi) >= nt and 2 * np.sum(x >= lo) >= nt


def test_median_closed_forms_and_invariances():
    t = np.arange(25, dtype=np.float32)
    a = np.stack([t, t[::-1], np.full(25, 3.5, np.float32)])[:, :, None]          # [3][25][1]
    out, med = oracle.median_subtract(a)
    assert med.ravel().tolist() == [12.0, 12.0, 3.5] and np.array_equal(out[0, :, 0], t - 12) and not out[2].any()
    out, med = oracle.median_subtract(np.asarray([1.0, 4.0], np.float32).reshape(1, 2, 1))
    assert med.ravel().tolist() == [2.5] and out.ravel().tolist() == [-1.5, 1.5]
    out, med = oracle.median_subtract(np.asarray([7.0], np.float32).reshape(1, 1, 1))
    assert med.ravel().tolist() == [7.0] and out.ravel().tolist() == [0.0]
    # one outlier does not move it (the reason the paper uses a median, L75 / L130)
    x = np.asarray([0, 1, 2, 3, 1e6], np.float32).reshape(1, 5, 1)
    assert oracle.median_subtract(x)[1].ravel().tolist() == [2.0]
    # permutation of the samples: same median; integer shift: exact equivariance; already subtracted: median 0
    rng = np.random.default_rng(0)
    a = rng.integers(-50, 50, size=(2, 40, 5)).astype(np.float32)
    _, m0 = oracle.median_subtract(a)
    _, m1 = oracle.median_subtract(a[:, rng.permutation(40), :])
    o2, m2 = oracle.median_subtract(a + 17.0)
    assert np.array_equal(m0, m1) and np.array_equal(m2, m0 + 17.0)
    assert not oracle.median_subtract(o2)[1].any()


def test_median_subtraction_cancels_in_the_search():
    """Reading R6/R29: the per-(pixel, DM) mean of O3 removes any per-channel constant, so subtracting the
    channel medians first changes no S/N beyond rounding -- which is why the median is NEXT 1 and not on the path."""
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl).numpy()[:, :, :40]
    r0 = oracle.search(cube, d, wl.width_list)
    r1 = oracle.search(oracle.median_subtract(cube)[0], d, wl.width_list)
    assert np.allclose(r0.snr, r1.snr, rtol=0, atol=2e-5)
    assert (r0.argmax == r1.argmax).all(axis=1).mean() > 0.95


# ---- NEXT 1 (second part): running standard deviation (reading R30) ----------------------------

def test_sigma_norm_scales_every_snr_and_keeps_the_argmax():
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl).numpy()[:, :, :30]
    r0 = oracle.search(cube, d, wl.width_list, details=True)
    r1 = oracle.search(cube, d, wl.width_list, details=True, sigma_norm=r0.sigma)          # own sigma: identity
    assert np.array_equal(r0.snr, r1.snr) and np.array_equal(r0.argmax, r1.argmax) and np.array_equal(r0.best, r1.best)
    r2 = oracle.search(cube, d, wl.width_list, details=True, sigma_norm=4.0 * r0.sigma)    # power of two: exact
    assert np.array_equal(r2.snr, r0.snr / 4.0) and np.array_equal(r2.argmax, r0.argmax)
    assert np.array_equal(r2.sigma, r0.sigma)                                              # still this call's sigma
    # a per-trial factor: each (pixel, k) row of the maxima scales by its own factor; the winner is the max of those
    rng = np.random.default_rng(0)
    f = rng.uniform(0.5, 2.0, size=r0.sigma.shape)
    r3 = oracle.search(cube, d, wl.width_list, details=True, sigma_norm=f * r0.sigma)
    want = r0.best / f[:, :, None]
    assert np.allclose(r3.best, want, rtol=1e-12, atol=0)
    assert np.allclose(r3.snr, want.reshape(want.shape[0], -1).max(axis=1), rtol=1e-12, atol=0)
    assert np.array_equal(r3.best_t, r0.best_t)
    # brute-force boxcar route agrees
    r4 = oracle.search(cube[:, :, :6], d, wl.width_list, brute=True, sigma_norm=(f * r0.sigma)[:6])
    assert np.allclose(r4.snr, r3.snr[:6], rtol=1e-9, atol=1e-12)
    # sigma_norm = 0 -> S = 0 (the O5 convention), as for a flat series
    z = oracle.search(cube[:, :, :3], d, wl.width_list, sigma_norm=np.zeros((3, len(wl.dm_list))))
    assert not z.snr.any()


def test_running_variance_recursion_closed_form():
    a = 0.25
    v = None
    for _ in range(6):
        v = oracle.running_variance(v, np.asarray([[2.0]]), a)
    assert v[0, 0] == 4.0                                           # constant sigma: fixed point
    v = np.asarray([[9.0]])
    for n in range(1, 8):                                           # step from 9 to 1: v_n = 1 + 8 (1-a)^n
        v = oracle.running_variance(v, np.asarray([[1.0]]), a)
        assert v[0, 0] == pytest.approx(1.0 + 8.0 * (1 - a) ** n, rel=1e-14)
    assert oracle.running_variance(np.asarray([[9.0]]), np.asarray([[3.0]]), 1.0)[0, 0] == 9.0    # alpha = 1: instantaneous
    # undefined trials: NaN sigma keeps the state; a first defined sigma starts it
    v = oracle.running_variance(np.asarray([[np.nan, 4.0]]), np.asarray([[3.0, np.nan]]), a)
    assert v.tolist() == [[9.0, 4.0]]


def test_running_sigma_stream_alpha_one_is_the_plain_stream_and_bias_is_removed():
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    rng = np.random.default_rng(4)
    npix = 12
    plain = oracle.StreamOracle(wl.nchan, npix, wl.nt, d, wl.width_list)
    run1 = oracle.RunningStreamOracle(wl.nchan, npix, wl.nt, d, wl.width_list, alpha=1.0)
    runs = oracle.RunningStreamOracle(wl.nchan, npix, wl.nt, d, wl.width_list, alpha=0.05)
    for i in range(5):
        chunk = rng.normal(size=(wl.nchan, wl.chunk_nt, npix)).astype(np.float32)
        if i == 4:   # a bright, wide, undispersed pulse in pixel 3: it inflates this push's own sigma (L130)
            chunk[:, 5:5 + 16, 3] += 3.0
        a, b, c = plain.push(chunk), run1.push(chunk), runs.push(chunk)
        assert np.array_equal(a.snr, b.snr) and np.array_equal(a.argmax, b.argmax)           # alpha = 1
    assert c.snr[3] > 1.15 * a.snr[3]            # the slowly updated sigma is not contaminated by the pulse
    others = np.arange(npix) != 3
    assert np.allclose(c.snr[others], a.snr[others], rtol=0.35)   # 25..64-sample sigmas scatter by ~15 %
