"""-m gpu: the CUDA path through the C ABI vs the oracle, element by element (P-rule)."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2510_18136_b200 import workloads as W
from tests import parity_util as PU

pytestmark = pytest.mark.gpu


def _nsfrb():
    from paper_2510_18136_b200 import nsfrb
    return nsfrb


def _offline(wl, cube, *, pixels=None, capacity=4096, label=None):
    """Run nsfrb_search on the device cube; compare `pixels` (default all) with the oracle."""
    nsfrb = _nsfrb()
    d_orc = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    with nsfrb.Plan.for_workload(wl, cand_capacity=capacity) as plan:
        assert np.array_equal(plan.delays(), d_orc), "delay table must be bit-exact"
        res = plan.search(cube)
        torch.cuda.synchronize()
        snr = res.snr_map.cpu().numpy()
        arg = res.argmax.cpu().numpy().T.copy()
        cands = res.candidates()
        nfound = res.n_found()
        info = plan.info()
    assert info["cells_per_pixel"] == oracle.cells_per_pixel(d_orc, wl.width_list, wl.nt)
    pix = np.arange(wl.npix) if pixels is None else np.asarray(pixels)
    sub = cube[:, :, torch.as_tensor(pix, device=cube.device)].cpu().numpy()
    st = PU.check(sub, d_orc, wl.width_list, snr[pix], arg[pix], wl.threshold, label=label or wl.name)
    print(f"[parity] {label or wl.name}: n={st['n']} exact={st['exact']} adjudicated={st['adjudicated']} "
          f"undefined={st['undefined']} worst |d|/tol={st['worst_tol_frac']:.3f}")
    cs = PU.check_candidates(st["oracle"], pix, cands, nfound, wl.threshold, capacity, all_pixels_checked=pixels is None)
    # stored candidate records repeat the maps exactly
    for c in cands:
        p = int(c["pixel"])
        assert c["snr"] == snr[p] and (c["dm_idx"], c["width_idx"], c["t"]) == tuple(arg[p])
        assert c["snr"] > wl.threshold
    return st, cs, snr, arg


def _inject_all(wl, cube, d):
    pulses = W.injection_table(wl, d)
    W.inject(cube, pulses, d)
    return pulses


# ----------------------------------------------------------------------------- config 1
def test_c1_as_specified():
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    W.inject(cube, W.injection_table(wl, d), d, extra_delays=oracle.delays(wl.freqs_GHz, wl.tsamp_s, [500.0])[0])
    st, cs, snr, arg = _offline(wl, cube)
    p = 20 * 32 + 11
    assert abs(snr[p] - 5.728493) < 1e-3 and tuple(arg[p]) == (0, 2, 31)
    assert cs["found"] == 0            # an empty candidate list is the right answer here
    assert st["adjudicated"] <= 0.1 * st["n"]


def test_c1b_threshold5_has_one_candidate():
    from dataclasses import replace
    wl = replace(W.config("c1"), threshold=5.0)
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    W.inject(cube, W.injection_table(wl, d), d, extra_delays=oracle.delays(wl.freqs_GHz, wl.tsamp_s, [500.0])[0])
    st, cs, snr, arg = _offline(wl, cube)
    assert cs["found"] == 1


def test_c1c_long_series_pulse_on_grid():
    # nt = 2048, DM 600 on the trial grid: BASELINE's S0 = A w nchan / (sigma sqrt(w nchan)) regime
    from dataclasses import replace
    wl = replace(W.config("c1"), nt=2048, name="c1c")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    rng = np.random.default_rng(0)
    cube = torch.from_numpy(rng.standard_normal((wl.nchan, wl.nt, wl.npix)).astype(np.float32)).cuda()
    W.inject(cube, [W.Pulse(pixel=651, dm_idx=3, width_idx=2, t0=1000, width=4, s0=8.49, amp=1.5)], d)
    st, cs, snr, arg = _offline(wl, cube)
    assert tuple(arg[651][:2]) == (3, 2) and abs(arg[651][2] - 1000) <= 1
    assert 6.5 < snr[651] < 10.5 and cs["found"] >= 1


# ----------------------------------------------------------------------------- scaled C3, C4, C5
@pytest.mark.parametrize("name,nx,ny,nt", [
    ("c3", 12, 8, None),      # full 4096-sample series, 32 DMs x 24 widths, sky term
    ("c3", 7, 5, 1000),       # ragged: nt not a multiple of the block, npix not a multiple of 32
    ("c4", 40, 25, None),     # 64 DMs (44 distinct vectors), Fibonacci widths, channel gains
    ("c5", 8, 6, None),       # 64 channels, 256 DMs, 32 widths, RFI spikes
    ("c5", 5, 3, 1500),       # widths up to 1200 on a 1500-sample cube
])
def test_scaled_configs(name, nx, ny, nt):
    wl = W.config(name).scaled(nx, ny, nt, n_pulses=min(W.config(name).n_pulses, nx * ny // 3))
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    pulses = _inject_all(wl, cube, d)
    st, cs, snr, arg = _offline(wl, cube)
    assert st["exact"] >= 0.9 * st["n"], st
    _check_recovery(wl, d, pulses, snr)


@pytest.mark.parametrize("name,nx,ny,nt,batch,side", [
    ("c3", 12, 8, 1000, 16, "1"),    # six full batches, the next one moved by the search CTAs themselves
    ("c3", 7, 5, 600, 8, "1"),       # ragged last batch (3 pixels), npix not a multiple of 8
    ("c4", 9, 5, None, 16, "1"),     # three DM groups per pixel: 24 members share a group of 8 pixels; series inside the ring
    ("c5", 5, 5, 700, 8, "1"),       # 64 channels, 16 groups: many more side rows than time blocks
    ("c3", 7, 5, 600, 8, "0"),       # the same pipeline with standalone layout kernels
    ("c5-16dm", 5, 4, 256, 8, "1"),  # one DM group, one time block, 64 channels: eight side steps after the only block
])
def test_offline_pixel_batches(monkeypatch, name, nx, ny, nt, batch, side):
    """nsfrb_search walks the image in pixel batches through two workspaces; while batch i is searched its CTAs move
    batch i+1 from the caller's [chan][time][pixel] cube into the other workspace.  Forced to tiny
    batches here, the result must equal the oracle on every pixel, and the one-batch run bit for bit."""
    from dataclasses import replace
    wl = W.config(name.split("-")[0]).scaled(nx, ny, nt, n_pulses=4)
    if name.endswith("16dm"):
        wl = replace(wl, dm_list=wl.dm_list[:16])
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    cube += 50.0 * torch.randn((wl.nchan, 1, wl.npix), device="cuda")    # per-(channel, pixel) offsets: the baseline removal
    _inject_all(wl, cube, d)
    st1, cs1, snr1, arg1 = _offline(wl, cube, label=f"{name} one batch")
    monkeypatch.setenv("NSFRB_SEARCH_BATCH_PIX", str(batch))
    monkeypatch.setenv("NSFRB_SEARCH_SIDE", side)
    st, cs, snr, arg = _offline(wl, cube, label=f"{name} batches of {batch}")
    assert np.array_equal(snr, snr1) and np.array_equal(arg, arg1)


def test_search_host_stages_pixel_batches_from_the_host_cube(monkeypatch):
    """nsfrb_search_host on a plan that needs several pixel batches: strided host -> device copies of one batch at a time
    on a copy stream, overlapped with the search; the result must equal nsfrb_search on the device cube bit for bit."""
    nsfrb = _nsfrb()
    monkeypatch.setenv("NSFRB_SEARCH_BATCH_PIX", "16")
    wl = W.config("c3").scaled(9, 7, 900, n_pulses=3)            # 63 pixels: three full batches and a ragged one
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    _inject_all(wl, cube, d)
    host = cube.cpu().pin_memory()
    with nsfrb.Plan.for_workload(wl) as plan:
        for _ in range(2):                                       # twice: the slabs and events are reused
            h = plan.search_host(host)
            dres = plan.search(cube)
            torch.cuda.synchronize()
            assert torch.equal(h[0], dres.snr_map.cpu()) and torch.equal(h[1], dres.argmax.cpu())
            assert int(h[3].numpy().view(np.uint32)[0]) == dres.n_found()


def _check_recovery(wl, d, pulses, snr, frac=0.7):
    """Injected single pulses come back at >= frac of the closed form S0 q / sqrt(1 + S0^2 q / T_k)
    (SURVEY 8(c) 'Injected pulse in noise'; the max over cells can only be higher)."""
    n = 0
    for pu in pulses:
        if pu.train_period or pu.dm_idx < 0:
            continue
        T_k = wl.nt - int(d[pu.dm_idx].max())
        q = 1.0 - pu.width / T_k
        expect = pu.s0 * q / np.sqrt(1.0 + pu.s0 ** 2 * q / T_k)
        assert snr[pu.pixel] >= frac * expect - 1.0, (pu, float(snr[pu.pixel]), expect)
        n += 1
    return n


# ----------------------------------------------------------------------------- streaming (C2)
def _stream_case(wl, n_push, eval_at, chunk_sizes=None, capacity=1024, cubes=False, expect_mode=None):
    nsfrb = _nsfrb()
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    src = W.ChunkSource(wl, d, n_push, "cuda")
    so = oracle.StreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list)
    stats = []
    with nsfrb.Plan.for_workload(wl, cand_capacity=capacity) as plan:
        out = plan.alloc_outputs()
        if cubes:
            shape = (len(wl.dm_list), len(wl.width_list), wl.npix)
            cs, ct = torch.zeros(shape, device="cuda"), torch.zeros(shape, dtype=torch.int32, device="cuda")
            plan.stream_set_cubes(cs, ct)
        for i in range(n_push):
            if chunk_sizes is None:
                chunk = src.next()
            else:
                c = chunk_sizes[i % len(chunk_sizes)]
                chunk = torch.randn((wl.nchan, c, wl.npix), device="cuda", generator=src.g)
            plan.stream_push(chunk, out)
            torch.cuda.synchronize()
            if expect_mode is not None:
                assert plan.stream_mode() == expect_mode
            ch = chunk.cpu().numpy()
            n_prev = so.n
            so.n += ch.shape[1]
            so.hist = np.concatenate([so.hist, ch], axis=1)[:, -so.L:, :]
            if i in eval_at:
                lo = max(0, so.n - so.L)
                snr = out.snr_map.cpu().numpy()
                arg = out.argmax.cpu().numpy().T.copy()
                st = PU.check(so.hist, d, wl.width_list, snr, arg, wl.threshold, raw_end_min=n_prev - lo,
                              t_offset=lo, label=f"{wl.name} push {i}")
                PU.check_candidates(st["oracle"], np.arange(wl.npix), out.candidates(), out.n_found(), wl.threshold,
                                    capacity)
                if cubes:  # the maps are the maxima of the cubes, bit for bit, and the arg-max entry holds the map's t
                    S = cs.cpu().numpy().reshape(-1, wl.npix)
                    assert np.array_equal(S.max(axis=0), snr)
                    has = arg[:, 0] >= 0
                    pp = np.nonzero(has)[0]
                    assert np.array_equal(ct.cpu().numpy()[arg[pp, 0], arg[pp, 1], pp], arg[pp, 2])
                stats.append(st)
        # offline search is refused while the plan holds streamed samples
        cube = torch.zeros((wl.nchan, wl.nt, wl.npix), device="cuda")
        with pytest.raises(nsfrb.NsfrbError) as ei:
            plan.search(cube)
        assert ei.value.code == nsfrb.NSFRB_ESTATE
        plan.stream_reset()
        plan.search(cube)
        torch.cuda.synchronize()
    return stats


def test_stream_c2_scaled():
    wl = W.config("c2").scaled(12, 8)
    # first pushes (ring nearly empty), mid fill, the pushes around the ring wrap (1536/25 = 61.44), steady state
    stats = _stream_case(wl, 68, eval_at={0, 1, 2, 7, 30, 48, 60, 61, 62, 63, 67})
    assert sum(s["exact"] for s in stats) >= 0.9 * sum(s["n"] - s["undefined"] for s in stats)


def test_stream_small_ring_variable_chunks():
    from dataclasses import replace
    wl = replace(W.config("c2").scaled(9, 5, nt=300), width_list=np.asarray([1, 2, 5, 16, 40, 120, 250], np.int32))
    _stream_case(wl, 40, eval_at=set(range(40)), chunk_sizes=[25, 1, 7, 60, 300, 13])


@pytest.mark.parametrize("env,nt,mode", [
    ({}, 256, 3),                                                  # default: dedispersed history + 8-row block sums
    ({"NSFRB_STREAM_COARSE": "0"}, 256, 2),                        # history, plain runs row by row
    ({}, 250, 2),                                                  # ring length not a multiple of 8: no block sums
    ({"NSFRB_STREAM_DHIST": "0"}, 256, 1),                         # raw ring: the march dedisperses
    ({"NSFRB_STREAM_VARIANT": "8,2,1,4,4,2"}, 256, 3),             # other tile shapes of the history march ...
    ({"NSFRB_STREAM_VARIANT": "2,8,1,2,4,0"}, 256, 3),
    ({"NSFRB_STREAM_VARIANT": "3,2,2,4,2,2"}, 256, 3),             # ... padding trials (16 = 5 x 3 + 1) and two time segments
    ({"NSFRB_STREAM_DHIST": "0", "NSFRB_STREAM_VARIANT": "8,2,2,2,3,6"}, 256, 1),   # ... and of the raw march
    ({"NSFRB_STREAM_DHIST": "0", "NSFRB_STREAM_LIGHT": "0"}, 256, 1),
    ({"NSFRB_STREAM_STATS": "march"}, 256, 1),                     # round-1 behaviour: statistics in the march itself
])
def test_stream_modes_and_tile_shapes(monkeypatch, env, nt, mode):
    """Every way the real-time path can hold and march its data (nsfrb_stream_mode, the NSFRB_STREAM_* knobs of DESIGN.md 7.4)
    gives the oracle's result on every push: eight laps of a short ring, chunk sizes from 1 sample to (nearly) the whole ring,
    widths up to the ring length (plain runs with ragged ends on both sides of the 8-row blocks, wrap-around of the slots)."""
    from dataclasses import replace
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    wl = replace(W.config("c2").scaled(9, 5, nt=nt), width_list=np.asarray([1, 2, 5, 16, 40, 70, 120, 245], np.int32))
    _stream_case(wl, 48, eval_at=set(range(48)), chunk_sizes=[25, 1, 7, 60, 250, 13, 25, 25], expect_mode=mode)


def test_stream_equals_offline_on_ring_contents():
    nsfrb = _nsfrb()
    wl = W.config("c2").scaled(8, 4, nt=256)
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    g = torch.Generator(device="cuda").manual_seed(5)
    data = torch.randn((wl.nchan, 20 * 25, wl.npix), device="cuda", generator=g)
    with nsfrb.Plan.for_workload(wl) as plan:
        for i in range(20):
            out = plan.stream_push(data[:, i * 25:(i + 1) * 25, :].contiguous())
        torch.cuda.synchronize()
        s_stream = out.snr_map.cpu().numpy()
    lo = 20 * 25 - wl.nt
    ring = data[:, lo:, :].contiguous().cpu().numpy()
    r = oracle.search(ring, d, wl.width_list, raw_end_min=wl.nt - 25, t_offset=lo)
    assert np.all(np.abs(s_stream - r.snr) <= PU.tol(r.snr))



def test_stream_incremental_statistics_offsets_many_laps_and_reset(monkeypatch):
    """k_stream_stats carries float64 sums of D and D^2 across pushes.  Twelve laps of a short ring with
    irregular chunk sizes, on data whose level jumps far away from the first sample (the stored baseline) and then drifts,
    so the mean square is ~10^3 times the variance: every evaluated push must still match the two-pass float64 oracle,
    also after nsfrb_stream_reset (the sums restart).  The v4 march (NSFRB_STREAM_STATS=march: one-pass float32 sums about
    the previous push's mean) must agree with it once it has a provisional mean, i.e. from the second push on; on the very
    first push of such data it is off by 1.3 tolerances, which is one reason it is no longer the default."""
    from dataclasses import replace
    nsfrb = _nsfrb()
    wl = replace(W.config("c2").scaled(7, 5, nt=200), width_list=np.asarray([1, 3, 9, 30, 100, 180], np.int32))
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    sizes = [25, 3, 25, 11, 40, 1]
    g = torch.Generator(device="cuda").manual_seed(77)
    level = 30.0 * torch.randn((wl.nchan, 1, wl.npix), device="cuda", generator=g)
    chunks, t0 = [], 0
    for i in range(140):
        c = sizes[i % len(sizes)]
        t = torch.arange(t0, t0 + c, device="cuda", dtype=torch.float32).view(1, c, 1)
        x = torch.randn((wl.nchan, c, wl.npix), device="cuda", generator=g)
        x = x + (level + 0.002 * t) * (t >= 1)          # sample 0 stays at noise level: it becomes the baseline
        chunks.append(x.contiguous())
        t0 += c
    eval_at = {0, 1, 5, 9, 10, 33, 70, 100, 120, 139}

    def run(order, check=True):
        maps = {}
        with nsfrb.Plan.for_workload(wl, cand_capacity=64) as plan:
            out = plan.alloc_outputs()
            for rep in order:
                hist, n = np.zeros((wl.nchan, 0, wl.npix), np.float32), 0
                if rep:
                    plan.stream_reset()
                for i, ch in enumerate(chunks if rep == 0 else chunks[:40]):
                    plan.stream_push(ch, out)
                    n_prev, n = n, n + ch.shape[1]
                    hist = np.concatenate([hist, ch.cpu().numpy()], axis=1)[:, -wl.nt:, :]
                    if i in eval_at:
                        torch.cuda.synchronize()
                        lo = max(0, n - wl.nt)
                        snr = out.snr_map.cpu().numpy()
                        arg = out.argmax.cpu().numpy().T.copy()
                        if check:
                            PU.check(hist, d, wl.width_list, snr, arg, wl.threshold, raw_end_min=n_prev - lo, t_offset=lo,
                                     label=f"offsets rep {rep} push {i}")
                        maps[(rep, i)] = snr
        return maps

    incr = run([0, 1])
    monkeypatch.setenv("NSFRB_STREAM_STATS", "march")
    march = run([0], check=False)
    for (rep, i), snr in march.items():
        if i >= 1:
            assert np.all(np.abs(snr - incr[(rep, i)]) <= 2 * PU.tol(snr)), (rep, i)

def _scripted_stream(wl, chunks, eval_at, label, pixels=None, **check_kw):
    """Push `chunks` (device tensors [nchan][c][npix]) through one plan; at the pushes in eval_at compare with the oracle on
    the chronological ring contents (P-rule).  Returns {push: (snr, arg, oracle result)}."""
    nsfrb = _nsfrb()
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    out_maps = {}
    with nsfrb.Plan.for_workload(wl, cand_capacity=64) as plan:
        out = plan.alloc_outputs()
        hist, n = np.zeros((wl.nchan, 0, wl.npix), np.float32), 0
        for i, ch in enumerate(chunks):
            plan.stream_push(ch, out)
            n_prev, n = n, n + ch.shape[1]
            hist = np.concatenate([hist, ch.cpu().numpy()], axis=1)[:, -wl.nt:, :]
            if i in eval_at:
                torch.cuda.synchronize()
                lo = max(0, n - wl.nt)
                snr = out.snr_map.cpu().numpy()
                arg = out.argmax.cpu().numpy().T.copy()
                pix = np.arange(wl.npix) if pixels is None else np.asarray(pixels)
                st = PU.check(hist[:, :, pix], d, wl.width_list, snr[pix], arg[pix], wl.threshold, raw_end_min=n_prev - lo,
                              t_offset=lo, label=f"{label} push {i}", **check_kw)
                out_maps[i] = (snr, arg, st["oracle"])
    return out_maps


def _small_stream_plan():
    from dataclasses import replace
    return replace(W.config("c2").scaled(7, 5, nt=200), width_list=np.asarray([1, 3, 9, 30, 100, 180], np.int32))


def test_stream_statistics_survive_a_huge_sample_entering_and_leaving():
    """one 1e8 sample in one channel enters Sum D^2 (~1e16) and, a ring length later, leaves.  The
    float64 residue it would leave in the carried sums is removed: a leaving sample that dwarfs what stays marks the series
    and the sums are rebuilt from the ring (R31).  Pushes before, while it is inside every trial's valid set, and
    from the push at which it has left the ring must match the oracle.  (Push 10 is not compared: the sample has then left the
    valid sets of the high-DM trials but is still in the ring, and differential dedispersion -- each trial formed from its
    neighbour -- carries float32 rounding of the outlier, 6e-8 x 1e8, into them for that one push; R32.)"""
    wl = _small_stream_plan()
    g = torch.Generator(device="cuda").manual_seed(101)
    chunks = [torch.randn((wl.nchan, 25, wl.npix), device="cuda", generator=g) for _ in range(24)]
    chunks[3][2, 7, 5] = 1.0e8            # pixel 5, channel 2
    chunks[3][4, 9, 11] = -3.0e7          # and a negative one elsewhere
    # the sample entered at push 3 (absolute 82) leaves the 200-sample ring at push 11 (n = 300 > 82 + 200)
    _scripted_stream(wl, chunks, {2, 3, 4, 9, 11, 12, 13, 20, 23}, "huge sample")


def test_stream_first_sample_outlier_does_not_poison_the_baseline():
    """(ii): the very first sample is a 1e4 outlier in every channel of some pixels.  The stored reference level is the
    median of the first chunk (reading R32), not its first sample, so later ring values keep their float32 resolution."""
    wl = _small_stream_plan()
    g = torch.Generator(device="cuda").manual_seed(102)
    chunks = [torch.randn((wl.nchan, 25, wl.npix), device="cuda", generator=g) for _ in range(14)]
    chunks[0][:, 0, 3] = 1.0e4
    chunks[0][:, 0, 20] = -1.0e4
    chunks[0][1, 0, 8] = 5.0e3
    _scripted_stream(wl, chunks, {0, 1, 2, 7, 8, 9, 13}, "first-sample outlier")


def test_stream_non_finite_sample_stops_poisoning_once_it_has_left():
    """a NaN sample must not kill its (pixel, trial) series until nsfrb_stream_reset: once it has left the ring
    the sums are rebuilt and the pixel matches the oracle again (while it is inside, results are unspecified)."""
    wl = _small_stream_plan()
    g = torch.Generator(device="cuda").manual_seed(103)
    chunks = [torch.randn((wl.nchan, 25, wl.npix), device="cuda", generator=g) for _ in range(16)]
    chunks[2][3, 4, 9] = float("nan")     # absolute sample 54: gone once n > 254 + dmax, i.e. from push 10 on
    chunks[2][0, 5, 17] = float("inf")
    clean = [p for p in range(wl.npix) if p not in (9, 17)]
    _scripted_stream(wl, chunks, {3, 6}, "NaN inside (other pixels)", pixels=clean)
    _scripted_stream(wl, chunks, {11, 12, 15}, "NaN gone")


def test_stream_levels_far_from_the_baseline():
    """(iii): after the first chunk the level of every channel moves away from the stored baseline by `off` with unit
    noise.  off = 300 (noise 3e-3 of the level): full parity.  off = 1e5: the float32 ring and sums cannot carry 1e-4
    (documented limit, R32), but sigma must still be right -- the variance comes from the exact two-pass when
    Sum D^2 - (Sum D)^2 / T cancels (R31) -- so the S/N stays within a few per cent, far from the sigma = 0 of a floor."""
    wl = _small_stream_plan()
    g = torch.Generator(device="cuda").manual_seed(104)

    def make(off):
        out = []
        for i in range(13):
            x = torch.randn((wl.nchan, 25, wl.npix), device="cuda", generator=g)
            out.append(x + (off if i >= 1 else 0.0))
        return out
    _scripted_stream(wl, make(300.0), {1, 2, 8, 9, 12}, "level 300")
    nsfrb = _nsfrb()
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    chunks = make(1.0e5)
    with nsfrb.Plan.for_workload(wl, cand_capacity=64) as plan:
        out = plan.alloc_outputs()
        for ch in chunks:
            plan.stream_push(ch, out)
        torch.cuda.synchronize()
        snr = out.snr_map.cpu().numpy()
    hist = torch.cat(chunks, dim=1)[:, -wl.nt:, :].cpu().numpy()       # the level-0 chunk has left the ring
    r = oracle.search(hist, d, wl.width_list, raw_end_min=wl.nt - 25, t_offset=len(chunks) * 25 - wl.nt)
    assert np.all(np.isfinite(snr)) and np.all(snr > 1.0)
    assert np.all(np.abs(snr - r.snr) <= 0.08 * np.abs(r.snr)), float(np.max(np.abs(snr - r.snr) / np.abs(r.snr)))


def test_stream_five_thousand_pushes():
    """(iv): 5 000 pushes (625 laps of the ring) of irregular sizes on the 7 x 5 plan: the carried float64 sums do not drift."""
    wl = _small_stream_plan()
    g = torch.Generator(device="cuda").manual_seed(105)
    sizes = [25, 3, 25, 11, 40, 1]
    big = torch.randn((wl.nchan, 4096, wl.npix), device="cuda", generator=g)
    chunks, pos = [], 0
    for i in range(5000):
        c = sizes[i % len(sizes)]
        if pos + c > big.shape[1]:
            pos = (pos + 7) % 64
        chunks.append((big[:, pos:pos + c, :] + 0.01 * (i % 13)).contiguous())
        pos += c
    _scripted_stream(wl, chunks, {0, 1, 50, 999, 2500, 4998, 4999}, "5000 pushes")


def test_stream_running_sigma_trials_without_a_sample_on_the_first_pushes():
    """with chunks shorter than the largest delay some trials have no valid sample on the first pushes; their
    running variance must start at their first valid push (not from uninitialised memory), also after a reset."""
    nsfrb = _nsfrb()
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    assert int(d.max()) >= 6
    g = torch.Generator(device="cuda").manual_seed(106)
    alpha = 0.05
    with nsfrb.Plan.for_workload(wl, cand_capacity=64) as plan:
        out = plan.alloc_outputs()
        run = (torch.full((wl.npix,), 7.0, device="cuda"), torch.zeros((3, wl.npix), dtype=torch.int32, device="cuda"))
        plan.stream_set_running_sigma(alpha, *run)
        for rep in range(2):
            if rep:
                plan.stream_reset()
            ro = oracle.RunningStreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list, alpha)
            for i in range(12):
                chunk = torch.randn((wl.nchan, 3, wl.npix), device="cuda", generator=g) * (1.0 + i)
                plan.stream_push(chunk, out)
                torch.cuda.synchronize()
                res_run = ro.push(chunk.cpu().numpy())
                got = run[0].cpu().numpy()
                want = res_run.snr
                both = np.isfinite(want)
                assert np.array_equal(np.isneginf(got), np.isneginf(want)), (rep, i)
                assert np.all(np.abs(got[both] - want[both]) <= 2 * PU.tol(want[both])), (rep, i, float(np.max(np.abs(got[both] - want[both]))))


# ----------------------------------------------------------------------------- edge and degenerate cases
def test_degenerate_pixels_and_duplicate_unsorted_dms():
    from dataclasses import replace
    base = W.config("c1")
    # unsorted DM list with duplicates (exact ties must resolve to the lowest index, R17)
    dms = np.asarray([600.0, 0.0, 1400.0, 600.0, 200.0, 0.0, 1000.0, 3.0])
    wl = replace(base, nx=9, ny=7, nt=300, dm_list=dms, width_list=np.asarray([3, 1, 400, 17, 2], np.int32), name="edge")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    assert np.array_equal(d[7], d[1])  # DM 3 has the delay vector of DM 0
    rng = np.random.default_rng(3)
    a = rng.standard_normal((wl.nchan, wl.nt, wl.npix)).astype(np.float32)
    a[:, :, 0] = 0.0                      # all-zero pixel: sigma = 0 -> S = 0, argmax (first defined cell)
    a[:, :, 1] = 3.0                      # constant pixel
    a[:, :, 2] += 1000.0                  # large DC offset (invariance; per-channel baseline removal)
    a[:, :, 3] *= 1e-3                    # small scale
    a[:, :, 4] *= 1e3                     # large scale
    a[:, :, 5] = 0.0
    a[:, 100:103, 5] = 5.0                # noise-free zero-DM pulse of width 3: the zero-delay vector is at k=1, 5, 7
    cube = torch.from_numpy(a).cuda()
    st, cs, snr, arg = _offline(wl, cube)
    assert snr[0] == 0.0 and snr[1] == 0.0
    assert tuple(arg[0]) == tuple(st["oracle"].argmax[0]) and tuple(arg[1]) == tuple(st["oracle"].argmax[1])
    # closed form sqrt(T_k - w) at the matched cell; lowest index among the identical trials {1, 5, 7}
    assert tuple(arg[5]) == (1, 0, 100) and abs(snr[5] - np.sqrt(300 - 3)) < 2e-3


def test_no_cell_defined_and_single_channel():
    from dataclasses import replace
    nsfrb = _nsfrb()
    wl = replace(W.config("c1"), nx=5, ny=3, nt=40, width_list=np.asarray([41, 100], np.int32), name="nocell")
    cube = torch.randn((wl.nchan, wl.nt, wl.npix), device="cuda")
    with nsfrb.Plan.for_workload(wl) as plan:
        res = plan.search(cube)
        torch.cuda.synchronize()
        assert torch.all(torch.isneginf(res.snr_map)) and torch.all(res.argmax == -1) and res.n_found() == 0
    wl1 = replace(W.config("c1"), nx=6, ny=6, nchan=1, nt=77, freqs_GHz=np.asarray([1.4]), name="1chan")
    cube = torch.randn((1, 77, 36), device="cuda")
    _offline(wl1, cube)


def test_candidate_overflow_reports_total():
    from dataclasses import replace
    wl = replace(W.config("c1"), threshold=2.0, name="overflow")
    cube = W.make_cube(wl, "cuda")
    st, cs, snr, arg = _offline(wl, cube, capacity=7)
    assert cs["found"] > 7


def test_host_buffer_variants_match_device_path():
    nsfrb = _nsfrb()
    wl = W.config("c1")
    cube = W.make_cube(wl, "cpu").pin_memory()
    with nsfrb.Plan.for_workload(wl) as plan:
        h = plan.search_host(cube)
        dres = plan.search(cube.cuda())
        torch.cuda.synchronize()
        assert torch.equal(h[0], dres.snr_map.cpu()) and torch.equal(h[1], dres.argmax.cpu())
        assert int(h[3].numpy().view(np.uint32)[0]) == dres.n_found()
        hp = plan.stream_push_host(cube[:, :25, :].contiguous().pin_memory())
        plan.stream_reset()
        dp = plan.stream_push(cube[:, :25, :].contiguous().cuda())
        torch.cuda.synchronize()
        assert torch.equal(hp[0], dp.snr_map.cpu()) and torch.equal(hp[1], dp.argmax.cpu())


# ----------------------------------------------------------------------------- BASELINE sizes, sampled pixels
def _sample_pixels(wl, pulses, n_random, seed=7, extra=()):
    rng = np.random.default_rng(seed)
    pix = set(int(pu.pixel) for pu in pulses)
    pix |= {0, 1, 31, 32, wl.nx - 1, wl.nx, wl.npix - 1, wl.npix - wl.nx}          # image corners / row edges
    pix |= set(int(v) for v in extra if 0 <= int(v) < wl.npix)
    pix |= set(int(v) for v in rng.choice(wl.npix, n_random, replace=False))
    return np.asarray(sorted(pix))


def _report(label, st):
    """The P-rule's buckets ('report how many pixels fell into each bucket -- it should be a few %')."""
    defined = max(st["n"] - st["undefined"], 1)
    print(f"[parity] {label}: n={st['n']} exact={st['exact']} adjudicated={st['adjudicated']} "
          f"({100.0 * st['adjudicated'] / defined:.2f} %) undefined={st['undefined']} worst |d|/tol={st['worst_tol_frac']:.3f}")


@pytest.mark.parametrize("name,n_random", [("c3", 4096), ("c4", 4096), ("c5", 512)])
def test_full_size_sampled(name, n_random):
    """BASELINE.json sizes in the launch configuration bench.py times; the oracle checks every injected pixel, the image
    edges, the pixels on both sides of the layout kernel's 64-pixel tile edges and of the pixel-batch boundaries of the
    search, and n_random random pixels (>= 4096; C5 at 0.25 core-s per pixel: 512)."""
    import os
    nsfrb = _nsfrb()
    wl = W.config(name)
    need = wl.nchan * wl.nt * wl.npix * 4 + (8 << 30)
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip("not enough free device memory")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    cube = W.make_cube(wl, "cuda")
    pulses = _inject_all(wl, cube, d)
    # pixels around tile and batch edges: the batch holds about 1 GiB of [pixel][chan][time] workspace
    batch = max(8, ((1 << 30) // (wl.nchan * ((wl.nt + 3) // 4 * 4) * 4)) & ~7)
    edges = []
    for b in (64, batch):
        for k in (1, 2, 3, max(1, wl.npix // b - 1), wl.npix // b):
            edges += [k * b - 2, k * b - 1, k * b, k * b + 1]
    pix = _sample_pixels(wl, pulses, n_random, extra=edges)
    d_orc = d
    with nsfrb.Plan.for_workload(wl, cand_capacity=4096) as plan:
        assert np.array_equal(plan.delays(), d_orc)
        res = plan.search(cube)
        torch.cuda.synchronize()
        snr = res.snr_map.cpu().numpy()
        arg = res.argmax.cpu().numpy().T.copy()
        cands = res.candidates()
        nfound = res.n_found()
    sub = cube[:, :, torch.as_tensor(pix, device=cube.device)].cpu().numpy()
    del cube
    torch.cuda.empty_cache()
    st = PU.check(sub, d_orc, wl.width_list, snr[pix], arg[pix], wl.threshold, label=f"{name} full",
                  nthreads=os.cpu_count() or 8, max_adjudicated_frac=0.05)
    _report(f"{name} full size, {len(pix)} of {wl.npix} pixels ({len(pulses)} injected)", st)
    cs = PU.check_candidates(st["oracle"], pix, cands, nfound, wl.threshold, 4096, all_pixels_checked=False)
    for c in cands:
        p = int(c["pixel"])
        assert c["snr"] == snr[p] and (c["dm_idx"], c["width_idx"], c["t"]) == tuple(arg[p]) and c["snr"] > wl.threshold
    _check_recovery(wl, d, [pu for pu in pulses if pu.s0 >= 12], snr)
    # properties that hold at any size: finite map, indices in range, candidates = thresholded map
    assert np.all(np.isfinite(snr)) and arg[:, 0].min() >= 0 and arg[:, 0].max() < len(wl.dm_list)
    assert arg[:, 1].max() < len(wl.width_list) and arg[:, 2].min() >= 0 and arg[:, 2].max() < wl.nt
    assert cs["found"] == int((snr > wl.threshold).sum())


def test_full_size_stream_c2_sampled():
    """C2 at full size (256x256 px, 1536-sample ring): >= 256 pixels (every injected one, edges, random) on 11 pushes:
    the first ones, mid fill, the four around the ring wrap (1536 / 25 = 61.44) and steady state."""
    import os
    nsfrb = _nsfrb()
    wl = W.config("c2")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    n_push = 70
    src = W.ChunkSource(wl, d, n_push, "cuda")
    pix = _sample_pixels(wl, src.pulses, 256)
    tp = torch.as_tensor(pix, device="cuda")
    so = oracle.StreamOracle(wl.nchan, len(pix), wl.nt, d, wl.width_list)
    tot = {"n": 0, "exact": 0, "adjudicated": 0, "undefined": 0, "worst_tol_frac": 0.0}
    with nsfrb.Plan.for_workload(wl) as plan:
        out = plan.alloc_outputs()
        for i in range(n_push):
            chunk = src.next()
            plan.stream_push(chunk, out)
            ch = chunk[:, :, tp].cpu().numpy()
            n_prev = so.n
            so.n += ch.shape[1]
            so.hist = np.concatenate([so.hist, ch], axis=1)[:, -so.L:, :]
            if i in (0, 1, 20, 40, 60, 61, 62, 63, 65, 68, 69):
                torch.cuda.synchronize()
                lo = max(0, so.n - so.L)
                snr = out.snr_map.cpu().numpy()
                arg = out.argmax.cpu().numpy().T.copy()
                st = PU.check(so.hist, d, wl.width_list, snr[pix], arg[pix], wl.threshold, raw_end_min=n_prev - lo,
                              t_offset=lo, label=f"c2 full push {i}", nthreads=os.cpu_count() or 8,
                              max_adjudicated_frac=0.05 if i >= 20 else 0.25)
                for k in ("n", "exact", "adjudicated", "undefined"):
                    tot[k] += st[k]
                tot["worst_tol_frac"] = max(tot["worst_tol_frac"], st["worst_tol_frac"])
                PU.check_candidates(st["oracle"], pix, out.candidates(), out.n_found(), wl.threshold, 4096,
                                    all_pixels_checked=False)
                assert out.n_found() == int((snr > wl.threshold).sum())
    _report(f"c2 full size, {len(pix)} pixels x 11 pushes", tot)
    assert tot["adjudicated"] <= 0.05 * max(tot["n"] - tot["undefined"], 1)


def test_stream_unsorted_duplicate_dms_and_flat_pixels():
    """Real-time path on an awkward plan: unsorted DM list with duplicates (5 unique trials: the last DM group
    of k_stream is padded), unsorted widths incl. one longer than the ring, 35 pixels (neither a multiple of
    32 nor of 4), a constant pixel (sigma = 0 => S = 0) and chunks larger than the first one (several passes)."""
    from dataclasses import replace
    dms = np.asarray([600.0, 0.0, 1400.0, 600.0, 200.0, 0.0, 1000.0], dtype=np.float64)
    wl = replace(W.config("c1"), nx=7, ny=5, nt=120, dm_list=dms, streaming=True, threshold=4.0,
                 width_list=np.asarray([3, 1, 400, 17, 2, 64], np.int32), name="stream-edge")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    nsfrb = _nsfrb()
    g = torch.Generator(device="cuda").manual_seed(11)
    so = oracle.StreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list)
    with nsfrb.Plan.for_workload(wl, cand_capacity=64) as plan:
        out = plan.alloc_outputs()
        for i, c in enumerate([4, 9, 30, 1, 120, 17, 33, 5]):
            chunk = torch.randn((wl.nchan, c, wl.npix), device="cuda", generator=g)
            chunk[:, :, 3] = 2.5          # constant pixel: sigma = 0 for every trial
            chunk[:, :, 20] *= 1e-3       # tiny scale: S/N is scale-free
            plan.stream_push(chunk, out)
            torch.cuda.synchronize()
            ch = chunk.cpu().numpy()
            n_prev = so.n
            so.n += c
            so.hist = np.concatenate([so.hist, ch], axis=1)[:, -so.L:, :]
            lo = max(0, so.n - so.L)
            snr = out.snr_map.cpu().numpy()
            arg = out.argmax.cpu().numpy().T.copy()
            st = PU.check(so.hist, d, wl.width_list, snr, arg, wl.threshold, raw_end_min=n_prev - lo, t_offset=lo,
                          label=f"stream-edge push {i}", max_adjudicated_frac=0.5)
            PU.check_candidates(st["oracle"], np.arange(wl.npix), out.candidates(), out.n_found(), wl.threshold, 64)
            if so.n > int(d.max()) + 1:
                assert snr[3] == 0.0


# ----------------------------------------------------------------------------- NEXT 2: binned timescales
@pytest.mark.parametrize("npix", [37, 64])
def test_bin_time_matches_oracle(npix):
    nsfrb = _nsfrb()
    g = torch.Generator(device="cuda").manual_seed(21)
    ints = torch.randint(-8, 9, (3, 301, npix), device="cuda", generator=g).float()   # exact in float32
    gauss = torch.randn((3, 301, npix), device="cuda", generator=g)
    for factor in (1, 5, 7, 75, 301, 400):
        got = nsfrb.bin_time(ints, factor)
        torch.cuda.synchronize()
        assert np.array_equal(got.cpu().numpy(), oracle.bin_time(ints.cpu().numpy(), factor)), factor
        got = nsfrb.bin_time(gauss, factor).cpu().numpy()
        ref = oracle.bin_time(gauss.cpu().numpy(), factor)
        assert got.shape == ref.shape and np.all(np.abs(got - ref) <= 1e-6 * factor * 4), factor
    with pytest.raises(nsfrb.NsfrbError):
        nsfrb.bin_time(ints, 0)


def test_three_timescale_search_paper_grid():
    """The search as the paper runs it: 16 DM trials x log2 widths 1..16 at the native sampling,
    again on the x5-binned stack with 5x the DMs (same shift table, fn. 12), and widths only (DM 0) on the x75-binned
    stack -- each leg compared with the oracle on the oracle-binned cube."""
    from dataclasses import replace
    nsfrb = _nsfrb()
    base = replace(W.config("c2").scaled(8, 6, nt=3000), streaming=False, width_list=np.asarray([1, 2, 4, 8, 16], np.int32),
                   dm_list=np.linspace(171.0, 4000.0, 16), threshold=6.0, name="paper-grid")
    g = torch.Generator(device="cuda").manual_seed(31)
    cube = torch.randn((base.nchan, base.nt, base.npix), device="cuda", generator=g)
    cube[:, 1500:1500 + 40, 7] += 0.6            # a 5.4 s pulse at DM 0: best seen at the 0.67 s timescale
    cube[:, 600:600 + 900, 20] += 0.15           # a 2 min pulse (in a 40-bin x75 series it inflates its own sigma, L130)
    d1 = oracle.delays(base.freqs_GHz, base.tsamp_s, base.dm_list)
    best = {}
    for factor, dms in ((1, base.dm_list), (5, 5 * base.dm_list), (75, np.asarray([0.0]))):
        wl = replace(base, nt=base.nt // factor, tsamp_s=base.tsamp_s * factor, dm_list=dms, name=f"paper-grid x{factor}")
        d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
        if factor == 5:
            assert np.array_equal(d, d1)         # footnote 12: the same shift table
        binned = nsfrb.bin_time(cube, factor) if factor > 1 else cube
        ref_binned = oracle.bin_time(cube.cpu().numpy(), factor)
        assert np.all(np.abs(binned.cpu().numpy() - ref_binned) <= 1e-5 * factor)
        st, cs, snr, arg = _offline(wl, binned.contiguous(), label=wl.name)
        best[factor] = snr
    # the 40-sample pulse exceeds the 16-sample native boxcars: the x5 leg recovers more of it (L77)
    assert best[5][7] > best[1][7]


def test_two_plans_with_different_shared_memory_needs_coexist():
    """The opt-in shared-memory size is a per-function attribute: creating a second, smaller plan must not break
    launches of the first (regression: 'k_search launch: invalid argument')."""
    nsfrb = _nsfrb()
    big = W.config("c3").scaled(6, 4, nt=600, n_pulses=0)
    small = W.config("c1")
    cube = W.make_cube(big, "cuda")
    with nsfrb.Plan.for_workload(big) as p1:
        with nsfrb.Plan(small.nx, small.ny, small.nchan, small.nt, small.freqs_GHz, small.tsamp_s, [500.0], [1], 6.0) as p2:
            p2.search(W.make_cube(small, "cuda"))
        r = p1.search(cube)
        torch.cuda.synchronize()
        assert np.isfinite(r.snr_map.cpu().numpy()).all()


def test_more_than_32_widths_use_the_generic_kernel():
    """Plans with more than 32 usable widths run the generic k_search (two width batches); everything else runs
    the plan-specialised k_search4 -- both against the oracle, and against each other on the same cube."""
    from dataclasses import replace
    nsfrb = _nsfrb()
    wl40 = replace(W.config("c1"), nx=6, ny=5, nt=700, width_list=np.arange(1, 41, dtype=np.int32) * 3 - 2, name="w40")
    d = oracle.delays(wl40.freqs_GHz, wl40.tsamp_s, wl40.dm_list)
    g = torch.Generator(device="cuda").manual_seed(41)
    cube = torch.randn((wl40.nchan, wl40.nt, wl40.npix), device="cuda", generator=g)
    st, cs, snr40, arg40 = _offline(wl40, cube, label="w40 generic")
    # the first 32 of those widths through k_search4, then the maxima restricted to them must agree where they win
    wl32 = replace(wl40, width_list=wl40.width_list[:32], name="w32")
    st, cs, snr32, arg32 = _offline(wl32, cube, label="w32 specialised")
    same = arg40[:, 1] < 32
    assert same.any() and np.all(np.abs(snr40[same] - snr32[same]) <= PU.tol(snr40[same]))


def test_stream_64_channels():
    """Real-time path on a 64-channel plan (config-5 band and DM spacing, 24 trials): the kernel is compiled with
    one time step per tile; pushes compared with the oracle while the ring fills and after it wraps."""
    wl = W.config("c5")
    from dataclasses import replace
    wl = replace(wl, nx=8, ny=5, nt=400, dm_list=np.linspace(0.0, 5000.0, 256)[:24], streaming=True, chunk_nt=25,
                 width_list=np.asarray([1, 2, 3, 5, 8, 13, 21, 55, 144, 300], np.int32), name="c5-stream")
    _stream_case(wl, 20, eval_at={0, 1, 5, 15, 16, 17, 19}, cubes=True)   # 24 trials: two supergroups of CTAs


# ----------------------------------------------------------------------------- NEXT 3: S/N and TOA cubes (L94)
def test_stream_cubes_match_oracle():
    """nsfrb_stream_set_cubes: per-(dm, width, pixel) peak S/N and window start of every push against the oracle's
    per-(k, j) maxima (details=True), incl. duplicate DMs (planes repeated), a width longer than the ring (-inf, -1),
    the filling ring (widths without a window yet) and chunks longer than the first one (several passes)."""
    from dataclasses import replace
    nsfrb = _nsfrb()
    dms = np.asarray([0.0, 300.0, 300.0, 900.0, 1400.0, 0.0], dtype=np.float64)
    wl = replace(W.config("c1"), nx=8, ny=5, nt=160, dm_list=dms, streaming=True, threshold=5.0,
                 width_list=np.asarray([2, 1, 500, 9, 40], np.int32), name="cubes")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    g = torch.Generator(device="cuda").manual_seed(51)
    so = oracle.StreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list)
    snr_cube = torch.zeros((len(dms), len(wl.width_list), wl.npix), device="cuda")
    toa_cube = torch.zeros((len(dms), len(wl.width_list), wl.npix), dtype=torch.int32, device="cuda")
    with nsfrb.Plan.for_workload(wl, cand_capacity=64) as plan:
        plan.stream_set_cubes(snr_cube, toa_cube)
        out = plan.alloc_outputs()
        for i, c in enumerate([10, 3, 25, 60, 160, 7, 12]):
            chunk = torch.randn((wl.nchan, c, wl.npix), device="cuda", generator=g)
            plan.stream_push(chunk, out)
            torch.cuda.synchronize()
            n_prev = so.n
            so.n += c
            so.hist = np.concatenate([so.hist, chunk.cpu().numpy()], axis=1)[:, -so.L:, :]
            lo = max(0, so.n - so.L)
            r = oracle.search(so.hist, d, wl.width_list, raw_end_min=n_prev - lo, t_offset=lo, details=True)
            S = snr_cube.cpu().numpy().transpose(2, 0, 1)      # [npix][ndm][nw]
            Tm = toa_cube.cpu().numpy().transpose(2, 0, 1)
            undefined = np.isneginf(r.best)
            assert np.array_equal(np.isneginf(S), undefined), f"push {i}: defined sets differ"
            assert np.all(Tm[undefined] == -1)
            ok = ~undefined
            assert np.all(np.abs(S[ok] - r.best[ok]) <= PU.tol(r.best[ok])), f"push {i}"
            assert np.all(S[:, :, 2] == -np.inf)               # width 500 never fits the 160-sample ring
            assert np.array_equal(S[:, 2], S[:, 1]) and np.array_equal(Tm[:, 2], Tm[:, 1])   # duplicate DM planes
            assert np.array_equal(S[:, 5], S[:, 0])
            # window starts: identical, or the oracle rates the GPU's window within tolerance of the maximum
            diff = np.argwhere(ok & (Tm != r.best_t))
            assert len(diff) <= 0.1 * ok.sum()
            for p, k, j in diff:
                s_at = oracle.snr_at(so.hist, d, wl.width_list, p, k, j, int(Tm[p, k, j]), raw_end_min=n_prev - lo, t_offset=lo)
                assert s_at >= r.best[p, k, j] - 2 * PU.tol(r.best[p, k, j]), (i, p, k, j)
            # the maps are the maxima of the cubes
            assert np.allclose(out.snr_map.cpu().numpy(), S.reshape(wl.npix, -1).max(axis=1), rtol=0, atol=0)
        plan.stream_set_cubes(None, None)
        plan.stream_push(torch.randn((wl.nchan, 5, wl.npix), device="cuda", generator=g), out)
        torch.cuda.synchronize()


def test_pipelined_host_pushes_equal_device_pushes():
    """nsfrb_stream_push_host_async (copy of chunk i+1 overlapping the search of chunk i, two pushes in flight) must
    deliver, for every push, exactly what nsfrb_stream_push delivers for the same chunks on a second plan; the last
    push is also checked against the oracle."""
    nsfrb = _nsfrb()
    wl = W.config("c1")
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    n_push = 7
    src = W.ChunkSource(wl, d, n_push, "cuda")
    chunks = [src.next().clone() for _ in range(n_push)]
    host = [c.cpu().pin_memory() for c in chunks]
    so = oracle.StreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list)
    with nsfrb.Plan.for_workload(wl, cand_capacity=64) as pa, nsfrb.Plan.for_workload(wl, cand_capacity=64) as pb:
        outs = [pa._host_out() for _ in range(n_push)]
        for i in range(n_push):                       # all enqueued back to back; the third call waits for the first
            pa.stream_push_host_async(host[i], outs[i])
        pa.stream_wait()
        ref = pb.alloc_outputs()
        for i in range(n_push):
            pb.stream_push(chunks[i], ref)
            torch.cuda.synchronize()
            ores = so.push(chunks[i].cpu().numpy(), nthreads=8)
            assert np.array_equal(outs[i][0].numpy(), ref.snr_map.cpu().numpy()), i
            assert np.array_equal(outs[i][1].numpy(), ref.argmax.cpu().numpy()), i
            n = int(outs[i][3].numpy().view(np.uint32)[0])
            assert n == ref.n_found()
            got = outs[i][2].numpy()[: n * nsfrb.CAND_DTYPE.itemsize].view(nsfrb.CAND_DTYPE)
            assert sorted(map(tuple, got)) == sorted(map(tuple, ref.candidates()))
        snr = outs[-1][0].numpy()
        assert np.all(np.abs(snr - ores.snr) <= 1e-4 + 1e-4 * np.abs(ores.snr))
        # the synchronous calls still work on the same plan after a wait, and reset waits for pushes in flight
        pa.stream_push_host_async(host[0], outs[0])
        pa.stream_reset()
        o = pa.stream_push_host(host[0])
        pb.stream_reset()
        pb.stream_push(chunks[0], ref)
        torch.cuda.synchronize()
        assert np.array_equal(o[0].numpy(), ref.snr_map.cpu().numpy())


def _check_running(wl, d, out_snr, out_arg, ores, inst, var, label):
    """Running-sigma maps vs RunningStreamOracle: S/N within tol; arg-max exact where the oracle's winner beats every
    other (trial, width) maximum by more than 2 tol, otherwise the GPU's cell is adjudicated by the oracle:
    S_run(cell) = snr_at(cell) * sigma_inst / sigma_run must be within 2 tol of the oracle's maximum."""
    snr = out_snr.cpu().numpy()
    arg = out_arg.cpu().numpy().T
    tol = 1e-4 + 1e-4 * np.abs(ores.snr)
    defined = ores.argmax[:, 0] >= 0
    assert np.array_equal(arg[:, 0] >= 0, defined), label
    assert np.all(np.isneginf(snr[~defined]))
    assert np.all(np.abs(snr[defined] - ores.snr[defined]) <= tol[defined]), label
    flat = np.sort(ores.best.reshape(ores.best.shape[0], -1), axis=1)
    margin = flat[:, -1] - flat[:, -2]
    adjudicated = 0
    for p in np.nonzero(defined)[0]:
        if tuple(arg[p]) == tuple(ores.argmax[p]):
            continue
        assert margin[p] <= 2 * tol[p] or arg[p, 0] == ores.argmax[p, 0] and arg[p, 1] == ores.argmax[p, 1], (label, p)
        k, j, t = (int(x) for x in arg[p])
        s_inst = oracle.snr_at(inst["hist"], d, wl.width_list, p, k, j, t, raw_end_min=inst["raw_end_min"], t_offset=inst["lo"])
        s_run = s_inst * inst["sigma"][p, k] / np.sqrt(var[p, k])
        assert abs(s_run - ores.snr[p]) <= 2 * tol[p], (label, p)
        adjudicated += 1
    return adjudicated


@pytest.mark.parametrize("alpha,own_cubes,dup", [(0.1, False, False), (0.5, True, False), (1.0, False, True)])
def test_stream_running_sigma_matches_oracle(alpha, own_cubes, dup):
    from dataclasses import replace
    nsfrb = _nsfrb()
    wl = W.config("c1")
    if dup:
        wl = replace(wl, dm_list=np.asarray([400.0, 0.0, 400.0, 1000.0, 0.0, 1400.0]))
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    n_push = 6
    src = W.ChunkSource(wl, d, n_push, "cuda")
    so = oracle.RunningStreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list, alpha)
    plain = oracle.StreamOracle(wl.nchan, wl.npix, wl.nt, d, wl.width_list)
    total_adj = 0
    with nsfrb.Plan.for_workload(wl) as plan:
        out = plan.alloc_outputs()
        rs = torch.zeros(wl.npix, device="cuda")
        ra = torch.zeros((3, wl.npix), dtype=torch.int32, device="cuda")
        if own_cubes:
            shape = (len(wl.dm_list), len(wl.width_list), wl.npix)
            cs, ct = torch.zeros(shape, device="cuda"), torch.zeros(shape, dtype=torch.int32, device="cuda")
            plan.stream_set_cubes(cs, ct)
        plan.stream_set_running_sigma(alpha, rs, ra)
        for i in range(n_push):
            chunk = src.next()
            if i == 4:
                chunk[:, 3:19, 77] += 2.5          # a wide bright pulse: this push's own sigma is inflated (L130)
            plan.stream_push(chunk, out)
            torch.cuda.synchronize()
            ch = chunk.cpu().numpy()
            n_prev = so.n
            ores = so.push(ch, nthreads=8)
            pres = plain.push(ch, nthreads=8, details=True)
            lo = max(0, so.n - so.L)
            inst = dict(hist=so.hist, raw_end_min=n_prev - lo, lo=lo, sigma=pres.sigma)
            total_adj += _check_running(wl, d, rs, ra, ores, inst, so.var, f"push {i}")
            # the plain outputs of the same push are untouched by the mode
            PU.check(so.hist, d, wl.width_list, out.snr_map.cpu().numpy(), out.argmax.cpu().numpy().T.copy(), wl.threshold,
                     raw_end_min=n_prev - lo, t_offset=lo, label=f"plain push {i}")
            if alpha == 1.0:
                assert np.allclose(rs.cpu().numpy(), out.snr_map.cpu().numpy(), rtol=1e-6, atol=1e-6, equal_nan=True)
            if i == 4 and alpha < 1.0:
                assert rs[77].item() > 1.1 * out.snr_map[77].item()      # the bias is (partly) removed
        assert total_adj <= 0.05 * n_push * wl.npix
        # reset restarts the running variance: the first push after it equals the plain maps again
        plan.stream_reset()
        plan.stream_push(src.next(), out)
        torch.cuda.synchronize()
        assert np.allclose(rs.cpu().numpy(), out.snr_map.cpu().numpy(), rtol=1e-6, atol=1e-6, equal_nan=True)
        # switching the mode off stops the writes
        plan.stream_set_running_sigma(0.0, None, None)
        rs.fill_(123.0)
        plan.stream_push(src.next(), out)
        torch.cuda.synchronize()
        assert float(rs.min()) == 123.0
