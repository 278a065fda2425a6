"""-m gpu, collected last: nsfrb_cluster_static (the no-allocation variant of nsfrb_cluster, workspace in a file-scope
__device__ array) against the existing nsfrb_cluster path, on two calls in a row that share the static workspace."""
import numpy as np
import pytest
import torch

from paper_2510_18136_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _same(a: dict, b: dict):
    # the existing cluster tests compare exactly (indices bit for bit, float64 means bit for bit): so does this one
    assert a["pixels"] == b["pixels"] and a["members"] == b["members"] and a["best"] == b["best"]
    assert np.array_equal(a["cands"], b["cands"])
    assert a["wsnr"] == b["wsnr"]


def test_cluster_static_matches_cluster_on_two_calls_in_a_row():
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    nx, ny, thr, topn = 301, 301, 6.0, 10          # 90 601 pixels: 45 CTAs, a ragged last slice
    psf = W.synthetic_psf(41, 0)
    maps = [W.synthetic_snr_map(nx, ny, psf, seed)[0].astype(np.float32) for seed in (0, 1)]
    maps[1][maps[1] > 9.0] = 5.0                    # second call: fewer candidates than the first one left in the scratch
    g = torch.Generator().manual_seed(3)
    arg = torch.randint(0, 16, (3, nx * ny), generator=g, dtype=torch.int32).cuda()
    dpsf = torch.from_numpy(psf).cuda()
    dmask, _ = nsfrb.psf_mask(dpsf, 90.0)
    with nsfrb.Plan(nx, ny, 2, 64, [1.3, 1.5], W.TSAMP_S, [0.0], [1], thr) as plan:
        want = [plan.cluster(torch.from_numpy(m.ravel().copy()).cuda(), arg, dpsf, dmask, topn).to_host() for m in maps]
    dmaps = [torch.from_numpy(m.ravel().copy()).cuda() for m in maps]
    out = nsfrb.alloc_cluster_result(topn)
    torch.cuda.synchronize()
    got = []
    for dm in dmaps:                                 # two calls in a row, same stream, same output buffers
        nsfrb.cluster_static(dm, arg, nx, ny, thr, dpsf, dmask, topn, out=out)
        got.append(out.to_host())
    assert len(want[0]["pixels"]) == topn and 0 < len(want[1]["pixels"]) <= topn
    for a, b in zip(got, want):
        _same(a, b)
    # a third call on the first map again: nothing of the second call survives in the shared workspace
    _same(nsfrb.cluster_static(dmaps[0], arg, nx, ny, thr, dpsf, dmask, topn, out=out).to_host(), want[0])
    # no candidate at all
    empty = nsfrb.cluster_static(dmaps[0], arg, nx, ny, 1e9, dpsf, dmask, topn, out=out).to_host()
    assert empty["pixels"] == [] and empty["best"] == -1


def test_cluster_static_rejects_sizes_beyond_its_workspace():
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    psf = torch.ones((3, 3), device="cuda")
    mask = torch.ones((3, 3), dtype=torch.uint8, device="cuda")
    snr = torch.zeros(64, device="cuda")
    arg = torch.zeros((3, 64), dtype=torch.int32, device="cuda")
    with pytest.raises(nsfrb.NsfrbError) as ei:      # 4097 x 4096 pixels > 2^24 (rejected before any pointer is touched)
        nsfrb.cluster_static(snr, arg, 4097, 4096, 6.0, psf, mask, 10)
    assert ei.value.code == nsfrb.NSFRB_EINVAL and "limit" in str(ei.value)
    with pytest.raises(nsfrb.NsfrbError) as ei:
        nsfrb.cluster_static(snr, arg, 8, 8, 6.0, psf, mask, 33, out=nsfrb.alloc_cluster_result(33))
    assert ei.value.code == nsfrb.NSFRB_EINVAL and "topn" in str(ei.value)
