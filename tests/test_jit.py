"""CPU tests of the plan-time specialisation of the real-time kernel (no GPU: NVRTC only cross-compiles)."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from paper_2510_18136_b200 import nsfrb, workloads as W


def _args(wl):
    return (wl.nx, wl.ny, wl.nchan, wl.nt, wl.freqs_GHz, wl.tsamp_s, wl.dm_list, wl.width_list)


def test_generated_source_carries_the_plan():
    wl = W.config("c2")
    src = nsfrb.jit_stream_kernel(*_args(wl), 25).decode()
    assert "#define NPIX 65536" in src and "#define NCHAN 16" in src and "#define NU 16" in src and "#define CMAX 25" in src
    # widths ascending, as the library was given them (tests/golden/width_lists.txt, n = 20)
    assert "W_TAB[NW] = {1,2,3,4,5,6,9,14,20,29,42,61,88,128,186,270,392,569,826,1200}" in src
    # delay rows of the table the plan computes (tests/golden/c2_dmax.txt pins their maxima)
    assert "DMAX_TAB[NU] = {0,1,1,2,3,4,4,5,6,6,7,8,8,9,10,11}" in src
    assert 'extern "C" __global__' in src and "k_stream" in src


def test_duplicate_trials_and_unused_widths_are_dropped_from_the_kernel():
    wl = W.config("c1")
    dms = np.asarray([600.0, 0.0, 600.0, 3.0])          # DM 3 has the delay vector of DM 0
    src = nsfrb.jit_stream_kernel(wl.nx, wl.ny, wl.nchan, 64, wl.freqs_GHz, wl.tsamp_s, dms, [5, 1, 400], 8).decode()
    assert "#define NU 2" in src and "K_OF_U[NU] = {1,0}" in src      # unique trials, ascending delay
    assert "W_TAB[NW] = {1,5}" in src and "J_OF_W[NW] = {1,0}" in src  # width 400 > ring: no cell, not compiled in


def test_default_shape_and_modes_are_in_the_prologue(monkeypatch):
    """Default: incremental statistics + dedispersed history with 8-row block sums, 4 trials x 4 groups per CTA, one time segment,
    six steps per tile.  NSFRB_STREAM_DHIST=0 gives the raw-ring march (light tiles, three steps per tile),
    NSFRB_STREAM_STATS=march the whole-ring march with the v4 shape; the raw march above 24 channels takes one step per tile."""
    wl = W.config("c2")
    src = nsfrb.jit_stream_kernel(*_args(wl), 25).decode()
    for d in ("#define INCR 1", "#define LIGHT 1", "#define DHIST 1", "#define COARSE 1", "#define SEG 1", "#define TT 6", "#define KK 4",
              "#define GPC 4", "#define PFD 2", "#define LRING 1536"):
        assert d in src, d
    assert "k_stream_stats" in src
    src = nsfrb.jit_stream_kernel(wl.nx, wl.ny, wl.nchan, 1532, wl.freqs_GHz, wl.tsamp_s, wl.dm_list, wl.width_list, 25).decode()
    assert "#define DHIST 1" in src and "#define COARSE 0" in src          # block sums need a ring length that is a multiple of 8
    monkeypatch.setenv("NSFRB_STREAM_DHIST", "0")
    src = nsfrb.jit_stream_kernel(*_args(wl), 25).decode()
    for d in ("#define INCR 1", "#define LIGHT 1", "#define DHIST 0", "#define COARSE 0", "#define SEG 1", "#define TT 3", "#define KK 8",
              "#define GPC 2", "#define PFD 4"):
        assert d in src, d
    monkeypatch.setenv("NSFRB_STREAM_LIGHT", "0")
    src = nsfrb.jit_stream_kernel(*_args(wl), 25).decode()
    assert "#define INCR 1" in src and "#define LIGHT 0" in src and "#define SEG 2" in src
    monkeypatch.delenv("NSFRB_STREAM_LIGHT")
    wl5 = W.config("c5")
    src = nsfrb.jit_stream_kernel(wl5.nx, wl5.ny, wl5.nchan, 1536, wl5.freqs_GHz, wl5.tsamp_s, wl5.dm_list[:16], wl5.width_list, 25).decode()
    assert "#define NCHAN 64" in src and "#define TT 1" in src and "#define SEG 2" in src
    monkeypatch.delenv("NSFRB_STREAM_DHIST")
    monkeypatch.setenv("NSFRB_STREAM_STATS", "march")
    src = nsfrb.jit_stream_kernel(*_args(wl), 25).decode()
    for d in ("#define INCR 0", "#define LIGHT 0", "#define DHIST 0", "#define SEG 2", "#define TT 2"):
        assert d in src, d


def test_bad_variant_is_rejected():
    wl = W.config("c1")
    with pytest.raises(nsfrb.NsfrbError):
        nsfrb.jit_stream_kernel(*_args(wl), 25, variant="zebra")


def test_kernel_cross_compiles_to_sm100a():
    wl = W.config("c1")
    cubin = nsfrb.jit_stream_kernel(*_args(wl), 25, cubin=True)
    assert cubin[:4] == b"\x7fELF"
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    path = os.path.join(os.environ.get("TMPDIR", "/tmp"), f"nsfrb_k_stream_{os.getpid()}.cubin")
    with open(path, "wb") as f:
        f.write(cubin)
    try:
        out = subprocess.run([cuobjdump, "-res-usage", path], capture_output=True, text=True).stdout
        assert "Function k_stream:" in out
        assert "Function k_stream_stats:" in out      # the incremental statistics live in the same module
        assert " LOCAL:0" in out.split("Function k_stream:")[1].splitlines()[1]   # no register array fell to local memory
        elf = subprocess.run([cuobjdump, "-elf", path], capture_output=True, text=True).stdout
        assert "sm_100a" in elf or "SM100a" in elf or "EF_CUDA_SM100" in elf, elf[:400]
    finally:
        os.remove(path)


def test_offline_kernel_source_and_cubin():
    """k_search4 (plan-specialised offline kernel): the source carries the plan, NVRTC cross-compiles it."""
    wl = W.config("c3")
    src = nsfrb.jit_search_kernel(*_args(wl)).decode()
    assert "#define NCHAN 16" in src and "#define NU 32" in src and "#define NW 24" in src and "#define NT 4096" in src
    assert "W_TAB[NW] = {1,2,3,4,5,6,7,9,12,16,22,30,40,55,75,102,139,189,257,350,476,648,882,1200}" in src
    assert 'extern "C" __global__' in src and "k_search4" in src
    cubin = nsfrb.jit_search_kernel(*_args(W.config("c1")), cubin=True)
    assert cubin[:4] == b"\x7fELF"
    with pytest.raises(nsfrb.NsfrbError):      # more than 32 usable widths: the generic kernel serves those plans
        nsfrb.jit_search_kernel(4, 4, 8, 512, W.config("c1").freqs_GHz, 0.1342, [0.0], list(range(1, 41)))
