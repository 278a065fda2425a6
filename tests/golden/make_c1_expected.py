"""Writes c1_oracle_expected.txt from the oracle alone (never from the CUDA path)."""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle  # noqa: E402
from paper_2510_18136_b200 import workloads as W  # noqa: E402

wl = W.config("c1")
d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
cube = W.make_cube(wl)
W.inject(cube, W.injection_table(wl, d), d, extra_delays=oracle.delays(wl.freqs_GHz, wl.tsamp_s, [500.0])[0])
r = oracle.search(cube.numpy(), d, wl.width_list)
p = 20 * wl.nx + 11
with open(os.path.join(HERE, "c1_oracle_expected.txt"), "w") as f:
    f.write("# oracle on BASELINE.json config 1 (make_c1_expected.py); SURVEY.md 8(c) quotes 5.728 (0,2,31), 0 cands\n")
    f.write(f"pulse_pixel {p} snr {r.snr[p]:.12f} argmax {r.argmax[p,0]} {r.argmax[p,1]} {r.argmax[p,2]}\n")
    f.write(f"map_max_pixel {int(r.snr.argmax())} ncands_thr6 {len(r.candidates(6.0))} ncands_thr5 {len(r.candidates(5.0))}\n")
