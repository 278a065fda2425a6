"""Builds libnsfrb.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2510_18136_b200.build [--force]

The .so is git-ignored but travels to the GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnsfrb.so")
SOURCES = ["nsfrb_api.cu", "nsfrb_kernels.cu", "nsfrb_search.cu", "nsfrb_stream.cu", "nsfrb_offline.cu", "nsfrb_cluster.cu", "nsfrb_median.cu", "nsfrb_peaks.cu", "nsfrb_imaging.cu"]
JIT_SRCS = [os.path.join(CSRC, "nsfrb_stream_kernel.cuh"),   # compiled at plan time (NVRTC); embedded as text
            os.path.join(CSRC, "nsfrb_search_kernel.cuh")]
HEADERS = JIT_SRCS + [os.path.join(CSRC, "nsfrb_internal.h"), os.path.join(os.path.dirname(HERE), "include", "nsfrb.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-cudart", "static",
    "-lnvrtc", "-Xlinker", "-rpath=/usr/local/cuda/lib64",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        for src_path in JIT_SRCS:   # each kernel source as one raw string literal
            with open(src_path) as f:
                text = f.read()
            assert ')NSFRBSRC"' not in text
            with open(src_path[:-len(".cuh")] + "_src.inc", "w") as f:
                f.write('R"NSFRBSRC(\n' + text + ')NSFRBSRC"\n')
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [_nvcc(), *NVCC_FLAGS] + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
