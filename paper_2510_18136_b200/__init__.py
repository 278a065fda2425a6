"""B200-native NSFRB image-plane single-pulse search (arxiv 2510.18136 search stage).

`paper_2510_18136_b200.nsfrb` is the thin ctypes binding over the C-ABI library
(csrc/ -> libnsfrb.so); it raises if the CUDA library is missing -- there is no CPU
fallback.  `paper_2510_18136_b200.workloads` holds the seeded synthetic inputs.
"""
__all__ = ["nsfrb", "workloads"]
