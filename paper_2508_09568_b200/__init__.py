"""paper_2508_09568_b200 -- B200-native per-bunch ideal-MHD update (arxiv 2508.09568).

`workloads` (numpy only) is importable without CUDA; `binding` loads the C-ABI library
libmhd_bunch.so (hand-written sm_100a kernels) and fails loudly if it is missing.
"""
__all__ = ["workloads", "binding"]
