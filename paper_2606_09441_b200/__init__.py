"""B200-native SIFT hot path (arxiv/paper_2606_09441): metadata decode + block-sparse prefill attention.

`workload` (seeded inputs) imports no CUDA code; `api` is the ctypes binding of the C-ABI library
built from `csrc/` and fails loudly if that library is missing.
"""
__version__ = "0.1.0"
