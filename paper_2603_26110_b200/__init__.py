"""B200-native TurboESM hot path (arxiv/paper_2603_26110): 3-bit KV quantize/pack + fused decode attention.

The product is the C-ABI library `libtq.so` (include/tq.h; CUDA kernels under csrc/) and the thin ctypes
binding in `binding.py`.  Importing this package does not load the library; the first call into
`binding` does, and fails loudly if the CUDA extension has not been built (there is no CPU fallback).
`workloads.py` only draws seeded synthetic inputs.
"""
__all__ = ["binding", "workloads", "build"]
