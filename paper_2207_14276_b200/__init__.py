"""B200-native ANI-2x-style potential (Deep-HP hot path, arXiv 2207.14276).

`binding` is the thin ctypes layer over the C-ABI library `libdhp.so` (include/dhp.h);
`workloads` holds the seeded synthetic inputs, `shard` the multi-GPU index arithmetic and NCCL plumbing.  Importing the package does not load the
CUDA library; the first call through `binding` does, and fails loudly if it is missing.
"""
__all__ = ["binding", "workloads", "shard"]
