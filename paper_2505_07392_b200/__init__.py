"""B200-native IGR Euler hot path (arXiv 2505.07392): C-ABI library `libigr.so` + thin binding.

`workloads` (seeded inputs) imports on any machine; `igr` (the binding) needs the built CUDA
library and fails loudly without it -- there is no CPU fallback.
"""
__all__ = ["workloads", "igr"]
