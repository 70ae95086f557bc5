"""B200-native Feynman-Kac exit-time hot path (arXiv 2104.14561, Algorithm 1).

`workloads` (inputs only, numpy) imports without CUDA.  The CUDA path lives behind the C ABI
in include/fk.h; `binding` loads the in-tree shared library and fails loudly when it is
missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
