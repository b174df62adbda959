"""B200-native Wolff single-cluster hot path (arXiv 1110.0899) behind the C-ABI of include/wolff.h.

Importing the package is cheap and has no side effects; the CUDA library is loaded on first use by
`binding.load()` / `binding.Wolff`, and that raises loudly if `libwolff_b200.so` is missing -- there is no
CPU fallback anywhere in this package.
"""
__all__ = ["binding", "build", "workloads"]
