"""B200-native split-step phase-screen propagation (TurPy hot path, arxiv 2604.07248).

The product is the C-ABI library declared in include/ssp.h (built in-tree as
paper_2604_07248_b200/libssp.so); `paper_2604_07248_b200.api` is its thin ctypes
binding.  Importing this package is cheap and never loads CUDA; the binding fails
loudly if the library has not been built.  There is no CPU fallback.
"""
__all__ = ["api", "synth", "build"]
