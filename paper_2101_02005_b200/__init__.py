"""B200-native line-by-line opacity hot path (HELIOS-K 2.0, arxiv 2101.02005).

The product is the C-ABI CUDA library declared in include/hk.h (built to
paper_2101_02005_b200/libhk.so by build.py); `binding` marshals torch tensors
to it.  Importing `binding` without the built library raises: no CPU fallback.
"""
__all__ = ["build", "binding"]
