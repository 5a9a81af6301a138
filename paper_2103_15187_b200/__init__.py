"""B200-native fp64 pressure projection (arXiv 2103.15187 hot path).

`paper_2103_15187_b200.binding` is the thin ctypes binding over the C-ABI library
libfsei.so (include/fsei.h); `paper_2103_15187_b200.inputs` holds the seeded input
generators.  Nothing is imported eagerly: the input generators work without CUDA, the
binding fails loudly when libfsei.so is missing (there is no CPU fallback).
"""
__all__ = ["binding", "inputs", "build"]
