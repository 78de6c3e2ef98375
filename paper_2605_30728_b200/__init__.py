"""B200-native Invariant Bit Packing: fused gather-and-decompress of indexed compressed rows (arxiv/paper_2605_30728).

The product is the C-ABI library `libibp.so` (include/ibp.h; sources in csrc/, sm_100a only).  `binding` is the thin
ctypes layer with the same names.  There is no CPU fallback: every step of the hot path runs in the CUDA kernels.
"""
__all__ = ["binding", "workloads", "datagen"]
