"""b200-eigh: dense complex-FP64 Hermitian eigensolver for B200 (sm_100a).

The product is the C-ABI library declared in include/eigh.h (built in-tree as
paper_2310_03341_b200/libeigh_b200.so) and the thin ctypes binding in `binding`.
There is no CPU fallback: every call into `binding` fails loudly when the CUDA library
is missing.  `workloads` only builds seeded test matrices.
"""
__version__ = "0.1.0"
