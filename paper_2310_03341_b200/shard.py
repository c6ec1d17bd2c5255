"""Column sharding of the eigenvector back-transformations over ranks (first slice).

S4a and S4b act on every column of Z independently (Z <- Q2 Z, Z <- Q1 Z) and are 72 % of the solve at N = 49152, so the
first multi-GPU cut is: S1-S3 replicated on every rank (identical bits: the solver is deterministic), each rank
back-transforms its own slab-aligned column range, and the ranges are gathered (or left distributed: the SCF epilogue
reduces densities over columns, a ~50 MB all-reduce as in PAPER.md:99).  This module holds the host-side plan only: no
arithmetic of the method, no CUDA.
"""
from __future__ import annotations

from typing import List, Tuple

SLAB = 64          # S4a works on slabs of 64 eigenvector columns (bt_sweep_kernel: 8 warps x 8 columns)


def column_shards(nev: int, world: int, slab: int = SLAB) -> List[Tuple[int, int]]:
    """[begin, end) column range of every rank: contiguous, slab-aligned (except the global tail), sizes differing by at
    most one slab, empty ranges for ranks beyond the number of slabs."""
    if nev < 0 or world < 1 or slab < 1:
        raise ValueError("column_shards: bad arguments")
    nslabs = -(-nev // slab)
    base, extra = divmod(nslabs, world)
    out, s = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        b, e = min(s * slab, nev), min((s + n) * slab, nev)
        out.append((b, e))
        s += n
    return out


def backtransform_flops(N: int, shard: Tuple[int, int]) -> float:
    """Credited flops of S4a + S4b for one shard (8 N^2 columns each): the quantity the shards balance."""
    return 2 * 8.0 * N * N * (shard[1] - shard[0])
