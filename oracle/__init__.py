"""CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle_eigh.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  paper_2310_03341_b200 never does.
"""
from . import densities  # noqa: F401  (SCF epilogue oracle, Eq. 16-17)
from . import assemble   # noqa: F401  (SCF prologue oracle, Eq. 5/7/8)
from .oracle import (build, eigh, eigh_ld, tridiagonalise, tridiag_ql, tridiag_ql_ld,
                     num_threads, sturm_count)

__all__ = ["build", "eigh", "eigh_ld", "tridiagonalise", "tridiag_ql", "tridiag_ql_ld",
           "num_threads", "sturm_count"]
