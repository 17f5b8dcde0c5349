"""CPU oracle for the column-generation VMAT hot path — TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It is independent of paper_1005_4396_b200 (the CUDA path): no shared code, and
neither imports the other.  See oracle/vmat_oracle.c for the arithmetic and its citations.
"""
from .vmat_oracle import (  # noqa: F401
    Oracle,
    build,
    num_threads,
    set_num_threads,
    penalty,
    smooth,
    smooth_occ,
    quantise,
    row_search,
)
