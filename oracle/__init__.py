"""fp64 CPU oracle for the PIMD hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2503_23728_b200/.
See oracle/pimd_oracle.c for the algorithm statement and the list of parity pins.
"""
from .ref import (  # noqa: F401
    RefPIMD,
    RefNet,
    philox4x32_10,
    normal3,
    nm_matrix,
    nlist_brute,
    nlist_cell,
    num_threads,
    set_num_threads,
    KB_EV,
    HBAR_EVFS,
    AMU_INTERNAL,
)
