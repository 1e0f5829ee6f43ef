"""CPU oracle for the staggered Dslash / CG / multi-shift CG path -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product (paper_1701_00426_b200) never does.
See staggered_oracle.c for the arithmetic and its citations, oracle.py for the ctypes wrapper.
"""
from .oracle import (  # noqa: F401
    dirac_full,
    dirac_site,
    dirac_range,
    dslash_half,
    mdagm,
    reconstruct_row3,
    cg,
    cg_multishift,
    rational_apply,
    fermion_force,
    gauge_staples,
    SYMANZIK_C0, SYMANZIK_C1,
    half_to_full,
    full_to_half,
    num_threads,
    set_num_threads,
)
