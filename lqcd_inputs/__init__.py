"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no stencil, no solver, no
row-3 reconstruction): it only draws random fields in the canonical layout of
DESIGN.md ("Canonical data").  Both `oracle/` and `paper_1701_00426_b200/`
consume the arrays it returns; neither imports the other.
"""
from .fields import (  # noqa: F401
    volume,
    haar_like_links,
    smooth_links,
    unit_links,
    gaussian_spinor,
    gaussian_half_spinor,
    rhmc_shifts,
    uniform_backfield,
    site_coords,
    half_index_of_parity,
)
