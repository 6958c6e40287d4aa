"""Seeded synthetic inputs for the coarse-grid Dirac operator apply.

This package serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.
It holds none of the method's arithmetic (no operator apply, no quantiser): it
only draws seeded random link matrices and vectors with the structure
BASELINE.json's configs ask for (recipe: DESIGN.md "Synthetic inputs").
"""
from .generator import (  # noqa: F401
    FIELD_YPLUS, FIELD_G, FIELD_IN, FIELD_ANY,
    normal, make_gamma_hermitian_links, make_arbitrary_links, make_vectors,
    site_index, lattice_volume, CONFIGS, config,
)
