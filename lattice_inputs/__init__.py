"""Seeded synthetic input generators shared by the oracle-side tests and the CUDA-side tests/bench.

This package holds NO arithmetic of the method (no gamma matrices, no stencil, no compression, no
polynomial): it only draws the random SU(3) gauge fields and spinor sources described in
BASELINE.json's configs (the paper's epsilon-regime gauge ensembles, are not
available; these seeded fields stand in for them - recipe in DESIGN.md section 4).

Canonical array conventions:
    dims  = (L0, L1, L2, L3), L0 = time extent T, x3 fastest in memory
    U     : complex128 [4(mu), L0, L1, L2, L3, 3(row), 3(col)]
    psi   : complex128 [L0, L1, L2, L3, 4(spin), 3(colour)]
"""
from .generators import (  # noqa: F401
    SEED_GAUGE,
    SEED_SOURCE,
    SEED_TRANSFORM,
    flux_su3,
    gaussian_spinor,
    gauge_field,
    haar_su3,
    lattice_name,
    parse_lattice,
    smooth_su3,
    unit_su3,
)
