"""Seeded synthetic-crystal input generators for the GW self-energy path.

This module is shared by the CPU oracle (``oracle/``) and by the CUDA path's
tests / bench.  It holds NONE of the method's arithmetic (no Sigma contraction,
no unfold, no block transform): it only builds inputs -- lattices, space-group
operations, representation matrices, and the seeded tensors G, V, W~ of
BASELINE.json's configs -- following SURVEY.md section 8(c) items G1-G10.

Paper: arXiv 2405.09494 (Dong & Gull).  Citations are PAPER.md:<line>.
"""
from .group import (  # noqa: F401
    real_harmonics, wigner_D_real, lattice_point_group, find_space_group,
    SpaceGroup, KMesh,
)
from .crystal import Crystal, make_crystal, CONFIG_NAMES  # noqa: F401
from .tensors import SymmetricInputs, RandomC1Inputs, make_inputs, tau_grid  # noqa: F401
