"""Seeded synthetic inputs shared by the oracle and the CUDA library.

This package holds NO arithmetic of the method (no Hamiltonian, no operators,
no contractions).  It only produces the *inputs* both sides read: integrals,
bond sector tables, random mixed-canonical MPS tensors, the two-site wave
function and random operator blocks (DESIGN.md "Input
recipe").  Everything is deterministic in (config, seed).
"""
from .configs import CONFIGS, Config, get_config  # noqa: F401
from .integrals import make_integrals  # noqa: F401
from .sectors import site_states, fuse, block_tables, bond_tables_for, fock_count  # noqa: F401
from .mps import (random_isometries, random_isometry, isometry_blocks, random_psi,  # noqa: F401
                  random_vector)
