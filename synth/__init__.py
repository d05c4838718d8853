"""Seeded synthetic inputs (Hamiltonians, initial MPS) shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the DMRG method itself: it only manufactures the inputs
(h_pq, (pq|rs), E_core, a seeded block-sparse orthonormal MPS) that both implementations read.
Recipes: BASELINE.json configs[0..4]; readings S6-S10, S15, S23 of SURVEY.md section 8(c).
"""
from .hamiltonians import (hex_graph, flake_centres, row_centres, ppp_integrals, rotate_orbitals, fiedler_order,
                           permute_orbitals, fes_like, make_config, random_dense, CONFIG_SEED)
from .mps import (random_mps, dual_gauge_mps, mixed_gauge, bond_sector_plan, full_sector_dims, mps_to_blob_arrays, blob_arrays_to_mps, SITE_Q)
