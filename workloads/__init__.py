"""Seeded synthetic input generators (water clusters, synthetic Gaussian basis, density matrix).

This module is shared by the CPU oracle's tests and by the CUDA path's tests/bench.  It holds
none of the XC-integration arithmetic: no grids, no partition weights, no collocation, no
functionals.  The only mathematics here is what is needed to *construct an input*: the closed-form
Gaussian overlap matrix S used to S-orthonormalise the random orbitals (so that tr(P S) = 2 N_occ).
"""
from .water_clusters import (CONFIGS, Workload, make_workload, overlap_matrix,  # noqa: F401
                             ncart, nfun, PURE, cart_components, ANGSTROM, spin_density_matrices)
