"""B200-native Ising max-cut annealer (arXiv 1807.10750): Python side of the C-ABI library.

`binding` marshals arguments into libising_b200.so (hand-written sm_100a kernels);
`workloads` holds the seeded synthetic input generators shared with the oracle tests.
"""
from . import workloads  # noqa: F401
from .binding import (  # noqa: F401
    ENGINE_CLUSTER, ENGINE_GRID, ENGINE_GRID_TAIL_CHAIN, ENGINE_PER_PHASE, ENGINE_SMALL, ISING_INIT_CONTINUE,
    ISING_INIT_GIVEN, ISING_INIT_PHILOX, ISING_LOAD_NO_CLUSTER, ISING_LOAD_NO_DENSE, ISING_LOAD_NO_SMALL,
    ISING_LOAD_NO_OVERLAP, ISING_LOAD_NO_TAIL_CHAIN, ISING_MODE_GS,
    ISING_MODE_EXACT_N, ISING_MODE_JACOBI, ISING_MODE_RACY, ISING_TIE_KEEP, ISING_TIE_MINUS, IsingError, Problem,
    anneal_workload, ising_anneal, ising_best_state, ising_current_state, ising_energy_cut, ising_free,
    ising_load_csr, ising_workspace_bytes, load_workload)
