"""CPU oracle for the HPRMAT hot path (arxiv 2512.11590).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It shares no code with paper_2512_11590_b200 (the CUDA path) and neither imports the other.
"""
from .oracle import (mesh, kinetic, assemble, rhs, solve, structured_residual, contract, rmatrix,  # noqa: F401
                     collision_matrix, rmatrix_nonlocal, num_threads, sector_tables, sector_matrices, propagate)
