"""CPU oracle of the projection step -- TEST INFRASTRUCTURE, NOT PRODUCT (see oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It imports nothing from the CUDA package.
"""
from .oracle import (  # noqa: F401
    BC_Z_PERIODIC, BC_Z_WALL, rhs, poisson, projection_step, projection_step_paper, correction,
    dft_axis, divergence, laplacian, threads,
    BC_PERIODIC, BC_NEUMANN, BC_DIRICHLET, r2r_axis, eigenvalues, divergence_bc, laplacian_bc, poisson_bc, rhs_bc,
    correction_bc, projection_step_bc, momentum_prediction, vof_step, vof_reconstruct, tanh_integral,
)
