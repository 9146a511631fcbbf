"""Seeded synthetic inputs for the exact-exchange hot path (shared by tests, bench and oracle drivers).

This package holds NONE of the method's arithmetic (no co-density, no FFT, no Poisson solve, no K psi):
it only draws parameters from a self-written SplitMix64 stream and evaluates sums of Gaussians on a grid,
optionally Loewdin-orthonormalises them, and tabulates the Green's functions (free-boundary 1/|d|; image sums of a
screened kernel for slab / wire boundary conditions) that the host hands to ``exx_plan_create`` as *data*.  The recipe is SURVEY.md section 8(d) / DESIGN.md "Input recipe".
"""
from .generator import (  # noqa: F401
    CONFIGS,
    SplitMix64,
    WorkloadSpec,
    cell_average_inverse_r,
    free_kernel_table,
    general_cell_khat,
    make_orbitals,
    make_workload,
    mixed_bc_kernel_table,
    small_spec,
)
