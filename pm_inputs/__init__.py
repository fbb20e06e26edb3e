"""Seeded synthetic particle sets and fields for the PM / NUFFT force path.

This package is the ONLY code shared by the fp64 oracle (``oracle/``) and the
CUDA path (``paper_2510_05206_b200``).  It contains no arithmetic of the method
itself (no assignment kernels, no Green's functions, no NUFFT kernels): it only
draws the inputs whose recipe DESIGN.md ("Input recipe") states.  The paper's
real workloads (N-GenIC / MONOFONIC initial conditions evolved against a
Gadget-4 reference) are not available; these generators stand
in for them with the same shapes (N = n_p^3 particles in Lagrangian lattice
order, periodic box, fp32 positions).
"""
from .generators import (  # noqa: F401
    CONFIGS,
    lattice_displaced,
    clustered_halos,
    gaussian_cotangent,
    random_mesh,
    uniform_random,
    make_config_positions,
)
