"""Seeded synthetic workload generators (BASELINE.json `configs`).

This package serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_17971_b200/`).  It assembles inputs only (K as CSR, lumped mass m,
targets y_d, bounds psi, seeds, hashes); it holds none of the method's
arithmetic (no H apply, no CG, no PDAS) and imports neither side.
"""
from .cht import (  # noqa: F401
    Workload,
    make_config,
    make_steady_2d,
    make_steady_3d,
    make_spacetime_2d,
    gaussian_targets,
    spacetime_targets,
    sha_arrays,
    CONFIGS,
    TWINS,
)
