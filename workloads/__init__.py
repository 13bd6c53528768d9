"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the method (no codec, no SpMV, no GMRES): it only
builds the CSR matrices, right-hand sides and basis inputs of BASELINE.json's five configs
(SURVEY.md §8(d)).  Everything is made on the host with
``numpy.random.default_rng(seed)``; both sides read the same arrays.
"""
from .generators import (  # noqa: F401
    CSR,
    Problem,
    laplace2d_5pt,
    convdiff3d_7pt,
    stencil3d_27pt,
    powerlaw_rows,
    make_config,
    ortho_basis,
    random_dense_system,
    CONFIG_NAMES,
)
