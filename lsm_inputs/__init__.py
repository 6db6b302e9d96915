"""Seeded synthetic input generators shared by the oracle tests, the GPU parity tests and bench.py.

This package builds ARRAYS ONLY (particle coordinates, spring lists, parameter values, boundary id lists).
It holds none of the method's arithmetic (no force, no integration, no reduction): the oracle (`oracle/`)
and the CUDA path (`paper_2201_04565_b200/`) each implement that on their own and share no code.
"""
from .generators import (  # noqa: F401
    Problem, BoundaryGroup, triangular_lattice, blob_image, two_phase_spring_params, porous_keep_mask,
    config1, config2, config3, config4, config5, shuffle_ids, velocity_ramp, single_specimen, cubic_lattice_3d, config3d, FIXED, MOVE,
)
