"""Seeded synthetic N-body inputs shared by the oracle tests and the CUDA tests/bench.

This module holds NONE of the method's arithmetic (no keys, no tree, no forces): it only
draws particle positions, velocities and masses.  Both sides (``oracle/`` and the CUDA
library) are handed the very same arrays.  Recipes are stated in DESIGN.md §"Input recipe";
the paper's own initial conditions (GalacticICS) are not available, so
these samplers stand in for them with the same component shapes.
"""
from .generators import (  # noqa: F401
    uniform01,
    plummer,
    milky_way,
    milky_way_clumpy,
    subsample_indices,
    config,
    CONFIGS,
)
