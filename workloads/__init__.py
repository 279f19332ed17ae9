"""Seeded synthetic inputs for the ECsim particle hot path (configs 0-4 of BASELINE.json).

This package serves BOTH the CPU oracle's tests and the CUDA path's tests/bench.  It holds none
of the method's arithmetic (no weights, no rotation matrix, no deposit): only a counter-based
random-number generator and the recipes of DESIGN.md "Input recipe" that turn it into particle
positions/velocities/charges and node fields.  It imports neither `oracle` nor the CUDA package.
"""
from .generator import (  # noqa: F401
    Config,
    Species,
    config,
    gen_fields,
    gen_species,
    cell_layout,
    N_CONFIGS,
)
from .arrays import PKEYS, grid_of, to_numpy  # noqa: F401
