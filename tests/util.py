"""Shared test helpers: glue between the input generator, the oracle and the CUDA binding."""
from __future__ import annotations

import numpy as np

import workloads as wl

from workloads import PKEYS, grid_of, to_numpy  # noqa: F401  (they live in workloads/arrays.py; bench.py uses them too)


def rand_particles(rng, n, grid, vscale=1.0, qscale=1.0):
    nx, ny, nz, dx, dy, dz = grid
    return dict(
        x=rng.uniform(0, nx * dx, n), y=rng.uniform(0, ny * dy, n), z=rng.uniform(0, nz * dz, n),
        u=vscale * rng.standard_normal(n), v=vscale * rng.standard_normal(n),
        w=vscale * rng.standard_normal(n), q=qscale * rng.uniform(0.5, 1.5, n) * rng.choice([-1.0, 1.0], n))


def rand_fields(rng, grid, escale=1.0, bscale=1.0):
    nodes = grid[0] * grid[1] * grid[2]
    return escale * rng.standard_normal((3, nodes)), bscale * rng.standard_normal((3, nodes))


def copy_part(p):
    return {k: v.copy() for k, v in p.items()}


def periodic_absdiff(a, b, L):
    d = np.abs(a - b)
    return np.minimum(d, L - d)
