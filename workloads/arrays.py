"""Array plumbing shared by the tests, bench.py and smoke(): names of the particle arrays, the grid tuple of a Config,
numpy copies of a generated species.  No arithmetic of the method."""
from __future__ import annotations

import numpy as np

PKEYS = ("x", "y", "z", "u", "v", "w", "q")


def grid_of(cfg):
    """(nx, ny, nz, dx, dy, dz) of a workloads.Config: the first six arguments of ecsim_init_grid / of the oracle."""
    return (cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz)


def to_numpy(part: dict) -> dict:
    """float64 numpy copies of a generated species (torch tensors, any device)."""
    return {k: np.ascontiguousarray(part[k].detach().cpu().numpy()).copy() for k in PKEYS}
