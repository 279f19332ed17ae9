"""CPU oracle of the ECsim particle hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

`oracle.step` / `oracle.cells` / `oracle.apply_M` / `oracle.diagnostics` wrap the plain C restatement of the paper's
equations in `ecsim_oracle.c`; `oracle.dense` is the hat-function definition written out in
numpy for tiny grids.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package; it imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import numpy as np

from . import build as _build
from . import dense  # noqa: F401

_lib = None
_D = ctypes.POINTER(ctypes.c_double)
_I32 = ctypes.POINTER(ctypes.c_int32)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.ecsim_oracle_step.restype = ctypes.c_int
        _lib.ecsim_oracle_step.argtypes = (
            [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [ctypes.c_int64, ctypes.c_double, ctypes.c_double]
            + [_D] * 6 + [_D] * 3 + [_D] * 3 + [_D] * 3 + [_D, ctypes.c_int])
        _lib.ecsim_oracle_cells.restype = ctypes.c_int
        _lib.ecsim_oracle_cells.argtypes = (
            [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [ctypes.c_int64] + [_D] * 3 + [_I32, _I32])
        _lib.ecsim_oracle_apply_M.restype = ctypes.c_int
        _lib.ecsim_oracle_apply_M.argtypes = [ctypes.c_int] * 3 + [_D] * 3
        _lib.ecsim_oracle_fix_position.restype = ctypes.c_int
        _lib.ecsim_oracle_fix_position.argtypes = [ctypes.c_int64] + [_D] * 3 + [ctypes.c_int] + [ctypes.c_double] * 3
        _lib.ecsim_oracle_threads.restype = ctypes.c_int
        _lib.ecsim_oracle_threads.argtypes = []
        _lib.ecsim_oracle_step_planes.restype = ctypes.c_int
        _lib.ecsim_oracle_step_planes.argtypes = (
            [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [ctypes.POINTER(ctypes.c_int64), ctypes.c_double, ctypes.c_double]
            + [_D] * 6 + [_D] * 3 + [_D] * 3 + [ctypes.c_int])
        _lib.ecsim_oracle_diagnostics.restype = ctypes.c_int
        _lib.ecsim_oracle_diagnostics.argtypes = ([ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [ctypes.c_int64]
                                                  + [_D] * 7 + [_D] * 4 + [_D] * 4)
    return _lib


def _p(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_D)


class Moments:
    """rho [nodes], J [3][nodes], M [nodes][27][3][3] and (optionally) their |addend| sums."""

    def __init__(self, nodes: int, with_abs: bool = True):
        self.rho = np.zeros(nodes)
        self.J = np.zeros((3, nodes))
        self.M = np.zeros((nodes, 27, 3, 3))
        self.rho_abs = np.zeros(nodes) if with_abs else None
        self.J_abs = np.zeros((3, nodes)) if with_abs else None
        self.M_abs = np.zeros((nodes, 27, 3, 3)) if with_abs else None


def step(grid, qom: float, dt: float, part: dict, E: np.ndarray, B: np.ndarray, mom: Moments,
         push: bool = True, want_vbar: bool = False):
    """One oracle step for one species.  `grid` = (nx, ny, nz, dx, dy, dz); `part` holds float64
    numpy arrays x,y,z,u,v,w,q (x..w updated in place when push).  Accumulates into `mom`.
    Returns vbar [3][n] if requested."""
    nx, ny, nz, dx, dy, dz = grid
    n = part["x"].shape[0]
    vbar = np.zeros((3, n)) if want_vbar else None
    rc = lib().ecsim_oracle_step(
        nx, ny, nz, dx, dy, dz, n, qom, dt,
        _p(part["x"]), _p(part["y"]), _p(part["z"]), _p(part["u"]), _p(part["v"]), _p(part["w"]),
        _p(part["q"]), _p(E), _p(B), _p(mom.rho), _p(mom.J), _p(mom.M),
        _p(mom.rho_abs), _p(mom.J_abs), _p(mom.M_abs), _p(vbar), 1 if push else 0)
    assert rc == 0
    return vbar


def cells(grid, x: np.ndarray, y: np.ndarray, z: np.ndarray):
    """(cell[n] int32, count[cells] int32): cell id of every particle and the histogram."""
    nx, ny, nz, dx, dy, dz = grid
    n = x.shape[0]
    cell = np.zeros(n, dtype=np.int32)
    count = np.zeros(nx * ny * nz, dtype=np.int32)
    rc = lib().ecsim_oracle_cells(nx, ny, nz, dx, dy, dz, n, _p(x), _p(y), _p(z),
                                  cell.ctypes.data_as(_I32), count.ctypes.data_as(_I32))
    assert rc == 0
    return cell, count


def apply_M(grid, M: np.ndarray, E: np.ndarray) -> np.ndarray:
    """sum_N' M_NN' E_N' per node, [3][nodes] (operator of Eq. 4-5)."""
    nx, ny, nz = grid[:3]
    out = np.zeros((3, nx * ny * nz))
    rc = lib().ecsim_oracle_apply_M(nx, ny, nz, _p(M), _p(E), _p(out))
    assert rc == 0
    return out


class Diagnostics:
    """rho [nodes], J [3][nodes] (un-rotated), P [6][nodes] (xx,xy,xz,yy,yz,zz), Q [3][nodes] and |addend| sums."""

    def __init__(self, nodes: int, with_abs: bool = True):
        self.rho = np.zeros(nodes)
        self.J = np.zeros((3, nodes))
        self.P = np.zeros((6, nodes))
        self.Q = np.zeros((3, nodes))
        self.rho_abs = np.zeros(nodes) if with_abs else None
        self.J_abs = np.zeros((3, nodes)) if with_abs else None
        self.P_abs = np.zeros((6, nodes)) if with_abs else None
        self.Q_abs = np.zeros((3, nodes)) if with_abs else None


def diagnostics(grid, part: dict, diag: Diagnostics):
    """Diagnostic moments of one species (R22-R24), accumulated into `diag`."""
    nx, ny, nz, dx, dy, dz = grid
    n = part["x"].shape[0]
    rc = lib().ecsim_oracle_diagnostics(
        nx, ny, nz, dx, dy, dz, n, _p(part["x"]), _p(part["y"]), _p(part["z"]), _p(part["u"]), _p(part["v"]),
        _p(part["w"]), _p(part["q"]), _p(diag.rho), _p(diag.J), _p(diag.P), _p(diag.Q),
        _p(diag.rho_abs), _p(diag.J_abs), _p(diag.P_abs), _p(diag.Q_abs))
    assert rc == 0


def threads() -> int:
    """Threads the timing variant `step_planes` will use (OpenMP max threads)."""
    return int(lib().ecsim_oracle_threads())


def step_planes(grid, qom: float, dt: float, part: dict, plane_start: np.ndarray, E: np.ndarray, B: np.ndarray,
                mom: Moments, push: bool = True):
    """TIMING VARIANT on all host cores: `step` called per x-plane of cells, even planes in parallel, then odd planes
    (no arithmetic of its own).  `part` must be ordered by x-plane of cells, plane i = [plane_start[i], plane_start[i+1])."""
    nx, ny, nz, dx, dy, dz = grid
    ps = np.ascontiguousarray(plane_start, dtype=np.int64)
    assert ps.shape[0] == nx + 1
    rc = lib().ecsim_oracle_step_planes(
        nx, ny, nz, dx, dy, dz, ps.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), qom, dt,
        _p(part["x"]), _p(part["y"]), _p(part["z"]), _p(part["u"]), _p(part["v"]), _p(part["w"]),
        _p(part["q"]), _p(E), _p(B), _p(mom.rho), _p(mom.J), _p(mom.M), 1 if push else 0)
    assert rc == 0, "particles are not ordered by x-plane of cells"


def fix_position(part: dict, axis_mask: int, px: float = 0.0, py: float = 0.0, pz: float = 0.0):
    """fixPosition (reading R25): pin the coordinates of the masked axes in place."""
    rc = lib().ecsim_oracle_fix_position(part["x"].shape[0], _p(part["x"]), _p(part["y"]), _p(part["z"]), axis_mask,
                                         px, py, pz)
    assert rc == 0
