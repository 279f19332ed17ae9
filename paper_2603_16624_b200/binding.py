"""ctypes binding of libecpush.so (include/ecpush.h).  Argument marshalling only.

`lib()` returns the loaded library with typed prototypes named exactly as in the header.
`Ecsim` is a small convenience wrapper that owns an `ecsim_ctx*`, lets PyTorch allocate the
workspace, and forwards torch CUDA tensors as raw device pointers.
"""
from __future__ import annotations

import ctypes
import os
import re
from typing import Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
HEADER = os.path.join(ROOT, "include", "ecpush.h")

VARIANT_ATOMIC = 0
VARIANT_FUSED = 1
ACC_NONE = 0
ACC_ALL = 1
ACC_M_ONLY = 2
M_27 = 0
M_14 = 1
STATIC_MAX_CELLS = 2097152      # ECSIM_STATIC_MAX_CELLS of ecpush.h: the grid the built-in scratch can serve

_c = ctypes
_P = _c.c_void_p
_lib = None


class EcsimError(RuntimeError):
    pass


def lib_path() -> str:
    return os.path.join(HERE, "libecpush.so")


def declared_symbols() -> list:
    """Names of every function include/ecpush.h declares (used by the ABI test)."""
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ecsim_[A-Za-z0-9_]+)\s*\(", text)))


_PROTOS = {
    "ecsim_init_grid": (_c.c_int, [_c.POINTER(_P), _c.c_int, _c.c_int, _c.c_int, _c.c_double, _c.c_double,
                                   _c.c_double, _c.c_int, _P]),
    "ecsim_workspace_bytes": (_c.c_size_t, [_P, _c.c_int64]),
    "ecsim_set_workspace": (_c.c_int, [_P, _P, _c.c_size_t]),
    "ecsim_load_particles": (_c.c_int, [_P, _c.c_int, _c.c_int64, _c.c_double] + [_P] * 7 + [_c.c_int]),
    "ecsim_sort_particles": (_c.c_int, [_P, _c.c_int, _P, _P]),
    "ecsim_validate_particles": (_c.c_int64, [_P, _c.c_int]),
    "ecsim_build_segments": (_c.c_int, [_P, _c.c_int]),
    "ecsim_cell_index": (_c.c_int, [_P, _c.c_int, _P]),
    "ecsim_push_and_moments": (_c.c_int, [_P, _c.c_int, _P, _P, _c.c_double, _c.c_double, _P, _P, _P, _c.c_int]),
    "ecsim_push_and_moments_all": (_c.c_int, [_P, _P, _P, _c.c_double, _c.c_double, _P, _P, _P, _c.c_int]),
    "ecsim_moments": (_c.c_int, [_P, _c.c_int, _P, _c.c_double, _P, _P, _P, _c.c_int]),
    "ecsim_moments_all": (_c.c_int, [_P, _P, _c.c_double, _P, _P, _P, _c.c_int]),
    "ecsim_push": (_c.c_int, [_P, _c.c_int, _P, _P, _c.c_double, _c.c_double]),
    "ecsim_push_all": (_c.c_int, [_P, _P, _P, _c.c_double, _c.c_double]),
    "ecsim_resident_bytes": (_c.c_size_t, [_P, _c.c_int64, _c.c_double]),
    "ecsim_make_resident": (_c.c_int, [_P, _c.c_int, _P, _c.c_size_t, _c.c_double]),
    "ecsim_export_particles": (_c.c_int, [_P, _c.c_int] + [_P] * 7),
    "ecsim_relayout_count": (_c.c_int64, [_P]),
    "ecsim_set_overflow_capacity": (_c.c_int, [_P, _c.c_int, _c.c_int64]),
    "ecsim_set_host_pipeline": (_c.c_int, [_P, _c.c_int]),
    "ecsim_host_pipelined_count": (_c.c_int64, [_P]),
    "ecsim_apply_M": (_c.c_int, [_P, _P, _P, _P, _c.c_int]),
    "ecsim_diagnostics": (_c.c_int, [_P, _c.c_int, _P, _P, _P, _P]),
    "ecsim_set_fixed_axes": (_c.c_int, [_P, _c.c_int, _c.c_double, _c.c_double, _c.c_double]),
    "ecsim_host_step_workspace_bytes": (_c.c_size_t, [_P, _c.c_int64]),
    "ecsim_push_and_moments_host": (_c.c_int, [_P, _c.c_int64, _c.c_double, _c.c_int] + [_P] * 9 +
                                    [_c.c_double, _c.c_double, _P, _P, _P, _c.c_int]),
    "ecsim_host_step_all_workspace_bytes": (_c.c_size_t, [_P, _c.c_int64, _c.c_int64]),
    "ecsim_push_and_moments_host_all": (_c.c_int, [_P, _P, _P, _c.c_int] + [_P] * 9 +
                                        [_c.c_double, _c.c_double, _P, _P, _P, _c.c_int]),
    "ecsim_set_variant": (_c.c_int, [_P, _c.c_int]),
    "ecsim_set_resort_fraction": (_c.c_int, [_P, _c.c_double]),
    "ecsim_set_fused_warps": (_c.c_int, [_P, _c.c_int]),
    "ecsim_set_m_layout": (_c.c_int, [_P, _c.c_int]),
    "ecsim_enable_timing": (_c.c_int, [_P, _c.c_int]),
    "ecsim_kernel_ms": (_c.c_int, [_P, _c.POINTER(_c.c_float)]),
    "ecsim_launch_count": (_c.c_int64, [_P]),
    "ecsim_stray_count": (_c.c_int64, [_P]),
    "ecsim_leaver_count": (_c.c_int64, [_P]),
    "ecsim_resort_count": (_c.c_int64, [_P]),
    "ecsim_probe_fp64": (_c.c_int, [_P, _c.c_int, _c.POINTER(_c.c_double), _c.POINTER(_c.c_float)]),
    "ecsim_destroy": (_c.c_int, [_P]),
    "ecsim_cell_segments_static": (_c.c_int, [_P, _c.c_int, _c.c_int, _c.c_int, _c.c_double, _c.c_double, _c.c_double,
                                              _c.c_int64, _P, _P, _P, _P, _P]),
    "ecsim_strerror": (_c.c_char_p, [_c.c_int]),
    "ecsim_last_error": (_c.c_char_p, []),
}


def lib():
    """Load libecpush.so (built in-tree by paper_2603_16624_b200.build).  Fails loudly."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise EcsimError(f"{path} is missing: build it with `python -m paper_2603_16624_b200.build` "
                             "(there is no CPU fallback)")
        L = _c.CDLL(path)
        for name, (res, args) in _PROTOS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        L = lib()
        raise EcsimError(f"{what}: {L.ecsim_strerror(rc).decode()} [{rc}] {L.ecsim_last_error().decode()}")


def _dptr(t, dtype=None):
    """Raw device pointer of a contiguous CUDA tensor (or None)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise EcsimError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise EcsimError(f"expected dtype {dtype}, got {t.dtype}")
    return _P(t.data_ptr())


def _hptr(t, dtype=None):
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise EcsimError("expected a contiguous host tensor")
    if dtype is not None and t.dtype != dtype:
        raise EcsimError(f"expected dtype {dtype}, got {t.dtype}")
    return _P(t.data_ptr())


def cell_segments_static(nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, x, y, z,
                         cell_count_out=None, start_out=None, stream=None):
    """ecsim_cell_segments_static: per-cell counts (int32[cells]) and / or the segment table (uint32[cells+1], stored in
    an int32 or uint32 tensor) of the particles at x, y, z, for callers that cannot allocate device memory: no context,
    no workspace, the scratch is an array built into libecpush.so (grids up to STATIC_MAX_CELLS cells).  Work is
    enqueued on `stream` (default: torch's current stream); calls that may overlap on the GPU race on the shared scratch."""
    import torch
    f64 = torch.float64
    n = int(x.numel())
    if stream is None:
        stream = torch.cuda.current_stream()
    if start_out is not None and start_out.dtype not in (torch.int32, torch.uint32):
        raise EcsimError(f"start_out: expected a 32-bit integer tensor, got {start_out.dtype}")
    _check(lib().ecsim_cell_segments_static(_P(stream.cuda_stream), nx, ny, nz, dx, dy, dz, n, _dptr(x, f64),
                                            _dptr(y, f64), _dptr(z, f64), _dptr(cell_count_out, torch.int32),
                                            _dptr(start_out)), "ecsim_cell_segments_static")


class Ecsim:
    """One libecpush context on the current CUDA device and (by default) torch's current stream."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, n_species: int,
                 stream=None):
        import torch
        self.torch = torch
        if not torch.cuda.is_available():
            raise EcsimError("libecpush needs a CUDA device (no CPU fallback)")
        self.L = lib()
        self.grid = (nx, ny, nz, dx, dy, dz)
        self.nodes = nx * ny * nz
        self.n_species = n_species
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        h = _P()
        _check(self.L.ecsim_init_grid(_c.byref(h), nx, ny, nz, dx, dy, dz, n_species,
                                      _P(self.stream.cuda_stream)), "ecsim_init_grid")
        self.h = h
        self._ws = None
        self._keep = {}
        self._resident = {}

    # -- workspace -----------------------------------------------------------------------------
    def workspace_bytes(self, n_max: int) -> int:
        return int(self.L.ecsim_workspace_bytes(self.h, n_max))

    def host_step_workspace_bytes(self, n: int) -> int:
        return int(self.L.ecsim_host_step_workspace_bytes(self.h, n))

    def set_workspace(self, n_max: int, host_step: bool = False):
        """Let torch allocate the scratch and lend it to the library."""
        nbytes = self.host_step_workspace_bytes(n_max) if host_step else self.workspace_bytes(n_max)
        ws = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device="cuda")
        off = (-ws.data_ptr()) % 256
        self._ws = ws
        _check(self.L.ecsim_set_workspace(self.h, _P(ws.data_ptr() + off), nbytes), "ecsim_set_workspace")
        return nbytes

    # -- particles -----------------------------------------------------------------------------
    def load_particles(self, species: int, qom: float, part: dict, sorted: bool = False):
        f64 = self.torch.float64
        n = int(part["x"].numel())
        ptrs = [_dptr(part[k], f64) for k in ("x", "y", "z", "u", "v", "w", "q")]
        self._keep[species] = part
        self._resident.pop(species, None)
        _check(self.L.ecsim_load_particles(self.h, species, n, qom, *ptrs, 1 if sorted else 0),
               "ecsim_load_particles")

    def validate_particles(self, species: int) -> int:
        n = int(self.L.ecsim_validate_particles(self.h, species))
        if n < 0:
            _check(n, "ecsim_validate_particles")
        return n

    def sort_particles(self, species: int, cell_count_out=None, perm_out=None):
        _check(self.L.ecsim_sort_particles(self.h, species, _dptr(cell_count_out, self.torch.int32),
                                           _dptr(perm_out)), "ecsim_sort_particles")

    def build_segments(self, species: int):
        _check(self.L.ecsim_build_segments(self.h, species), "ecsim_build_segments")

    def cell_index(self, species: int, cell_out):
        _check(self.L.ecsim_cell_index(self.h, species, _dptr(cell_out, self.torch.int32)), "ecsim_cell_index")

    # -- the hot path --------------------------------------------------------------------------
    def push_and_moments(self, species: int, E, B, dt: float, theta: float, rho, Jhat, M, accumulate: int = 0):
        f64 = self.torch.float64
        _check(self.L.ecsim_push_and_moments(self.h, species, _dptr(E, f64), _dptr(B, f64), dt, theta,
                                             _dptr(rho, f64), _dptr(Jhat, f64), _dptr(M, f64),
                                             int(accumulate)), "ecsim_push_and_moments")

    def push_and_moments_all(self, E, B, dt: float, theta: float, rho, Jhat, M, accumulate: int = 0):
        f64 = self.torch.float64
        _check(self.L.ecsim_push_and_moments_all(self.h, _dptr(E, f64), _dptr(B, f64), dt, theta,
                                                 _dptr(rho, f64), _dptr(Jhat, f64), _dptr(M, f64),
                                                 int(accumulate)), "ecsim_push_and_moments_all")

    # -- the two halves as separate calls (moment gathering -> field solve -> mover) -----------
    def moments(self, species: int, B, dt: float, rho, Jhat, M, accumulate: int = 0):
        f64 = self.torch.float64
        _check(self.L.ecsim_moments(self.h, species, _dptr(B, f64), dt, _dptr(rho, f64), _dptr(Jhat, f64),
                                    _dptr(M, f64), int(accumulate)), "ecsim_moments")

    def moments_all(self, B, dt: float, rho, Jhat, M, accumulate: int = 0):
        f64 = self.torch.float64
        _check(self.L.ecsim_moments_all(self.h, _dptr(B, f64), dt, _dptr(rho, f64), _dptr(Jhat, f64),
                                        _dptr(M, f64), int(accumulate)), "ecsim_moments_all")

    def push(self, species: int, E, B, dt: float, theta: float):
        f64 = self.torch.float64
        _check(self.L.ecsim_push(self.h, species, _dptr(E, f64), _dptr(B, f64), dt, theta), "ecsim_push")

    def push_all(self, E, B, dt: float, theta: float):
        f64 = self.torch.float64
        _check(self.L.ecsim_push_all(self.h, _dptr(E, f64), _dptr(B, f64), dt, theta), "ecsim_push_all")

    # -- resident species: the sort-preserving push ---------------------------------------------------------
    def resident_bytes(self, n: int, slack: float = 0.25) -> int:
        return int(self.L.ecsim_resident_bytes(self.h, n, slack))

    def make_resident(self, species: int, slack: float = 0.25):
        """Let torch allocate the species' gapped double buffers and hand the species over to the library."""
        part = self._keep[species]
        nbytes = self.resident_bytes(int(part["x"].numel()), slack)
        buf = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device="cuda")
        off = (-buf.data_ptr()) % 256
        _check(self.L.ecsim_make_resident(self.h, species, _P(buf.data_ptr() + off), nbytes, slack),
               "ecsim_make_resident")
        self._resident[species] = buf
        return nbytes

    def export_particles(self, species: int, out: dict):
        f64 = self.torch.float64
        ptrs = [_dptr(out[k], f64) for k in ("x", "y", "z", "u", "v", "w", "q")]
        _check(self.L.ecsim_export_particles(self.h, species, *ptrs), "ecsim_export_particles")

    def set_host_pipeline(self, mode: int):
        _check(self.L.ecsim_set_host_pipeline(self.h, int(mode)), "ecsim_set_host_pipeline")

    def host_pipelined_count(self) -> int:
        return int(self.L.ecsim_host_pipelined_count(self.h))

    def set_overflow_capacity(self, species: int, entries: int):
        _check(self.L.ecsim_set_overflow_capacity(self.h, species, int(entries)), "ecsim_set_overflow_capacity")

    def relayout_count(self) -> int:
        return int(self.L.ecsim_relayout_count(self.h))

    def set_fixed_axes(self, axis_mask: int, px: float = 0.0, py: float = 0.0, pz: float = 0.0):
        _check(self.L.ecsim_set_fixed_axes(self.h, axis_mask, px, py, pz), "ecsim_set_fixed_axes")

    def diagnostics(self, species: int, rho, J, P, Q):
        f64 = self.torch.float64
        _check(self.L.ecsim_diagnostics(self.h, species, _dptr(rho, f64), _dptr(J, f64), _dptr(P, f64), _dptr(Q, f64)),
               "ecsim_diagnostics")

    # -- mass-matrix storage and operator ---------------------------------------------------------------------
    def set_m_layout(self, layout: int):
        _check(self.L.ecsim_set_m_layout(self.h, layout), "ecsim_set_m_layout")

    def apply_M(self, M, E, out, accumulate: bool = False):
        f64 = self.torch.float64
        _check(self.L.ecsim_apply_M(self.h, _dptr(M, f64), _dptr(E, f64), _dptr(out, f64), 1 if accumulate else 0),
               "ecsim_apply_M")

    def push_and_moments_host(self, qom: float, sorted: bool, part: dict, E, B, dt: float, theta: float,
                              rho, Jhat, M, accumulate: int = 0):
        f64 = self.torch.float64
        n = int(part["x"].numel())
        ptrs = [_hptr(part[k], f64) for k in ("x", "y", "z", "u", "v", "w", "q")]
        _check(self.L.ecsim_push_and_moments_host(self.h, n, qom, 1 if sorted else 0, *ptrs, _hptr(E, f64),
                                                  _hptr(B, f64), dt, theta, _hptr(rho, f64), _hptr(Jhat, f64),
                                                  _hptr(M, f64), int(accumulate)),
               "ecsim_push_and_moments_host")

    def set_workspace_host_all(self, n_max: int, n_total: int):
        nbytes = int(self.L.ecsim_host_step_all_workspace_bytes(self.h, n_max, n_total))
        ws = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device="cuda")
        off = (-ws.data_ptr()) % 256
        self._ws = ws
        _check(self.L.ecsim_set_workspace(self.h, _P(ws.data_ptr() + off), nbytes), "ecsim_set_workspace")
        return nbytes

    def push_and_moments_host_all(self, qoms, sorted: bool, parts, E, B, dt: float, theta: float, rho, Jhat, M,
                                  accumulate: int = 0):
        """parts: list (one per species) of dicts of host tensors x..q; rho [nsp][nodes], Jhat [nsp][3][nodes] host."""
        f64 = self.torch.float64
        nsp = len(parts)
        n = (_c.c_int64 * nsp)(*[int(p["x"].numel()) for p in parts])
        qm = (_c.c_double * nsp)(*[float(v) for v in qoms])
        cols = []
        for k in ("x", "y", "z", "u", "v", "w", "q"):
            cols.append((_P * nsp)(*[_hptr(p[k], f64) for p in parts]))
        _check(self.L.ecsim_push_and_moments_host_all(self.h, n, qm, 1 if sorted else 0, *cols, _hptr(E, f64),
                                                      _hptr(B, f64), dt, theta, _hptr(rho, f64), _hptr(Jhat, f64),
                                                      _hptr(M, f64), int(accumulate)),
               "ecsim_push_and_moments_host_all")

    # -- knobs and instrumentation -------------------------------------------------------------
    def set_variant(self, variant: int):
        _check(self.L.ecsim_set_variant(self.h, variant), "ecsim_set_variant")

    def set_resort_fraction(self, f: float):
        _check(self.L.ecsim_set_resort_fraction(self.h, f), "ecsim_set_resort_fraction")

    def set_fused_warps(self, w: int):
        _check(self.L.ecsim_set_fused_warps(self.h, w), "ecsim_set_fused_warps")

    def enable_timing(self, on: bool = True):
        _check(self.L.ecsim_enable_timing(self.h, 1 if on else 0), "ecsim_enable_timing")

    def kernel_ms(self) -> float:
        ms = _c.c_float()
        _check(self.L.ecsim_kernel_ms(self.h, _c.byref(ms)), "ecsim_kernel_ms")
        return float(ms.value)

    def launch_count(self) -> int:
        return int(self.L.ecsim_launch_count(self.h))

    def stray_count(self) -> int:
        return int(self.L.ecsim_stray_count(self.h))

    def leaver_count(self) -> int:
        return int(self.L.ecsim_leaver_count(self.h))

    def resort_count(self) -> int:
        return int(self.L.ecsim_resort_count(self.h))

    def probe_fp64(self, iters: int = 4096):
        tf, ms = _c.c_double(), _c.c_float()
        _check(self.L.ecsim_probe_fp64(self.h, iters, _c.byref(tf), _c.byref(ms)), "ecsim_probe_fp64")
        return float(tf.value), float(ms.value)

    def close(self):
        if getattr(self, "h", None):
            self.L.ecsim_destroy(self.h)
            self.h = None
            self._ws = None
            self._keep = {}
            self._resident = {}

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
