"""Counter-based seeded generator for the five BASELINE.json configs (recipe: DESIGN.md §"Input recipe").

Everything is a pure function of (seed, species, cell, index-in-cell, stream): any cell's particles
can be regenerated alone, on any torch device, without generating the rest.  The arithmetic is
integer hashing (splitmix64 finaliser) plus elementary float64 functions; nothing of the ECsim
method lives here.

Bit-reproducibility: integer hashing and the uniform variates are bit-identical on every device.
Gaussians go through log/cos/sin, whose last bit may differ between CPU and CUDA libm; tests
therefore always hand the SAME generated tensors to both sides (generate once, copy), never
generate twice on different devices.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence, Tuple

import torch

N_CONFIGS = 5

_M64 = (1 << 64) - 1


def _s64(c: int) -> int:
    """Two's-complement view of a 64-bit constant as a Python int torch accepts for int64."""
    c &= _M64
    return c - (1 << 64) if c >= (1 << 63) else c


_C1 = 0xBF58476D1CE4E5B9
_C2 = 0x94D049BB133111EB
_GOLD = 0x9E3779B97F4A7C15


def _mix_py(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * _C1) & _M64
    z = ((z ^ (z >> 27)) * _C2) & _M64
    return z ^ (z >> 31)


def _key(seed: int, *ids: int) -> int:
    """Stream key from a seed and a tuple of small integers (species, purpose, component...)."""
    k = _mix_py(seed * _GOLD + 0x1234567)
    for i in ids:
        k = _mix_py(k ^ ((i + 1) * _GOLD))
    return k


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _s64(_C1)
    z = (z ^ _lsr(z, 27)) * _s64(_C2)
    return z ^ _lsr(z, 31)


def _uniform(key: int, ctr: torch.Tensor) -> torch.Tensor:
    """53-bit uniform in [0,1) for each int64 counter value."""
    h = _mix(ctr * _s64(_GOLD) + _s64(key))
    return _lsr(h, 11).to(torch.float64) * (2.0 ** -53)


def _gauss_pair(key: int, ctr: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
    """Box-Muller: two independent N(0,1) per counter (uses counters 2*ctr, 2*ctr+1)."""
    u1 = _uniform(key, ctr * 2)
    u2 = _uniform(key, ctr * 2 + 1)
    r = torch.sqrt(-2.0 * torch.log1p(-u1))  # 1-u1 in (0,1]
    t = (2.0 * math.pi) * u2
    return r * torch.cos(t), r * torch.sin(t)


@dataclasses.dataclass(frozen=True)
class Species:
    name: str
    qom: float          # q/m of the species (beta_p = qom*dt/2)
    vth: float          # thermal speed per component
    q_sign: float       # sign of the macro-particle charge
    drift: Tuple[float, float, float] = (0.0, 0.0, 0.0)


@dataclasses.dataclass(frozen=True)
class Config:
    idx: int
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    dt: float
    theta: float
    seed: int
    species: Tuple[Species, ...]
    ppc: int                 # particles per cell per species (peak value for 'harris')
    density: str             # 'uniform' | 'harris'
    q_abs: float             # |q_p| of every macro-particle
    fields: str              # 'fourier' | 'harris' | 'strong'
    e_amp: float             # std of the Gaussian E per node component
    hot_fraction: float = 0.0
    hot_scale: float = 1.0
    shuffled: bool = False   # particle order = seeded random permutation (config 4)
    steps: int = 1

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def nodes(self) -> int:
        return self.cells

    @property
    def lengths(self) -> Tuple[float, float, float]:
        return (self.nx * self.dx, self.ny * self.dy, self.nz * self.dz)


def config(idx: int, scale: Optional[Tuple[int, int, int]] = None) -> Config:
    """The five BASELINE.json configs.  `scale=(nx,ny,nz)` overrides the grid (same recipe,
    smaller box) so that tests can run a config's distributions at a size the oracle finishes."""
    e = Species("electrons", -64.0, 0.05, -1.0)
    i = Species("ions", 1.0, 0.00625, +1.0)
    if idx == 0:
        c = Config(0, "cfg0_8cube", 8, 8, 8, 1.0, 1.0, 1.0, 0.1, 0.5, 0, (e, i), 32, "uniform",
                   1.0 / 32, "fourier", 1e-2)
    elif idx == 1:
        c = Config(1, "cfg1_32cube", 32, 32, 32, 1.0, 1.0, 1.0, 0.1, 0.5, 0, (e, i), 64, "uniform",
                   1.0 / 64, "fourier", 1e-2, steps=11)
    elif idx == 2:
        e2 = dataclasses.replace(e, qom=-256.0)
        c = Config(2, "cfg2_128cube", 128, 128, 128, 1.0, 1.0, 1.0, 0.1, 0.5, 0, (e2, i), 64,
                   "uniform", 1.0 / 64, "fourier", 1e-2)
    elif idx == 3:
        e3 = dataclasses.replace(e, drift=(0.0, 0.0, -0.02))
        i3 = dataclasses.replace(i, drift=(0.0, 0.0, +0.02))
        c = Config(3, "cfg3_harris", 96, 96, 48, 1.0, 1.0, 1.0, 0.1, 0.5, 0, (e3, i3), 256, "harris",
                   1.1 / 256, "harris", 1e-3)
    elif idx == 4:
        e4 = dataclasses.replace(e, vth=0.1)
        i4 = dataclasses.replace(i, vth=0.0125)
        c = Config(4, "cfg4_strongB", 64, 64, 64, 1.0, 1.0, 1.0, 0.1, 0.5, 0, (e4, i4), 128, "uniform",
                   1.0 / 128, "strong", 1e-2, hot_fraction=0.01, hot_scale=10.0, shuffled=True)
    else:
        raise ValueError(f"no config {idx}")
    if scale is not None:
        c = dataclasses.replace(c, nx=scale[0], ny=scale[1], nz=scale[2],
                                name=c.name + "_%dx%dx%d" % tuple(scale))
    return c


def cell_layout(cfg: Config, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """(count[cells], start[cells+1]) int64 for ONE species, cell id = (i*ny + j)*nz + k."""
    if cfg.density == "uniform":
        per_j = torch.full((cfg.ny,), cfg.ppc, dtype=torch.int64)
    elif cfg.density == "harris":
        # n(y) = sech^2((y - Ly/2)/lambda) + 0.1, lambda = 4 cells, sampled at cell centres,
        # peak (n = 1.1) <-> cfg.ppc particles per cell
        yj = (torch.arange(cfg.ny, dtype=torch.float64) + 0.5) * cfg.dy
        n = 1.0 / torch.cosh((yj - 0.5 * cfg.ny * cfg.dy) / (4.0 * cfg.dy)) ** 2 + 0.1
        per_j = torch.clamp(torch.round(cfg.ppc * n / 1.1), min=1).to(torch.int64)
    else:
        raise ValueError(cfg.density)
    count = per_j.view(1, cfg.ny, 1).expand(cfg.nx, cfg.ny, cfg.nz).reshape(-1).contiguous()
    start = torch.zeros(cfg.cells + 1, dtype=torch.int64)
    start[1:] = torch.cumsum(count, 0)
    return count.to(device), start.to(device)


def _node_coords(cfg: Config, device):
    i = torch.arange(cfg.nx, dtype=torch.float64, device=device) * cfg.dx
    j = torch.arange(cfg.ny, dtype=torch.float64, device=device) * cfg.dy
    k = torch.arange(cfg.nz, dtype=torch.float64, device=device) * cfg.dz
    return i, j, k


def gen_fields(cfg: Config, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """E^{n+theta}, B^n at nodes, each float64 [3][nodes], node = (i*ny + j)*nz + k."""
    nx, ny, nz = cfg.nx, cfg.ny, cfg.nz
    nodes = cfg.nodes
    node = torch.arange(nodes, dtype=torch.int64, device=device)
    E = torch.empty(3, nodes, dtype=torch.float64, device=device)
    for c in range(3):
        g, _ = _gauss_pair(_key(cfg.seed, 100, c), node)
        E[c] = cfg.e_amp * g
    B = torch.zeros(3, nx, ny, nz, dtype=torch.float64, device=device)
    xi, yj, zk = _node_coords(cfg, device)
    Lx, Ly, Lz = cfg.lengths
    if cfg.fields == "fourier":
        # B = (0,0,1) + (1e-2/9) * sum_axis sum_{m=1..3} sin(2 pi m r_a / L_a + phase)
        for c in range(3):
            for a, (r, L, shape) in enumerate(((xi, Lx, (nx, 1, 1)), (yj, Ly, (1, ny, 1)),
                                               (zk, Lz, (1, 1, nz)))):
                acc = torch.zeros_like(r)
                for m in (1, 2, 3):
                    ph = 2.0 * math.pi * float(_uniform(_key(cfg.seed, 101, c, a, m),
                                                        torch.zeros(1, dtype=torch.int64))[0])
                    acc = acc + torch.sin((2.0 * math.pi * m / L) * r + ph)
                B[c] += (1e-2 / 9.0) * acc.view(shape)
        B[2] += 1.0
    elif cfg.fields == "harris":
        # B_x = tanh((y - Ly/2)/lambda), lambda = 4 cells; 5 % guide field along z
        B[0] += torch.tanh((yj - 0.5 * Ly) / (4.0 * cfg.dy)).view(1, ny, 1)
        B[2] += 0.05
    elif cfg.fields == "strong":
        # |B| log-uniform in [0.1, 10] per node, direction isotropic
        u = _uniform(_key(cfg.seed, 102, 0), node)
        mu = 2.0 * _uniform(_key(cfg.seed, 102, 1), node) - 1.0
        ph = 2.0 * math.pi * _uniform(_key(cfg.seed, 102, 2), node)
        mag = torch.pow(torch.tensor(10.0, dtype=torch.float64, device=device), 2.0 * u - 1.0)
        s = torch.sqrt(torch.clamp(1.0 - mu * mu, min=0.0))
        B = torch.stack((mag * s * torch.cos(ph), mag * s * torch.sin(ph), mag * mu)).view(3, nx, ny, nz)
    else:
        raise ValueError(cfg.fields)
    return E, B.reshape(3, nodes).contiguous()


def gen_species(cfg: Config, s: int, device="cpu", cells: Optional[Sequence[int]] = None,
                shuffle: Optional[bool] = None) -> dict:
    """Particles of species `s`: dict of float64 tensors x,y,z,u,v,w,q (SoA) plus int64 `cell`
    (the cell each particle was sampled in) and `n`.  `cells` restricts generation to the given
    cell ids (cell-major order, never shuffled).  Full sets are cell-sorted unless cfg.shuffled."""
    sp = cfg.species[s]
    count, start = cell_layout(cfg, device)
    if cells is None:
        cell = torch.repeat_interleave(torch.arange(cfg.cells, dtype=torch.int64, device=device), count)
        idx = torch.arange(cell.numel(), dtype=torch.int64, device=device) - start[cell]
    else:
        cid = torch.as_tensor(cells, dtype=torch.int64, device=device)
        cnt = count[cid]
        cell = torch.repeat_interleave(cid, cnt)
        first = torch.cumsum(cnt, 0) - cnt
        idx = torch.arange(cell.numel(), dtype=torch.int64, device=device) - torch.repeat_interleave(first, cnt)
    ctr = cell * 1024 + idx          # ppc <= 1023 for every config
    ck = cell % cfg.nz
    cj = (cell // cfg.nz) % cfg.ny
    ci = cell // (cfg.nz * cfg.ny)
    out = {}
    for name, c0, d, stream in (("x", ci, cfg.dx, 0), ("y", cj, cfg.dy, 1), ("z", ck, cfg.dz, 2)):
        out[name] = (c0.to(torch.float64) + _uniform(_key(cfg.seed, s, stream), ctr)) * d
    g0, g1 = _gauss_pair(_key(cfg.seed, s, 3), ctr)
    g2, _ = _gauss_pair(_key(cfg.seed, s, 4), ctr)
    scale = torch.full_like(g0, sp.vth)
    if cfg.hot_fraction > 0.0:
        hot = _uniform(_key(cfg.seed, s, 5), ctr) < cfg.hot_fraction
        scale = torch.where(hot, scale * cfg.hot_scale, scale)
    out["u"] = sp.drift[0] + scale * g0
    out["v"] = sp.drift[1] + scale * g1
    out["w"] = sp.drift[2] + scale * g2
    out["q"] = torch.full_like(g0, sp.q_sign * cfg.q_abs)
    out["cell"] = cell
    do_shuffle = cfg.shuffled if shuffle is None else shuffle
    if do_shuffle and cells is None:
        # seeded permutation: order particles by a hash of their counter (stable sort)
        h = _mix(ctr * _s64(_GOLD) + _s64(_key(cfg.seed, s, 6)))
        perm = torch.sort(h, stable=True).indices
        for k in list(out.keys()):
            out[k] = out[k][perm].contiguous()
        out["perm"] = perm
    out["n"] = int(cell.numel())
    return out
