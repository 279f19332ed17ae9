"""Slab domain decomposition (paper_2603_16624_b200/slabs.py) WITHOUT a GPU:
  * all ranks in one process (LocalRing): even and uneven splits, world = 1 (self-exchange = the periodic wrap), 3 steps
    with halo add + migration after every step, against the single-domain oracle;
  * two real ranks over torch.distributed / gloo (the N > 1 path the tier asks to cover on CPU).
The per-slab compute engine here is the CPU oracle on the slab's local grid; tests/test_gpu_slabs.py runs libecpush."""
from __future__ import annotations

import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

import workloads as wl
from paper_2603_16624_b200.slabs import PKEYS, LocalRing, SlabGrid
from slab_driver import (check_against_global, global_reference_step, oracle_engine, tagged_global_particles)
from util import grid_of

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_local_ring(cfg, world, steps, engine):
    E, B = wl.gen_fields(cfg)
    gparts = tagged_global_particles(cfg)
    ref = [{k: p[k].numpy().copy() for k in PKEYS} for p in gparts]
    grids = [SlabGrid(*grid_of(cfg), world, r) for r in range(world)]
    ring = LocalRing(world)
    parts = [[g.split_particles(p) for p in gparts] for g in grids]
    fields = [(g.local_fields(E), g.local_fields(B)) for g in grids]
    nsp = len(cfg.species)
    moved = 0
    for step in range(steps):
        out = [engine(grids[r], cfg, parts[r], *fields[r]) for r in range(world)]
        halos = [grids[r].halo_planes(*out[r]) for r in range(world)]
        got = ring.shift_right(halos)
        for r in range(world):
            grids[r].add_halo(got[r], *out[r])
        for s in range(nsp):
            packs = [grids[r].leavers(parts[r][s], cfg.dt) for r in range(world)]
            fl, fr = ring.exchange([p[1] for p in packs], [p[2] for p in packs])
            moved += sum(int(p[1].shape[1] + p[2].shape[1]) for p in packs)
            for r in range(world):
                parts[r][s] = grids[r].merge(parts[r][s], packs[r][0], fl[r], fr[r])
        per, total = global_reference_step(cfg, ref, E, B)
        check_against_global(cfg, grids, [grids[r].owned(out[r][0], 1) for r in range(world)],
                             [grids[r].owned(out[r][1], 2) for r in range(world)],
                             [grids[r].owned(out[r][2], 0) for r in range(world)],
                             [[grids[r].to_global(parts[r][s]) for s in range(nsp)] for r in range(world)], ref, per, total,
                             f"world {world} step {step}")
    return moved


@pytest.mark.parametrize("world", [1, 2, 3])
def test_slabs_in_one_process_match_the_single_domain_oracle(world):
    import dataclasses
    base = wl.config(0, (8, 5, 4))
    hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.5, 0.5)))   # plenty of slab crossings
    cfg = dataclasses.replace(base, species=hot, ppc=12, dt=0.2)
    moved = run_local_ring(cfg, world, 3, oracle_engine)
    assert moved > 50


def test_slab_grid_bookkeeping():
    g = [SlabGrid(10, 3, 2, 0.5, 1.0, 1.0, 3, r) for r in range(3)]
    assert [(s.i0, s.i1) for s in g] == [(0, 3), (3, 6), (6, 10)]
    assert g[0].left == 2 and g[0].right == 1 and g[0].nxl_left == 4
    assert g[2].local_dims[:3] == (6, 3, 2)
    F = torch.arange(3 * 60, dtype=torch.float64).reshape(3, 60)
    Fl = g[2].local_fields(F).reshape(3, 6, 6)
    G = F.reshape(3, 10, 6)
    for l, gi in enumerate([6, 7, 8, 9, 0, 5]):                 # planes 0..nxl = 6..9, 0 (right halo); plane nxl+1 = 5 (left)
        assert torch.equal(Fl[:, l], G[:, gi])
    with pytest.raises(ValueError):
        SlabGrid(2, 3, 3, 1.0, 1.0, 1.0, 3, 0)


def test_a_particle_that_ends_two_planes_out_is_refused_not_misrouted():
    """ECsim steps beyond the CFL limit, so a particle can cross more than one cell plane in a step.  Ending ONE plane
    outside the slab after several cells is fine; ending two planes out would look like a leaver to the other side."""
    g = SlabGrid(12, 2, 2, 0.5, 1.0, 1.0, 3, 1)                 # nxl = 4: slab planes 0..3, right ghost 4, left ghost 5
    dt = 0.25

    def one(x_old, u):
        x_new = (x_old + dt * u) % ((g.nxl + 2) * g.dx)         # the push on the periodic local grid
        p = {k: torch.zeros(1, dtype=torch.float64) for k in PKEYS}
        p["x"][0], p["u"][0] = x_new, u
        return p

    # three cells to the right, ending in the right ghost plane: a legitimate right leaver, in the receiver's frame
    stay, pr, pl = g.leavers(one(0.6, 6.4), dt)                 # 0.6 -> 2.2 = plane 4
    assert not bool(stay[0]) and pr.shape[1] == 1 and pl.shape[1] == 0 and abs(float(pr[0, 0]) - 0.2) < 1e-12
    stay, pr, pl = g.leavers(one(0.1, -1.2), dt)                # 0.1 -> -0.2 = plane 5 (left ghost)
    assert pl.shape[1] == 1 and abs(float(pl[0, 0]) - (g.nxl_left * g.dx - 0.2)) < 1e-12
    # from the last plane by +2 planes: lands in the LEFT ghost plane with u > 0
    with pytest.raises(RuntimeError, match="nearest neighbours"):
        g.leavers(one(1.9, 3.0), dt)                            # 1.9 -> 2.65 = plane 5
    with pytest.raises(RuntimeError, match="nearest neighbours"):
        g.leavers(one(1.9, 3.0))                                # the sign check needs no dt
    # from the first plane by -2 planes: lands in the RIGHT ghost plane with u < 0
    with pytest.raises(RuntimeError, match="nearest neighbours"):
        g.leavers(one(0.1, -2.8))                               # 0.1 -> -0.6 = plane 4
    # a whole period of the local grid and more: the position and the sign look innocent, the origin does not
    with pytest.raises(RuntimeError, match="nearest neighbours"):
        g.leavers(one(0.2, 13.0), dt)                           # 0.2 -> 3.45 -> wraps to 0.45: "stayed"
    # a thermal species with vth dt / dx > 1: some particle always ends too far out
    rng = torch.Generator().manual_seed(3)
    n = 4000
    p = {k: torch.zeros(n, dtype=torch.float64) for k in PKEYS}
    x_old = torch.rand(n, generator=rng, dtype=torch.float64) * g.nxl * g.dx
    p["u"] = torch.randn(n, generator=rng, dtype=torch.float64) * (1.5 * g.dx / dt)
    p["x"] = (x_old + dt * p["u"]) % ((g.nxl + 2) * g.dx)
    with pytest.raises(RuntimeError, match="nearest neighbours"):
        g.leavers(p, dt)


WORKER = r'''
import os, sys
root = os.environ["ECPUSH_ROOT"]
sys.path[:0] = [root, os.path.join(root, "tests")]
import dataclasses
import numpy as np, torch, torch.distributed as dist
import workloads as wl
from paper_2603_16624_b200.slabs import PKEYS, DistRing, SlabGrid
from slab_driver import check_against_global, global_reference_step, oracle_engine, tagged_global_particles
from util import grid_of

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
base = wl.config(0, (8, 5, 4))
hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.5, 0.5)))
cfg = dataclasses.replace(base, species=hot, ppc=12, dt=0.2)
E, B = wl.gen_fields(cfg)
gparts = tagged_global_particles(cfg)
grid = SlabGrid(*grid_of(cfg), world, rank)
ring = DistRing()
parts = [grid.split_particles(p) for p in gparts]
El, Bl = grid.local_fields(E), grid.local_fields(B)
ref = [{k: p[k].numpy().copy() for k in PKEYS} for p in gparts]
nsp = len(cfg.species)
for step in range(3):
    rho, J, M = oracle_engine(grid, cfg, parts, El, Bl)
    grid.add_halo(ring.shift_right(grid.halo_planes(rho, J, M)), rho, J, M)
    for s in range(nsp):
        stay, pr, pl = grid.leavers(parts[s], cfg.dt)
        fl, fr = ring.exchange(pr, pl)
        parts[s] = grid.merge(parts[s], stay, fl, fr)
    mine = (grid.owned(rho, 1).clone(), grid.owned(J, 2).clone(), grid.owned(M, 0).clone(),
            [{k: v.numpy() for k, v in grid.to_global(parts[s]).items()} for s in range(nsp)])
    gathered = [None] * world
    dist.gather_object(mine, gathered if rank == 0 else None, dst=0)
    if rank == 0:
        grids = [SlabGrid(*grid_of(cfg), world, r) for r in range(world)]
        per, total = global_reference_step(cfg, ref, E, B)
        check_against_global(cfg, grids, [g[0] for g in gathered], [g[1] for g in gathered], [g[2] for g in gathered],
                             [g[3] for g in gathered], ref, per, total, f"gloo step {step}")
dist.barrier()
dist.destroy_process_group()
print(f"rank {rank} ok")
'''


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_gloo_ranks_halo_add_and_migration(tmp_path):
    script = tmp_path / "slab_worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, ECPUSH_ROOT=ROOT)
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
         "--master-port", str(_free_port()), str(script)], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "rank 0 ok" in out.stdout and "rank 1 ok" in out.stdout
