"""-m gpu: the slab-decomposed run (paper_2603_16624_b200/slabs.py) with libecpush as the per-slab engine, against the
single-domain oracle.  One GPU: the slabs of a LocalRing are stepped one after the other, each with its own context on
its local (nxl + 2 planes) periodic grid; halo add and migration run on device tensors (the same code a DistRing drives
over NCCL with one rank per GPU)."""
from __future__ import annotations

import dataclasses

import pytest
import torch

import paper_2603_16624_b200 as pk
import workloads as wl
from paper_2603_16624_b200.slabs import PKEYS, LocalRing, SlabGrid
from slab_driver import check_against_global, global_reference_step, tagged_global_particles
from util import grid_of

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world,m_layout", [(2, pk.M_27), (3, pk.M_27)])
def test_slab_decomposed_steps_match_single_domain_oracle(world, m_layout):
    base = wl.config(0, (9, 5, 4))
    hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.5, 0.5)))
    cfg = dataclasses.replace(base, species=hot, ppc=24, dt=0.2)
    nsp = len(cfg.species)
    E, B = wl.gen_fields(cfg)
    gparts = tagged_global_particles(cfg)
    ref = [{k: p[k].numpy().copy() for k in PKEYS} for p in gparts]
    grids = [SlabGrid(*grid_of(cfg), world, r) for r in range(world)]
    ring = LocalRing(world)
    parts = [[{k: v.cuda() for k, v in g.split_particles(p).items()} for p in gparts] for g in grids]
    fields = [(g.local_fields(E).cuda(), g.local_fields(B).cuda()) for g in grids]
    ctxs = []
    for g in grids:
        c = pk.Ecsim(*g.local_dims, nsp)
        c.set_workspace(2 * sum(int(p["x"].numel()) for p in gparts))      # room for every migration
        ctxs.append(c)
    moved = 0
    for step in range(3):
        out = []
        for r, g in enumerate(grids):
            for s, sp in enumerate(cfg.species):
                ctxs[r].load_particles(s, sp.qom, parts[r][s], sorted=False)   # arrivals were appended: bin again
            rho = torch.full((nsp, g.local_nodes), float("nan"), dtype=torch.float64, device="cuda")
            J = torch.full((nsp, 3, g.local_nodes), float("nan"), dtype=torch.float64, device="cuda")
            M = torch.full((g.local_nodes, 243), float("nan"), dtype=torch.float64, device="cuda")
            ctxs[r].push_and_moments_all(fields[r][0], fields[r][1], cfg.dt, cfg.theta, rho, J, M)
            out.append((rho, J, M))
        torch.cuda.synchronize()
        got = ring.shift_right([grids[r].halo_planes(*out[r]) for r in range(world)])
        for r in range(world):
            grids[r].add_halo(got[r], *out[r])
        for s in range(nsp):
            packs = [grids[r].leavers(parts[r][s], cfg.dt) for r in range(world)]
            fl, fr = ring.exchange([p[1] for p in packs], [p[2] for p in packs])
            moved += sum(int(p[1].shape[1] + p[2].shape[1]) for p in packs)
            for r in range(world):
                parts[r][s] = grids[r].merge(parts[r][s], packs[r][0], fl[r], fr[r])
        per, total = global_reference_step(cfg, ref, E, B)
        check_against_global(
            cfg, grids, [grids[r].owned(out[r][0], 1).cpu() for r in range(world)],
            [grids[r].owned(out[r][1], 2).cpu() for r in range(world)], [grids[r].owned(out[r][2], 0).cpu() for r in range(world)],
            [[{k: v.cpu().numpy() for k, v in grids[r].to_global(parts[r][s]).items()} for s in range(nsp)] for r in range(world)],
            ref, per, total, f"world {world} step {step}")
    assert moved > 100
    for c in ctxs:
        c.close()
