"""-m gpu parity on the WHOLE grid at BASELINE.json's full sizes for the two configurations whose oracle run is cheap
enough: configs[3] (Harris sheet, 96x96x48 cells, 37.6 M particles, ~25 s of single-thread oracle)
and configs[4] (strong field, 64^3 cells, 67.1 M particles given in random order, ~45 s).  Every node of rho, Jhat and M
and every particle is compared with the oracle, not sampled blocks (test_gpu_fullsize.py / _more.py keep the sampled
checks, which remain the only feasible ones for the 268 M particles of configs[2]).

configs[4]: the library's counting sort runs first (its bit-exactness at this size is test_gpu_fullsize_more.py's
business); the sorted arrays are then the input of BOTH sides, so that particles can be compared index by index.
"""
from __future__ import annotations

import numpy as np
import pytest
import torch

import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import alloc_moments, assert_moments_close, assert_particles_close, oracle_run
from util import PKEYS, grid_of

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx", [3, 4])
def test_whole_grid_parity_at_full_size(idx):
    free, _ = torch.cuda.mem_get_info()
    if free < 30e9:
        pytest.skip("needs ~30 GB of device memory")
    cfg = wl.config(idx)
    dev = torch.device("cuda")
    nsp = len(cfg.species)
    E, B = wl.gen_fields(cfg, device=dev)
    parts = []
    for s in range(nsp):
        p = wl.gen_species(cfg, s, device=dev)
        parts.append({k: p[k].contiguous() for k in PKEYS})
        del p
    n_s = [int(p["x"].numel()) for p in parts]
    assert sum(n_s) > 30_000_000                                  # the full-size workload, not a scaled one
    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace(max(n_s))
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts[s], sorted=not cfg.shuffled)
        if cfg.shuffled:
            ctx.sort_particles(s)                                 # in place: parts[s] now holds the cell-sorted species
    torch.cuda.synchronize()
    before = [{k: parts[s][k].cpu().numpy().copy() for k in PKEYS} for s in range(nsp)]
    rho, J, M = alloc_moments(cfg.nodes, nsp)
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
    torch.cuda.synchronize()
    assert ctx.stray_count() == 0
    (total, per_species), = oracle_run(cfg, before, E, B)         # advances `before` in place
    for s in range(nsp):
        assert_moments_close(rho[s], J[s], None, per_species[s], f"configs[{idx}] whole grid, species {s}")
        got = {k: parts[s][k].cpu().numpy() for k in PKEYS}
        assert np.array_equal(got["q"], before[s]["q"])
        assert_particles_close(got, before[s], cfg, f"configs[{idx}] whole grid, species {s}")
    assert_moments_close(None, None, M, total, f"configs[{idx}] whole grid")
    ctx.close()
