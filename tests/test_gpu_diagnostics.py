"""-m gpu parity of SURVEY §8(f)3: the diagnostic moments (charge density, un-rotated current,
pressure tensor, heat flux; readings R22-R24) -- ecsim_diagnostics against oracle.diagnostics, element by element
within 1e-10 of the per-scalar |addend| sums, for dense species (sorted, with strays, atomic variant) and resident ones."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import MOM_TOL, alloc_moments, from_numpy, gen_all, make_ctx, to_cuda
from util import PKEYS, grid_of, rand_fields, rand_particles, to_numpy

pytestmark = pytest.mark.gpu


def _alloc(nodes):
    nan = float("nan")
    return (torch.full((nodes,), nan, dtype=torch.float64, device="cuda"),
            torch.full((3, nodes), nan, dtype=torch.float64, device="cuda"),
            torch.full((6, nodes), nan, dtype=torch.float64, device="cuda"),
            torch.full((3, nodes), nan, dtype=torch.float64, device="cuda"))


def _check(got, d: "oracle.Diagnostics", what):
    for name, g, ref, norm in (("rho", got[0], d.rho, d.rho_abs), ("J", got[1], d.J, d.J_abs),
                               ("P", got[2], d.P, d.P_abs), ("Q", got[3], d.Q, d.Q_abs)):
        gn = g.cpu().numpy()
        assert np.all(np.isfinite(gn)), f"{what}: {name} not finite"
        err = np.abs(gn - ref)
        assert np.all(err <= MOM_TOL * norm), f"{what}: {name} worst {err.max():.3e} vs {norm.max():.3e}"


@pytest.mark.parametrize("variant", [pk.VARIANT_FUSED, pk.VARIANT_ATOMIC], ids=["fused", "atomic"])
@pytest.mark.parametrize("case", [(0, None), (3, (6, 48, 6)), (2, (5, 6, 7))], ids=["cfg0", "cfg3", "cfg2"])
def test_diagnostics_match_oracle(case, variant):
    idx, scale = case
    cfg = wl.config(idx, scale)
    E, B, parts = gen_all(cfg, shuffle=False)
    ctx = make_ctx(cfg, max(p["n"] for p in parts), variant)
    for s, sp in enumerate(cfg.species):
        pc = to_cuda(parts[s])
        keep = {k: pc[k].clone() for k in PKEYS}
        ctx.load_particles(s, sp.qom, pc, sorted=True)
        got = _alloc(cfg.nodes)
        ctx.diagnostics(s, *got)
        torch.cuda.synchronize()
        d = oracle.Diagnostics(cfg.nodes)
        oracle.diagnostics(grid_of(cfg), to_numpy(parts[s]), d)
        _check(got, d, f"species {s}")
        for k in PKEYS:
            assert torch.equal(pc[k], keep[k])                 # particles untouched
    ctx.close()


def test_diagnostics_after_pushes_strays_and_resident():
    """After two pushes without a re-sort (dense: strays go through the atomic side kernel) and on a resident species."""
    cfg = wl.config(1, (6, 5, 7))
    E, B, parts = gen_all(cfg)
    for resident in (False, True):
        parts_np = [to_numpy(p) for p in parts]
        pcs = [to_cuda(p) for p in parts]
        ctx = make_ctx(cfg, max(p["n"] for p in parts))
        ctx.set_resort_fraction(100.0)
        for s, sp in enumerate(cfg.species):
            ctx.load_particles(s, sp.qom, pcs[s], sorted=True)
            if resident:
                ctx.make_resident(s)
        rho, J, M = alloc_moments(cfg.nodes, 2)
        for _ in range(2):
            ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
        torch.cuda.synchronize()
        for s in range(2):
            if resident:
                cur = {k: torch.empty_like(pcs[s][k]) for k in PKEYS}
                ctx.export_particles(s, cur)
            else:
                cur = pcs[s]
            torch.cuda.synchronize()
            cur_np = {k: cur[k].cpu().numpy() for k in PKEYS}
            got = _alloc(cfg.nodes)
            ctx.diagnostics(s, got[0], got[1], got[2], got[3])
            if not resident:
                assert ctx.stray_count() > 0
            d = oracle.Diagnostics(cfg.nodes)
            oracle.diagnostics(grid_of(cfg), cur_np, d)
            _check(got, d, f"resident={resident} species {s}")
        ctx.close()


def test_diagnostics_null_outputs_and_ragged_grid():
    grid = (4, 5, 3, 0.7, 1.3, 0.9)
    rng = np.random.default_rng(31)
    p = rand_particles(rng, 2500, grid, vscale=0.6)
    pc = to_cuda(from_numpy(p))
    ctx = pk.Ecsim(*grid, 1)
    ctx.set_workspace(2500)
    ctx.load_particles(0, -2.0, pc, sorted=False)
    got = _alloc(60)
    ctx.diagnostics(0, None, None, got[2], None)               # only the pressure tensor
    torch.cuda.synchronize()
    cur = {k: pc[k].cpu().numpy() for k in PKEYS}              # (the call sorted the species in place)
    d = oracle.Diagnostics(60)
    oracle.diagnostics(grid, cur, d)
    assert np.all(np.abs(got[2].cpu().numpy() - d.P) <= MOM_TOL * d.P_abs)
    assert bool(torch.isnan(got[0]).all()) and bool(torch.isnan(got[1]).all()) and bool(torch.isnan(got[3]).all())
    ctx.close()


def test_diagnostics_of_a_resident_species_with_homeless_particles():
    """Segments without slack and hot particles: some particles sit in the overflow list; the diagnostics count them."""
    import dataclasses
    base = wl.config(0, (6, 6, 6))
    hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.0, 0.5)))
    cfg = dataclasses.replace(base, dt=0.2, ppc=40, species=hot)
    E, B, parts = gen_all(cfg)
    pcs = [to_cuda(p) for p in parts]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    ctx.set_resort_fraction(100.0)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, pcs[s], sorted=True)
        ctx.make_resident(s, 0.0)
    rho, J, M = alloc_moments(cfg.nodes, 2)
    for _ in range(2):
        ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
    torch.cuda.synchronize()
    assert ctx.relayout_count() == 0
    for s in range(2):
        cur = {k: torch.empty_like(pcs[s][k]) for k in PKEYS}
        ctx.export_particles(s, cur)
        got = _alloc(cfg.nodes)
        ctx.diagnostics(s, *got)
        torch.cuda.synchronize()
        d = oracle.Diagnostics(cfg.nodes)
        oracle.diagnostics(grid_of(cfg), {k: cur[k].cpu().numpy() for k in PKEYS}, d)
        _check(got, d, f"species {s}")
    ctx.close()
