"""-m gpu parity at BASELINE.json's FULL sizes for the paths test_gpu_fullsize.py does not reach
("close the parity gap at full size"):

  * configs[4] (64^3, 2 x 33,554,432 particles in seeded RANDOM order): the bucketed two-step counting sort at
    shift = 17, 256 buckets x 65536 tiles of 512 records -- per-cell counts bit-exact against oracle.cells, perm a permutation, the
    seven moved arrays equal in[perm] bit for bit, cells ascending -- then one all-species step compared with the
    oracle on sampled 3x3x3 blocks of cells (same sampling argument as test_gpu_fullsize.py);
  * configs[1] (32^3, 4,194,304 particles): the whole "one step, then 10 consecutive steps, fields fixed" protocol,
    every step compared element by element (moments of the whole grid, every particle).  The oracle is restarted
    from the library's particle state after every step, so 1e-13 is a per-step bound;
  * configs[2] (128^3, 268,435,456 particles), SECOND consecutive step without a re-sort: the stray path at full
    size (millions of particles outside their segment), sampled blocks; then the explicit re-sort of the 134 M
    nearly sorted electrons, checked bit-exactly like the config-4 sort.
"""
from __future__ import annotations

import types

import numpy as np
import pytest
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import MOM_TOL, assert_moments_close, assert_particles_close
from util import PKEYS, grid_of

pytestmark = pytest.mark.gpu


def _need(gb):
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 1e9:
        pytest.skip(f"needs ~{gb} GB of device memory")


def _gen_on_device(cfg):
    dev = torch.device("cuda")
    E, B = wl.gen_fields(cfg, device=dev)
    parts = []
    for s in range(len(cfg.species)):
        p = wl.gen_species(cfg, s, device=dev)
        parts.append({k: p[k].contiguous() for k in PKEYS})
        del p
    torch.cuda.empty_cache()
    return E, B, parts


def _block_cells(cfg, origin):
    i0, j0, k0 = origin
    return [(((i0 + di) % cfg.nx) * cfg.ny + (j0 + dj) % cfg.ny) * cfg.nz + (k0 + dk) % cfg.nz
            for di in range(3) for dj in range(3) for dk in range(3)]


def _inner_nodes(cfg, origin):
    i0, j0, k0 = origin
    return [(((i0 + a) % cfg.nx) * cfg.ny + (j0 + b) % cfg.ny) * cfg.nz + (k0 + c) % cfg.nz
            for a in (1, 2) for b in (1, 2) for c in (1, 2)]


def _check_sort_bit_exact(cfg, ctx, s, part, what):
    """ecsim_sort_particles of species s (arrays `part`, on the device) against oracle.cells: counts bit-exact,
    perm a permutation, moved arrays == in[perm] bit for bit, cells ascending.  Returns the counts (numpy)."""
    n = int(part["x"].numel())
    before = {k: part[k].clone() for k in PKEYS}
    cell_ref, count_ref = oracle.cells(grid_of(cfg), before["x"].cpu().numpy(), before["y"].cpu().numpy(),
                                       before["z"].cpu().numpy())
    count = torch.empty(cfg.cells, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")          # uint32 payload
    ctx.sort_particles(s, count, perm)
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), count_ref), f"{what}: per-cell counts differ from the oracle"
    pm = perm.to(torch.int64) & 0xFFFFFFFF
    seen = torch.zeros(n, dtype=torch.int32, device="cuda")
    seen.index_add_(0, pm, torch.ones(n, dtype=torch.int32, device="cuda"))
    assert bool((seen == 1).all()), f"{what}: perm is not a permutation"
    del seen
    for k in PKEYS:
        assert torch.equal(part[k], before[k][pm]), f"{what}: array {k} is not in[perm]"
    sorted_cells = torch.from_numpy(cell_ref).cuda()[pm]
    assert bool((sorted_cells[1:] >= sorted_cells[:-1]).all()), f"{what}: cells not ascending"
    got_cell = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.cell_index(s, got_cell)
    assert torch.equal(got_cell, sorted_cells.to(torch.int32)), f"{what}: ecsim_cell_index after the sort"
    del before, sorted_cells, got_cell, pm, perm
    torch.cuda.empty_cache()
    return count_ref


def _sampled_block_check(cfg, origin, sel, before_np, after_parts, E, B, rho, J, M, what):
    """Oracle on the particles of a 3x3x3 block of cells (before_np: per species, pre-step host copies; sel: their
    indices in the device arrays) on the full-size grid; compares the block's 8 inner nodes and its particles."""
    nodes = _inner_nodes(cfg, origin)
    En, Bn = E.cpu().numpy(), B.cpu().numpy()
    total = oracle.Moments(cfg.nodes)
    for s, sp in enumerate(cfg.species):
        m = oracle.Moments(cfg.nodes)
        oracle.step(grid_of(cfg), sp.qom, cfg.dt, before_np[s], En, Bn, m)
        got_rho = rho[s, nodes].cpu().numpy()
        got_J = J[s][:, nodes].cpu().numpy()
        assert np.all(np.abs(got_rho - m.rho[nodes]) <= MOM_TOL * m.rho_abs[nodes]), f"{what}: rho species {s}"
        assert np.all(np.abs(got_J - m.J[:, nodes]) <= MOM_TOL * m.J_abs[:, nodes]), f"{what}: Jhat species {s}"
        total.M[nodes] += m.M[nodes]
        total.M_abs[nodes] += m.M_abs[nodes]
        got = {k: after_parts[s][k][sel[s]].cpu().numpy() for k in PKEYS}
        assert_particles_close(got, before_np[s], cfg, f"{what} species {s}")
    got_M = M[nodes].cpu().numpy()
    assert np.all(np.isfinite(got_M))
    err = np.abs(got_M - total.M[nodes])
    assert np.all(err <= MOM_TOL * total.M_abs[nodes]), f"{what}: M worst {err.max():.3e}"


# ------------------------------------------------------------------ configs[4]: random order, full size

CFG4_BLOCKS = [(10, 20, 30), (62, 62, 62), (0, 63, 31), (33, 0, 0)]


def test_config4_full_size_sort_is_bit_exact_and_step_matches_oracle():
    _need(30)
    cfg = wl.config(4)
    E, B, parts = _gen_on_device(cfg)
    nsp = len(cfg.species)
    n_max = max(int(p["x"].numel()) for p in parts)
    assert n_max == 33_554_432
    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace(n_max)
    counts = []
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts[s], sorted=False)
        counts.append(_check_sort_bit_exact(cfg, ctx, s, parts[s], f"config 4 species {s}"))
    # sampled blocks: after the sort cell c of species s owns [start_s[c], start_s[c+1])
    starts = [np.concatenate(([0], np.cumsum(c.astype(np.int64)))) for c in counts]
    sels, befores = {}, {}
    for origin in CFG4_BLOCKS:
        cells = _block_cells(cfg, origin)
        sels[origin] = [torch.cat([torch.arange(int(starts[s][c]), int(starts[s][c + 1]), device="cuda") for c in cells])
                        for s in range(nsp)]
        befores[origin] = [{k: parts[s][k][sels[origin][s]].cpu().numpy().copy() for k in PKEYS} for s in range(nsp)]
    qsum = [float(parts[s]["q"].sum()) for s in range(nsp)]
    rho = torch.full((nsp, cfg.nodes), float("nan"), dtype=torch.float64, device="cuda")
    J = torch.full((nsp, 3, cfg.nodes), float("nan"), dtype=torch.float64, device="cuda")
    M = torch.full((cfg.nodes, 27, 3, 3), float("nan"), dtype=torch.float64, device="cuda")
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
    torch.cuda.synchronize()
    assert ctx.stray_count() == 0
    for origin in CFG4_BLOCKS:
        _sampled_block_check(cfg, origin, sels[origin], befores[origin], parts, E, B, rho, J, M, f"config 4 block {origin}")
    V = cfg.dx * cfg.dy * cfg.dz
    for s in range(nsp):
        assert abs(float(rho[s].sum()) * V - qsum[s]) <= 1e-11 * abs(qsum[s])
    ctx.close()


@pytest.mark.parametrize("n,dims", [(40_000_003, (64, 64, 64)), (134_217_729, (128, 128, 128))], ids=["40M_512_buckets", "134M_1024_buckets"])
def test_sort_of_larger_species_in_arbitrary_order_is_bit_exact(n, dims):
    """The two larger geometries of the record-based sort (sort.cuh: 512 buckets x tiles of 1024 above 2^25 particles, 1024
    buckets x tiles of 2048 above 2^26), which no BASELINE.json config reaches in random order: uniform random particles,
    a ragged last tile and bucket; same bit-exact checks as configs[4]."""
    _need(40 if n > 100_000_000 else 16)
    g = torch.Generator(device="cuda")
    g.manual_seed(n)
    cfg = types.SimpleNamespace(nx=dims[0], ny=dims[1], nz=dims[2], dx=1.0, dy=0.5, dz=2.0, cells=dims[0] * dims[1] * dims[2])
    part = {k: torch.rand(n, dtype=torch.float64, device="cuda", generator=g) for k in PKEYS}
    part["x"] *= cfg.nx * cfg.dx
    part["y"] *= cfg.ny * cfg.dy
    part["z"] *= cfg.nz * cfg.dz
    ctx = pk.Ecsim(*grid_of(cfg), 1)
    ctx.set_workspace(n)
    ctx.load_particles(0, -1.0, part, sorted=False)
    _check_sort_bit_exact(cfg, ctx, 0, part, f"{n} random particles")
    ctx.close()


# ------------------------------------------------------------------ configs[1]: 1 + 10 steps, full size

def _tag_ids(q, q0):
    n = q.shape[0]
    return q0 * (1.0 + np.arange(n) * 2.0 ** -30)


def _ids(q, q0):
    return np.rint((q / q0 - 1.0) * 2.0 ** 30).astype(np.int64)


def test_config1_full_size_eleven_step_protocol():
    """configs[1] as BASELINE.json states it: 32^3, 64 ppc, cell-sorted, one step then 10 more with the fields held
    fixed; whatever re-binning the library needs happens inside the calls.  q carries a particle id in its low bits
    (both sides get the same q) so that particles can be matched after the library's re-sorts."""
    cfg = wl.config(1)
    E, B = wl.gen_fields(cfg)
    grid = grid_of(cfg)
    parts_np = []
    for s, sp in enumerate(cfg.species):
        p = wl.gen_species(cfg, s)
        d = {k: p[k].numpy().copy() for k in PKEYS}
        d["q"] = _tag_ids(d["q"], sp.q_sign * cfg.q_abs)
        parts_np.append(d)
    assert sum(p["x"].shape[0] for p in parts_np) == 4_194_304
    parts_cuda = [{k: torch.from_numpy(p[k]).cuda() for k in PKEYS} for p in parts_np]
    ctx = pk.Ecsim(*grid, 2)
    ctx.set_workspace(max(p["x"].shape[0] for p in parts_np))
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    E_c, B_c = E.cuda(), B.cuda()
    En, Bn = E.numpy(), B.numpy()
    rho = torch.empty(2, cfg.nodes, dtype=torch.float64, device="cuda")
    J = torch.empty(2, 3, cfg.nodes, dtype=torch.float64, device="cuda")
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64, device="cuda")
    strays = 0
    assert cfg.steps == 11
    for step in range(cfg.steps):
        rho.fill_(float("nan")); J.fill_(float("nan")); M.fill_(float("nan"))
        ctx.push_and_moments_all(E_c, B_c, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
        torch.cuda.synchronize()
        strays += ctx.stray_count()
        total = oracle.Moments(cfg.nodes)
        for s, sp in enumerate(cfg.species):
            m = oracle.Moments(cfg.nodes)
            oracle.step(grid, sp.qom, cfg.dt, parts_np[s], En, Bn, m)
            assert_moments_close(rho[s], J[s], None, m, f"config 1 step {step} species {s}")
            total.M += m.M
            total.M_abs += m.M_abs
            del m
        assert_moments_close(None, None, M, total, f"config 1 step {step}")
        del total
        for s, sp in enumerate(cfg.species):
            q0 = sp.q_sign * cfg.q_abs
            got = {k: parts_cuda[s][k].cpu().numpy() for k in PKEYS}
            order = np.argsort(_ids(got["q"], q0))
            got = {k: got[k][order] for k in PKEYS}
            assert np.array_equal(_ids(got["q"], q0), np.arange(got["q"].shape[0]))
            assert_particles_close(got, parts_np[s], cfg, f"config 1 step {step} species {s}")
            parts_np[s] = got            # restart the oracle from the library's state: per-step bound
    assert strays > 0
    ctx.close()


# ------------------------------------------------------------------ configs[2]: second step (strays), then the re-sort

CFG2_BLOCKS = [(40, 77, 3), (126, 126, 126), (0, 0, 0)]


def test_config2_full_size_second_step_strays_and_resort():
    _need(75)
    cfg = wl.config(2)
    E, B, parts = _gen_on_device(cfg)
    nsp = len(cfg.species)
    n_s = [int(p["x"].numel()) for p in parts]
    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace(max(n_s))
    ctx.set_resort_fraction(100.0)                  # step 2 must take the stray path, not a re-sort
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts[s], sorted=True)
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64, device="cuda")
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64, device="cuda")
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64, device="cuda")
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
    torch.cuda.synchronize()
    assert ctx.stray_count() == 0
    # particles that sit in the sampled blocks NOW (after step 1), wherever they are stored
    cell = torch.empty(max(n_s), dtype=torch.int32, device="cuda")
    sels = {o: [] for o in CFG2_BLOCKS}
    for s in range(nsp):
        ctx.cell_index(s, cell)
        torch.cuda.synchronize()
        for o in CFG2_BLOCKS:
            want = torch.tensor(_block_cells(cfg, o), dtype=torch.int32, device="cuda")
            sels[o].append(torch.nonzero(torch.isin(cell[:n_s[s]], want)).flatten())
    del cell
    befores = {o: [{k: parts[s][k][sels[o][s]].cpu().numpy().copy() for k in PKEYS} for s in range(nsp)]
               for o in CFG2_BLOCKS}
    rho.fill_(float("nan")); J.fill_(float("nan")); M.fill_(float("nan"))
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
    torch.cuda.synchronize()
    assert ctx.resort_count() == 0
    assert ctx.stray_count() > 1_000_000             # electrons: ~2 % of 134 M left their cell in step 1
    for o in CFG2_BLOCKS:
        _sampled_block_check(cfg, o, sels[o], befores[o], parts, E, B, rho, J, M, f"config 2 step 2 block {o}")
    del M, befores, sels
    torch.cuda.empty_cache()
    # the re-sort of a nearly sorted 134 M-particle species (nearly_sorted branch of ecsim_sort_particles)
    _check_sort_bit_exact(cfg, ctx, 0, parts[0], "config 2 electrons after two pushes")
    ctx.close()


# ------------------------------------------------------------------ configs[2], resident species: second sort-preserving step

def test_config2_full_size_resident_second_step():
    """configs[2] at full size with RESIDENT species: after one sort-preserving push (3.1 M particles moved
    to their new cells' segments) the second step is compared with the oracle on sampled 3x3x3 blocks; zero strays, zero
    re-sorts, the particle set conserved (ids in the low bits of q), charge conserved on the whole grid."""
    _need(110)
    cfg = wl.config(2)
    E, B, parts = _gen_on_device(cfg)
    nsp = len(cfg.species)
    n_s = [int(p["x"].numel()) for p in parts]
    q0 = [sp.q_sign * cfg.q_abs for sp in cfg.species]
    for s in range(nsp):
        parts[s]["q"] = q0[s] * (1.0 + torch.arange(n_s[s], dtype=torch.float64, device="cuda") * 2.0 ** -30)
    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace(max(n_s))
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts[s], sorted=True)
        ctx.make_resident(s, 0.25)
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64, device="cuda")
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64, device="cuda")
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64, device="cuda")
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
    torch.cuda.synchronize()
    assert ctx.stray_count() == 0 and ctx.leaver_count() > 1_000_000
    # the state after step 1, cell-ordered; the particles that sit in the sampled blocks now
    blocks = [(40, 77, 3), (126, 126, 126)]
    befores, ids = {}, {}
    cur = {k: torch.empty(max(n_s), dtype=torch.float64, device="cuda") for k in PKEYS}
    for s in range(nsp):
        ctx.export_particles(s, cur)
        torch.cuda.synchronize()
        ci = torch.clamp(torch.floor(cur["x"][:n_s[s]] / cfg.dx), 0, cfg.nx - 1).to(torch.int32)
        cj = torch.clamp(torch.floor(cur["y"][:n_s[s]] / cfg.dy), 0, cfg.ny - 1).to(torch.int32)
        ck = torch.clamp(torch.floor(cur["z"][:n_s[s]] / cfg.dz), 0, cfg.nz - 1).to(torch.int32)
        cell = (ci * cfg.ny + cj) * cfg.nz + ck
        del ci, cj, ck
        for o in blocks:
            want = torch.tensor(_block_cells(cfg, o), dtype=torch.int32, device="cuda")
            sel = torch.nonzero(torch.isin(cell, want)).flatten()
            b = {k: cur[k][sel].cpu().numpy().copy() for k in PKEYS}
            befores.setdefault(o, []).append(b)
            ids.setdefault(o, []).append(np.rint((b["q"] / q0[s] - 1.0) * 2.0 ** 30).astype(np.int64))
        del cell
    rho.fill_(float("nan")); J.fill_(float("nan")); M.fill_(float("nan"))
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
    torch.cuda.synchronize()
    assert ctx.stray_count() == 0 and ctx.resort_count() == 0
    V = cfg.dx * cfg.dy * cfg.dz
    after = []
    for s in range(nsp):
        ctx.export_particles(s, cur)
        torch.cuda.synchronize()
        got_id = torch.round((cur["q"][:n_s[s]] / q0[s] - 1.0) * 2.0 ** 30).to(torch.int64)
        order = torch.argsort(got_id)
        assert bool((got_id[order] == torch.arange(n_s[s], device="cuda")).all()), "particle set not conserved"
        after.append({o: {k: cur[k][:n_s[s]][order[torch.from_numpy(ids[o][s]).cuda()]].cpu().numpy() for k in PKEYS} for o in blocks})
        del got_id, order
        qsum = float(cur["q"][:n_s[s]].sum())
        assert abs(float(rho[s].sum()) * V - qsum) <= 1e-11 * abs(qsum)
    En, Bn = E.cpu().numpy(), B.cpu().numpy()
    for o in blocks:
        nodes = _inner_nodes(cfg, o)
        total = oracle.Moments(cfg.nodes)
        for s, sp in enumerate(cfg.species):
            m = oracle.Moments(cfg.nodes)
            oracle.step(grid_of(cfg), sp.qom, cfg.dt, befores[o][s], En, Bn, m)
            assert np.all(np.abs(rho[s, nodes].cpu().numpy() - m.rho[nodes]) <= MOM_TOL * m.rho_abs[nodes])
            assert np.all(np.abs(J[s][:, nodes].cpu().numpy() - m.J[:, nodes]) <= MOM_TOL * m.J_abs[:, nodes])
            total.M[nodes] += m.M[nodes]
            total.M_abs[nodes] += m.M_abs[nodes]
            assert_particles_close(after[s][o], befores[o][s], cfg, f"resident step 2 block {o} species {s}")
        got_M = M[nodes].cpu().numpy()
        assert np.all(np.abs(got_M - total.M[nodes]) <= MOM_TOL * total.M_abs[nodes])
    ctx.close()
