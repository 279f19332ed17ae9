"""-m gpu parity tests: libecpush (CUDA, through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Sizes: what the oracle finishes in seconds, spanning many
cells/warps/CTAs and ragged tails.  Full-size sampled checks live in test_gpu_fullsize.py."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import (alloc_moments, assert_moments_close, assert_particles_close, from_numpy, gen_all,
                      make_ctx, oracle_run, to_cuda)
from util import PKEYS, grid_of, rand_fields, rand_particles, to_numpy

pytestmark = pytest.mark.gpu

# (config index, grid override): every BASELINE.json config's distributions at an oracle-sized box
CASES = {
    "cfg0_full": (0, None),
    "cfg1_16cube": (1, (16, 16, 16)),
    "cfg2_12x16x20": (2, (12, 16, 20)),
    "cfg3_harris_6x96x6": (3, (6, 96, 6)),
    "cfg4_strong_12cube": (4, (12, 12, 12)),
}


def run_species_calls(ctx, cfg, parts_cuda, E, B, sorted_hint):
    """Per-species ecsim_push_and_moments calls; M accumulated over species (L59), rho/Jhat per species."""
    nsp = len(cfg.species)
    rho, J, M = alloc_moments(cfg.nodes, nsp)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=sorted_hint)
    for s in range(nsp):
        ctx.push_and_moments(s, E, B, cfg.dt, cfg.theta, rho[s], J[s], M, accumulate=(pk.ACC_M_ONLY if s > 0 else pk.ACC_NONE))
    torch.cuda.synchronize()
    return rho, J, M


# ------------------------------------------------------------------ integer work: bit-exact

@pytest.mark.parametrize("case", ["cfg0_full", "cfg3_harris_6x96x6", "cfg4_strong_12cube"])
def test_cell_index_and_counting_sort_are_bit_exact(case):
    idx, scale = CASES[case]
    cfg = wl.config(idx, scale)
    part = wl.gen_species(cfg, 0, shuffle=True)
    pn = to_numpy(part)
    cell_ref, count_ref = oracle.cells(grid_of(cfg), pn["x"], pn["y"], pn["z"])
    n = part["n"]
    ctx = make_ctx(cfg, n)
    pc = to_cuda(part)
    ctx.load_particles(0, cfg.species[0].qom, pc, sorted=False)
    cell = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.cell_index(0, cell)
    assert np.array_equal(cell.cpu().numpy(), cell_ref)
    count = torch.empty(cfg.cells, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")   # uint32 payload
    ctx.sort_particles(0, count, perm)
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), count_ref)
    pm = perm.cpu().numpy().astype(np.int64) & 0xFFFFFFFF
    assert np.array_equal(np.sort(pm), np.arange(n))                     # a permutation
    for k in PKEYS:
        assert np.array_equal(pc[k].cpu().numpy(), pn[k][pm]), k        # arrays moved exactly
    assert np.all(np.diff(cell_ref[pm]) >= 0)                            # grouped by cell, ascending
    ctx.cell_index(0, cell)
    assert np.array_equal(cell.cpu().numpy(), cell_ref[pm])
    ctx.close()


@pytest.mark.parametrize("n,dims", [(1, (3, 4, 5)), (31, (3, 4, 5)), (1024, (5, 7, 3)), (1025, (5, 7, 3)), (2047, (16, 9, 11)),
                                    (8193, (2, 2, 2)), (300001, (40, 33, 21)), (2500000, (24, 20, 28))])
@pytest.mark.parametrize("want_perm", [True, False], ids=["perm", "noperm"])
def test_sort_of_arbitrary_order_tile_and_bucket_tails(n, dims, want_perm):
    """The record-based two-step move (sort.cuh) at sizes around its tile (1024 records) and bucket (2^shift places)
    boundaries: one ragged tile, several buckets with a partial last one, dense and sparse cells, with and without the
    permutation output; then a second sort of the now sorted species (the near-identity path)."""
    rng = np.random.default_rng(n)
    grid = (*dims, 0.5, 1.25, 2.0)
    cells = dims[0] * dims[1] * dims[2]
    pn = rand_particles(rng, n, grid)
    cell_ref, count_ref = oracle.cells(grid, pn["x"], pn["y"], pn["z"])
    ctx = pk.Ecsim(*grid, 1)
    ctx.set_workspace(n)
    pc = {k: torch.from_numpy(pn[k]).cuda() for k in PKEYS}
    ctx.load_particles(0, -3.0, pc, sorted=False)
    count = torch.empty(cells, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda") if want_perm else None
    ctx.sort_particles(0, count, perm)
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), count_ref)
    got = {k: pc[k].cpu().numpy() for k in PKEYS}
    if want_perm:
        pm = perm.cpu().numpy().astype(np.int64) & 0xFFFFFFFF
        assert np.array_equal(np.sort(pm), np.arange(n))
        for k in PKEYS:
            assert np.array_equal(got[k], pn[k][pm]), k
    else:
        # without the permutation: the multiset of particles is unchanged (q carries distinct random values)
        order_in, order_out = np.argsort(pn["q"], kind="stable"), np.argsort(got["q"], kind="stable")
        for k in PKEYS:
            assert np.array_equal(got[k][order_out], pn[k][order_in]), k
    cell_sorted, _ = oracle.cells(grid, got["x"], got["y"], got["z"])
    assert np.all(np.diff(cell_sorted) >= 0)
    # a second sort moves nothing across cells and keeps every particle
    ctx.sort_particles(0, count, None)
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), count_ref)
    again = {k: pc[k].cpu().numpy() for k in PKEYS}
    cell_again, _ = oracle.cells(grid, again["x"], again["y"], again["z"])
    assert np.array_equal(cell_again, cell_sorted)
    assert np.array_equal(np.sort(again["q"]), np.sort(pn["q"]))
    ctx.close()


# ------------------------------------------------------------------ the hot path, all five configs

@pytest.mark.parametrize("variant", [pk.VARIANT_FUSED, pk.VARIANT_ATOMIC], ids=["fused", "atomic"])
@pytest.mark.parametrize("case", list(CASES))
def test_push_and_moments_match_oracle(case, variant):
    idx, scale = CASES[case]
    if variant == pk.VARIANT_ATOMIC and case not in ("cfg0_full", "cfg4_strong_12cube"):
        pytest.skip("the atomic prior-art variant is covered on two configs")
    cfg = wl.config(idx, scale)
    E, B, parts = gen_all(cfg)
    parts_np = [to_numpy(p) for p in parts]
    parts_cuda = [to_cuda(p) for p in parts]
    n_max = max(p["n"] for p in parts)
    ctx = make_ctx(cfg, n_max, variant)
    perms = None
    if cfg.shuffled and variant == pk.VARIANT_FUSED:
        # config 4: particles arrive in random order; sort explicitly to learn the permutation
        perms = []
        for s, sp in enumerate(cfg.species):
            ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=False)
            perm = torch.empty(parts[s]["n"], dtype=torch.int32, device="cuda")
            ctx.sort_particles(s, None, perm)
            perms.append(perm.cpu().numpy().astype(np.int64) & 0xFFFFFFFF)
        rho, J, M = alloc_moments(cfg.nodes, len(cfg.species))
        for s in range(len(cfg.species)):
            ctx.push_and_moments(s, E, B, cfg.dt, cfg.theta, rho[s], J[s], M, accumulate=(pk.ACC_M_ONLY if s > 0 else pk.ACC_NONE))
        torch.cuda.synchronize()
    else:
        rho, J, M = run_species_calls(ctx, cfg, parts_cuda, E, B, sorted_hint=not cfg.shuffled)
    if variant == pk.VARIANT_FUSED:
        assert ctx.stray_count() == 0
    (total, per_species), = oracle_run(cfg, parts_np, E, B)
    for s in range(len(cfg.species)):
        ref = parts_np[s] if perms is None else {k: parts_np[s][k][perms[s]] for k in PKEYS}
        assert_particles_close(parts_cuda[s], ref, cfg, f"{case} species {s}")
        assert_moments_close(rho[s], J[s], None, per_species[s], f"{case} species {s}")
    assert_moments_close(None, None, M, total, case)
    ctx.close()


def test_all_species_call_matches_oracle():
    cfg = wl.config(0)
    E, B, parts = gen_all(cfg)
    parts_np = [to_numpy(p) for p in parts]
    parts_cuda = [to_cuda(p) for p in parts]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    rho, J, M = alloc_moments(cfg.nodes, 2)
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
    torch.cuda.synchronize()
    (total, per_species), = oracle_run(cfg, parts_np, E, B)
    for s in range(2):
        assert_particles_close(parts_cuda[s], parts_np[s], cfg, f"species {s}")
        assert_moments_close(rho[s], J[s], None, per_species[s], f"species {s}")
    assert_moments_close(None, None, M, total, "all species")
    # accumulate = 1 on top of existing arrays doubles them
    parts_cuda2 = [to_cuda(p) for p in parts]
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda2[s], sorted=True)
    rho1 = rho.clone()
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_M_ONLY)
    torch.cuda.synchronize()
    total.M *= 2
    total.M_abs *= 2
    assert_moments_close(None, None, M, total, "accumulate M only")
    assert torch.equal(rho, rho1)                       # rho overwritten with the same values
    parts_cuda3 = [to_cuda(p) for p in parts]
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda3[s], sorted=True)
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_ALL)
    torch.cuda.synchronize()
    for s in range(2):
        per_species[s].rho *= 2
        per_species[s].rho_abs *= 2
        per_species[s].J *= 2
        per_species[s].J_abs *= 2
        assert_moments_close(rho[s], J[s], None, per_species[s], f"accumulate all, species {s}")
    ctx.close()


def test_fused_step_is_bitwise_reproducible():
    """The fused path has no atomics: runs on identical inputs give bit-identical outputs (race probe;
    compute-sanitizer is closed on this GPU pool)."""
    cfg = wl.config(3, (6, 24, 6))
    E, B, parts = gen_all(cfg)
    outs = []
    for _ in range(3):
        parts_cuda = [to_cuda(p) for p in parts]
        ctx = make_ctx(cfg, max(p["n"] for p in parts))
        for s, sp in enumerate(cfg.species):
            ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
        rho, J, M = alloc_moments(cfg.nodes, 2)
        ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
        torch.cuda.synchronize()
        assert ctx.stray_count() == 0
        outs.append((rho, J, M, parts_cuda))
        ctx.close()
    for other in outs[1:]:
        for a, b in zip(outs[0][:3], other[:3]):
            assert torch.equal(a, b)
        for s in range(2):
            for k in PKEYS:
                assert torch.equal(outs[0][3][s][k], other[3][s][k])


# ------------------------------------------------------------------ several steps: strays and re-sorts

def _tag_ids(part_np, q0):
    """Carry a particle id in the low bits of q (both sides get the same q)."""
    n = part_np["q"].shape[0]
    part_np["q"] = q0 * (1.0 + np.arange(n) * 2.0 ** -30)


def _ids(q, q0):
    return np.rint((q / q0 - 1.0) * 2.0 ** 30).astype(np.int64)


@pytest.mark.parametrize("resort_fraction", [0.01, 100.0], ids=["resort", "strays_only"])
def test_eleven_steps_fields_fixed(resort_fraction):
    """Config 1's protocol (one step, then 10 more with fields held fixed) on a 10x8x12 box."""
    cfg = wl.config(1, (10, 8, 12))
    E, B, parts = gen_all(cfg)
    parts_np = [to_numpy(p) for p in parts]
    for s, sp in enumerate(cfg.species):
        _tag_ids(parts_np[s], sp.q_sign * cfg.q_abs)
    parts_cuda = [to_cuda(from_numpy(p)) for p in parts_np]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    ctx.set_resort_fraction(resort_fraction)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    ref_steps = oracle_run(cfg, parts_np, E, B, steps=cfg.steps)
    strays_seen = 0
    for step in range(cfg.steps):
        rho, J, M = alloc_moments(cfg.nodes, 2)
        for s in range(2):
            ctx.push_and_moments(s, E, B, cfg.dt, cfg.theta, rho[s], J[s], M, accumulate=(pk.ACC_M_ONLY if s > 0 else pk.ACC_NONE))
            strays_seen += ctx.stray_count()
        total, per_species = ref_steps[step]
        for s in range(2):
            assert_moments_close(rho[s], J[s], None, per_species[s], f"step {step} species {s}")
        assert_moments_close(None, None, M, total, f"step {step}")
    for s, sp in enumerate(cfg.species):
        got = {k: parts_cuda[s][k].cpu().numpy() for k in PKEYS}
        order = np.argsort(_ids(got["q"], sp.q_sign * cfg.q_abs))
        got = {k: got[k][order] for k in PKEYS}
        assert np.array_equal(_ids(got["q"], sp.q_sign * cfg.q_abs), np.arange(parts[s]["n"]))
        assert_particles_close(got, parts_np[s], cfg, f"final species {s}")
    assert strays_seen > 0                      # the stray (atomic) path was exercised
    if resort_fraction < 1.0:
        assert ctx.resort_count() > 0           # electrons (1 %/step leave their cell) were re-sorted
    else:
        assert ctx.resort_count() == 0
    ctx.close()


# ------------------------------------------------------------------ edge cases

def _single_species_cfg(grid, qom, dt):
    import dataclasses
    base = wl.config(0)
    sp = dataclasses.replace(base.species[0], qom=qom)
    return dataclasses.replace(base, nx=grid[0], ny=grid[1], nz=grid[2], dx=grid[3], dy=grid[4], dz=grid[5],
                               dt=dt, species=(sp,), name="edge")


@pytest.mark.parametrize("variant", [pk.VARIANT_FUSED, pk.VARIANT_ATOMIC], ids=["fused", "atomic"])
def test_ragged_cells_anisotropic_grid_unsorted_input(variant):
    """Random particles on a 4x5x3 grid with spacing (0.7,1.3,0.9): empty cells, cells with 1..200
    particles (ragged 32-batches), strong field, particles exactly on nodes, faces and at L - ulp."""
    grid = (4, 5, 3, 0.7, 1.3, 0.9)
    cfg = _single_species_cfg(grid, -7.0, 0.3)
    rng = np.random.default_rng(11)
    p = rand_particles(rng, 3000, grid, vscale=0.3)
    # pile 200 particles into one cell, leave the rest thin
    p["x"][:200] = 0.7 * (2 + rng.uniform(0, 1, 200))
    p["y"][:200] = 1.3 * (3 + rng.uniform(0, 1, 200))
    p["z"][:200] = 0.9 * (1 + rng.uniform(0, 1, 200))
    Lx, Ly, Lz = cfg.lengths
    # special positions: on a node, on faces, just below the upper box edge, at 0
    p["x"][200:206] = [0.0, 1.4, np.nextafter(Lx, 0), 0.7, 2.1, 0.35]
    p["y"][200:206] = [0.0, 2.6, np.nextafter(Ly, 0), 0.1, 3.9, 6.4999]
    p["z"][200:206] = [0.0, 0.9, np.nextafter(Lz, 0), 1.8, 0.45, 2.6999]
    En, Bn = rand_fields(rng, grid, escale=0.5, bscale=3.0)
    E, B = torch.from_numpy(En).cuda(), torch.from_numpy(Bn).cuda()
    pc = to_cuda(from_numpy(p))
    ctx = make_ctx(cfg, 3000, variant, n_species=1)
    ctx.load_particles(0, -7.0, pc, sorted=False)
    perm = None
    if variant == pk.VARIANT_FUSED:
        pt = torch.empty(3000, dtype=torch.int32, device="cuda")
        ctx.sort_particles(0, None, pt)
        perm = pt.cpu().numpy().astype(np.int64) & 0xFFFFFFFF
    rho, J, M = alloc_moments(cfg.nodes, 1)
    ctx.push_and_moments(0, E, B, cfg.dt, cfg.theta, rho[0], J[0], M)
    torch.cuda.synchronize()
    mom = oracle.Moments(cfg.nodes)
    oracle.step(grid, -7.0, cfg.dt, p, En, Bn, mom)
    ref = p if perm is None else {k: p[k][perm] for k in PKEYS}
    assert_particles_close(pc, ref, cfg, "ragged")
    assert_moments_close(rho[0], J[0], M, mom, "ragged")
    ctx.close()


def test_unsorted_input_declared_sorted_is_still_correct():
    """`sorted` is only a hint: a shuffled species declared sorted goes through the stray path."""
    cfg = wl.config(0, (4, 4, 4))
    E, B = wl.gen_fields(cfg)
    E, B = E.cuda(), B.cuda()
    part = wl.gen_species(cfg, 0, shuffle=True)
    pn = to_numpy(part)
    pc = to_cuda(part)
    ctx = make_ctx(cfg, part["n"], n_species=1)
    ctx.load_particles(0, cfg.species[0].qom, pc, sorted=True)
    rho, J, M = alloc_moments(cfg.nodes, 1)
    ctx.push_and_moments(0, E, B, cfg.dt, cfg.theta, rho[0], J[0], M)
    assert ctx.stray_count() > part["n"] // 2
    mom = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), cfg.species[0].qom, cfg.dt, pn, E.cpu().numpy(), B.cpu().numpy(), mom)
    assert_particles_close(pc, pn, cfg, "lying hint")
    assert_moments_close(rho[0], J[0], M, mom, "lying hint")
    ctx.close()


def test_empty_species_and_single_particle():
    cfg = wl.config(0, (4, 4, 4))
    E, B = wl.gen_fields(cfg)
    E, B = E.cuda(), B.cuda()
    ctx = make_ctx(cfg, 16, n_species=1)
    empty = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in PKEYS}
    ctx.load_particles(0, 1.0, empty, sorted=True)
    rho, J, M = alloc_moments(cfg.nodes, 1)
    ctx.push_and_moments(0, E, B, cfg.dt, cfg.theta, rho[0], J[0], M)
    torch.cuda.synchronize()
    assert float(rho.abs().max()) == 0.0 and float(J.abs().max()) == 0.0 and float(M.abs().max()) == 0.0
    one = dict(x=np.array([3.999]), y=np.array([0.0]), z=np.array([2.5]), u=np.array([0.4]),
               v=np.array([-0.2]), w=np.array([0.9]), q=np.array([-0.5]))
    pc = to_cuda(from_numpy(one))
    ctx.load_particles(0, -3.0, pc, sorted=True)
    ctx.push_and_moments(0, E, B, cfg.dt, cfg.theta, rho[0], J[0], M)
    torch.cuda.synchronize()
    mom = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), -3.0, cfg.dt, one, E.cpu().numpy(), B.cpu().numpy(), mom)
    assert_particles_close(pc, one, cfg, "single")
    assert_moments_close(rho[0], J[0], M, mom, "single")
    ctx.close()


def test_error_paths_on_device():
    cfg = wl.config(0, (4, 4, 4))
    ctx = pk.Ecsim(*grid_of(cfg), 1)
    E, B = wl.gen_fields(cfg)
    E, B = E.cuda(), B.cuda()
    rho, J, M = alloc_moments(cfg.nodes, 1)
    with pytest.raises(pk.EcsimError, match="no particles loaded"):
        ctx.push_and_moments(0, E, B, 0.1, 0.5, rho[0], J[0], M)
    part = to_cuda(wl.gen_species(cfg, 0))
    ctx.load_particles(0, -64.0, part, sorted=True)
    with pytest.raises(pk.EcsimError, match="workspace"):
        ctx.push_and_moments(0, E, B, 0.1, 0.5, rho[0], J[0], M)
    ctx.set_workspace(int(part["x"].numel()))
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.push_and_moments(0, E, B, -0.1, 0.5, rho[0], J[0], M)      # dt <= 0
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.push_and_moments(0, E, B, 0.1, 0.2, rho[0], J[0], M)       # theta outside [0.5, 1]
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.push_and_moments(3, E, B, 0.1, 0.5, rho[0], J[0], M)       # species out of range
    ctx.push_and_moments(0, E, B, 0.1, 0.5, rho[0], J[0], M)
    torch.cuda.synchronize()
    ctx.close()


# ------------------------------------------------------------------ host-buffer (end-to-end) entry

def test_host_buffer_step_matches_oracle():
    cfg = wl.config(0)
    E, B = wl.gen_fields(cfg)
    part = wl.gen_species(cfg, 0)
    pn = to_numpy(part)
    host = {k: part[k].clone().pin_memory() for k in PKEYS}
    n = part["n"]
    ctx = pk.Ecsim(*grid_of(cfg), 1)
    ctx.set_workspace(n, host_step=True)
    rho = torch.empty(cfg.nodes, dtype=torch.float64).pin_memory()
    J = torch.empty(3, cfg.nodes, dtype=torch.float64).pin_memory()
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64).pin_memory()
    ctx.push_and_moments_host(cfg.species[0].qom, True, host, E.contiguous(), B.contiguous(), cfg.dt, cfg.theta,
                              rho, J, M)
    mom = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), cfg.species[0].qom, cfg.dt, pn, E.numpy(), B.numpy(), mom)
    assert_particles_close(host, pn, cfg, "host step")
    assert_moments_close(rho, J, M, mom, "host step")
    ctx.close()


def test_host_buffer_all_species_step_matches_oracle():
    cfg = wl.config(0)
    E, B = wl.gen_fields(cfg)
    parts = [wl.gen_species(cfg, s) for s in range(2)]
    parts_np = [to_numpy(p) for p in parts]
    host = [{k: p[k].clone().pin_memory() for k in PKEYS} for p in parts]
    ctx = pk.Ecsim(*grid_of(cfg), 2)
    ctx.set_workspace_host_all(max(p["n"] for p in parts), sum(p["n"] for p in parts))
    rho = torch.empty(2, cfg.nodes, dtype=torch.float64).pin_memory()
    J = torch.empty(2, 3, cfg.nodes, dtype=torch.float64).pin_memory()
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64).pin_memory()
    ctx.push_and_moments_host_all([sp.qom for sp in cfg.species], True, host, E.contiguous(), B.contiguous(), cfg.dt,
                                  cfg.theta, rho, J, M)
    (total, per_species), = oracle_run(cfg, parts_np, E, B)
    for s in range(2):
        assert_particles_close(host[s], parts_np[s], cfg, f"host all, species {s}")
        assert_moments_close(rho[s], J[s], None, per_species[s], f"host all, species {s}")
    assert_moments_close(None, None, M, total, "host all")
    # the single-species host call still works on the same context afterwards
    ctx.close()


@pytest.mark.parametrize("idx,scale", [(0, None), (3, (6, 48, 6)), (2, (9, 4, 5))], ids=["cfg0", "cfg3", "cfg2_odd"])
def test_pipelined_host_step_matches_oracle(idx, scale):
    """The host-buffer entry as a three-stream pipeline over slabs of x-planes (upload | compute | download); forced on a
    small input with ecsim_set_host_pipeline(2).  Same parity as the serial path; both M layouts."""
    cfg = wl.config(idx, scale)
    E, B = wl.gen_fields(cfg)
    parts = [wl.gen_species(cfg, s, shuffle=False) for s in range(2)]
    for layout in (pk.M_27, pk.M_14):
        parts_np = [to_numpy(p) for p in parts]
        host = [{k: p[k].clone().pin_memory() for k in PKEYS} for p in parts]
        ctx = pk.Ecsim(*grid_of(cfg), 2)
        ctx.set_workspace_host_all(max(p["n"] for p in parts), sum(p["n"] for p in parts))
        ctx.set_host_pipeline(2)
        ctx.set_m_layout(layout)
        rho = torch.full((2, cfg.nodes), float("nan"), dtype=torch.float64).pin_memory()
        J = torch.full((2, 3, cfg.nodes), float("nan"), dtype=torch.float64).pin_memory()
        M = torch.full((cfg.nodes, 27 if layout == pk.M_27 else 14, 3, 3), float("nan"), dtype=torch.float64).pin_memory()
        ctx.push_and_moments_host_all([sp.qom for sp in cfg.species], True, host, E.contiguous(), B.contiguous(), cfg.dt,
                                      cfg.theta, rho, J, M)
        assert ctx.host_pipelined_count() == 1
        (total, per_species), = oracle_run(cfg, parts_np, E, B)
        for s in range(2):
            assert_particles_close(host[s], parts_np[s], cfg, f"pipelined host step, species {s}")
            assert_moments_close(rho[s], J[s], None, per_species[s], f"pipelined host step, species {s}")
        if layout == pk.M_27:
            assert_moments_close(None, None, M, total, "pipelined host step")
        else:
            Mn = M.numpy()
            assert np.all(np.isfinite(Mn))
            assert np.all(np.abs(Mn - total.M[:, 13:]) <= 1e-10 * total.M_abs[:, 13:])
        ctx.close()


def test_pipelined_host_step_rejects_unsorted_input_declared_sorted():
    cfg = wl.config(0)
    E, B = wl.gen_fields(cfg)
    part = wl.gen_species(cfg, 0, shuffle=True)
    host = {k: part[k].clone().pin_memory() for k in PKEYS}
    ctx = pk.Ecsim(*grid_of(cfg), 1)
    ctx.set_workspace(part["n"], host_step=True)
    ctx.set_host_pipeline(2)
    rho = torch.empty(cfg.nodes, dtype=torch.float64).pin_memory()
    J = torch.empty(3, cfg.nodes, dtype=torch.float64).pin_memory()
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64).pin_memory()
    with pytest.raises(pk.EcsimError, match="out of order|invalid"):
        ctx.push_and_moments_host(cfg.species[0].qom, True, host, E.contiguous(), B.contiguous(), cfg.dt, cfg.theta, rho, J, M)
    # declared unsorted: the serial path sorts, and is right
    pn = to_numpy(part)
    host = {k: part[k].clone().pin_memory() for k in PKEYS}
    ctx.push_and_moments_host(cfg.species[0].qom, False, host, E.contiguous(), B.contiguous(), cfg.dt, cfg.theta, rho, J, M)
    mom = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), cfg.species[0].qom, cfg.dt, pn, E.numpy(), B.numpy(), mom)
    assert_moments_close(rho, J, M, mom, "host step, unsorted")
    ctx.close()


@pytest.mark.parametrize("warps", [8, 16])
def test_other_warp_counts_of_the_fused_kernel(warps):
    """ecsim_set_fused_warps: the 8 x 224- and 16 x 128-register instantiations of the fused kernel (default 12 x 168)."""
    cfg = wl.config(3, (6, 48, 6))
    E, B, parts = gen_all(cfg)
    parts_np = [to_numpy(p) for p in parts]
    parts_cuda = [to_cuda(p) for p in parts]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    ctx.set_fused_warps(warps)
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.set_fused_warps(13)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    rho, J, M = alloc_moments(cfg.nodes, 2)
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
    torch.cuda.synchronize()
    (total, per_species), = oracle_run(cfg, parts_np, E, B)
    for s in range(2):
        assert_particles_close(parts_cuda[s], parts_np[s], cfg, f"species {s}")
        assert_moments_close(rho[s], J[s], None, per_species[s], f"species {s}")
    assert_moments_close(None, None, M, total, f"{warps} warps")
    ctx.close()


def test_pipelined_host_step_with_some_outputs_absent():
    """NULL outputs are skipped in the pipeline too: only rho, then only M."""
    cfg = wl.config(0)
    E, B = wl.gen_fields(cfg)
    part = wl.gen_species(cfg, 0)
    for want in ("rho", "M"):
        pn = to_numpy(part)
        host = {k: part[k].clone().pin_memory() for k in PKEYS}
        ctx = pk.Ecsim(*grid_of(cfg), 1)
        ctx.set_workspace(part["n"], host_step=True)
        ctx.set_host_pipeline(2)
        rho = torch.full((cfg.nodes,), float("nan"), dtype=torch.float64).pin_memory() if want == "rho" else None
        M = torch.full((cfg.nodes, 27, 3, 3), float("nan"), dtype=torch.float64).pin_memory() if want == "M" else None
        ctx.push_and_moments_host(cfg.species[0].qom, True, host, E.contiguous(), B.contiguous(), cfg.dt, cfg.theta, rho, None, M)
        assert ctx.host_pipelined_count() == 1
        mom = oracle.Moments(cfg.nodes)
        oracle.step(grid_of(cfg), cfg.species[0].qom, cfg.dt, pn, E.numpy(), B.numpy(), mom)
        assert_particles_close(host, pn, cfg, "host step")
        assert_moments_close(rho, None, M, mom, f"host step, only {want}")
        ctx.close()


def test_validate_particles_counts_what_the_path_cannot_take():
    cfg = wl.config(0, (4, 4, 4))
    part = to_cuda(wl.gen_species(cfg, 0))
    ctx = make_ctx(cfg, int(part["x"].numel()), n_species=1)
    ctx.load_particles(0, -64.0, part, sorted=True)
    assert ctx.validate_particles(0) == 0
    part["x"][3] = float("nan")
    part["y"][5] = cfg.lengths[1]            # == L: outside [0, L)
    part["z"][7] = -1e-300
    part["w"][9] = float("inf")
    part["q"][11] = float("nan")
    part["x"][11] = float("nan")             # two faults, one particle
    assert ctx.validate_particles(0) == 5
    ctx.close()
