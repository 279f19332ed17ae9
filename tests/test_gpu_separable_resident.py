"""-m gpu parity of SURVEY §8(f)1: the separable entry points (ecsim_moments / ecsim_push) and the
sort-preserving push of RESIDENT species (library-managed gapped double buffers; L149), against the CPU oracle.

  * ecsim_moments == the oracle with do_push = 0 (x, v bitwise untouched); ecsim_push == the oracle's mover;
    ecsim_moments followed by ecsim_push == ecsim_push_and_moments, bit for bit (same per-particle arithmetic);
  * resident species: every step of a multi-step run matches the oracle element by element (moments on the whole
    grid, every particle through an id carried in q), with ZERO strays, ZERO re-sorts, and the particle set conserved;
  * segments that fill up: a tiny slack forces the overflow list and a fresh layout (ecsim_relayout_count), same parity.
"""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import (alloc_moments, assert_moments_close, assert_particles_close, from_numpy, gen_all, make_ctx,
                      oracle_run, to_cuda)
from util import PKEYS, grid_of, rand_fields, rand_particles, to_numpy

pytestmark = pytest.mark.gpu


def _tag_ids(q, q0):
    return q0 * (1.0 + np.arange(q.shape[0]) * 2.0 ** -30)


def _ids(q, q0):
    return np.rint((q / q0 - 1.0) * 2.0 ** 30).astype(np.int64)


def _export(ctx, s, n):
    out = {k: torch.empty(n, dtype=torch.float64, device="cuda") for k in PKEYS}
    ctx.export_particles(s, out)
    torch.cuda.synchronize()
    return {k: out[k].cpu().numpy() for k in PKEYS}


def _by_id(p, q0):
    order = np.argsort(_ids(p["q"], q0))
    return {k: p[k][order] for k in PKEYS}


# ------------------------------------------------------------------ separable entry points, dense layout

@pytest.mark.parametrize("variant", [pk.VARIANT_FUSED, pk.VARIANT_ATOMIC], ids=["fused", "atomic"])
@pytest.mark.parametrize("case", [(0, None), (3, (6, 48, 6)), (4, (10, 10, 10))], ids=["cfg0", "cfg3", "cfg4"])
def test_moments_then_push_match_oracle(case, variant):
    idx, scale = case
    cfg = wl.config(idx, scale)
    E, B, parts = gen_all(cfg, shuffle=False)
    nsp = len(cfg.species)
    parts_np = [to_numpy(p) for p in parts]
    parts_cuda = [to_cuda(p) for p in parts]
    ctx = make_ctx(cfg, max(p["n"] for p in parts), variant)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    # --- moments only: deposit, particles untouched (bitwise)
    rho, J, M = alloc_moments(cfg.nodes, nsp)
    for s in range(nsp):
        ctx.moments(s, B, cfg.dt, rho[s], J[s], M, accumulate=(pk.ACC_M_ONLY if s else pk.ACC_NONE))
    torch.cuda.synchronize()
    En, Bn = E.cpu().numpy(), B.cpu().numpy()
    total = oracle.Moments(cfg.nodes)
    for s, sp in enumerate(cfg.species):
        m = oracle.Moments(cfg.nodes)
        keep = {k: parts_np[s][k].copy() for k in PKEYS}
        oracle.step(grid_of(cfg), sp.qom, cfg.dt, parts_np[s], En, Bn, m, push=False)
        for k in PKEYS:
            assert np.array_equal(parts_np[s][k], keep[k])
            assert np.array_equal(parts_cuda[s][k].cpu().numpy(), keep[k]), f"ecsim_moments changed {k}"
        assert_moments_close(rho[s], J[s], None, m, f"moments species {s}")
        total.M += m.M
        total.M_abs += m.M_abs
    assert_moments_close(None, None, M, total, "moments")
    # --- push only: the oracle's mover (its deposit goes to a throw-away)
    for s in range(nsp):
        ctx.push(s, E, B, cfg.dt, cfg.theta)
    torch.cuda.synchronize()
    for s, sp in enumerate(cfg.species):
        oracle.step(grid_of(cfg), sp.qom, cfg.dt, parts_np[s], En, Bn, oracle.Moments(cfg.nodes, with_abs=False))
        assert_particles_close(parts_cuda[s], parts_np[s], cfg, f"push species {s}")
    ctx.close()


def test_moments_plus_push_is_bitwise_the_fused_call():
    cfg = wl.config(2, (6, 7, 8))
    E, B, parts = gen_all(cfg)
    outs = []
    for split in (False, True):
        parts_cuda = [to_cuda(p) for p in parts]
        ctx = make_ctx(cfg, max(p["n"] for p in parts))
        for s, sp in enumerate(cfg.species):
            ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
        rho, J, M = alloc_moments(cfg.nodes, 2)
        if split:
            ctx.moments_all(B, cfg.dt, rho, J, M)
            ctx.push_all(E, B, cfg.dt, cfg.theta)
        else:
            ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
        torch.cuda.synchronize()
        outs.append((rho, J, M, parts_cuda))
        ctx.close()
    for a, b in zip(outs[0][:3], outs[1][:3]):
        assert torch.equal(a, b)
    for s in range(2):
        for k in PKEYS:
            assert torch.equal(outs[0][3][s][k], outs[1][3][s][k]), k


def test_separable_calls_with_strays_dense():
    """moments / push on a dense species whose particles have left their cells (strays): several steps, no re-sort."""
    cfg = wl.config(1, (6, 5, 7))
    E, B, parts = gen_all(cfg)
    parts_np = [to_numpy(p) for p in parts]
    parts_cuda = [to_cuda(p) for p in parts]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    ctx.set_resort_fraction(100.0)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    strays = 0
    for step in range(4):
        rho, J, M = alloc_moments(cfg.nodes, 2)
        ctx.moments_all(B, cfg.dt, rho, J, M)
        strays += ctx.stray_count()
        ctx.push_all(E, B, cfg.dt, cfg.theta)
        torch.cuda.synchronize()
        (total, per_species), = oracle_run(cfg, parts_np, E, B)
        for s in range(2):
            assert_moments_close(rho[s], J[s], None, per_species[s], f"step {step} species {s}")
            assert_particles_close(parts_cuda[s], parts_np[s], cfg, f"step {step} species {s}")
        assert_moments_close(None, None, M, total, f"step {step}")
    assert strays > 0 and ctx.resort_count() == 0
    ctx.close()


# ------------------------------------------------------------------ resident species: the sort-preserving push

def _resident_run(cfg, steps, slack, mode, E, B, parts_np, expect_relayout=None, resort_fraction=None):
    """`mode`: 'fused' (ecsim_push_and_moments_all), 'split' (moments_all + push_all) or 'single' (per-species calls)."""
    nsp = len(cfg.species)
    q0 = [sp.q_sign * cfg.q_abs for sp in cfg.species]
    n_s = [p["x"].shape[0] for p in parts_np]
    parts_cuda = [to_cuda(from_numpy(p)) for p in parts_np]
    ctx = make_ctx(cfg, max(n_s + [1]))
    if resort_fraction is not None:
        ctx.set_resort_fraction(resort_fraction)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=False)
        ctx.make_resident(s, slack)
    # the caller's arrays are no longer referenced: scribble over them
    for s in range(nsp):
        for k in PKEYS:
            parts_cuda[s][k].fill_(float("nan"))
    # export right away: the same particle set
    for s in range(nsp):
        if n_s[s]:
            got = _by_id(_export(ctx, s, n_s[s]), q0[s])
            for k in PKEYS:
                assert np.array_equal(got[k], parts_np[s][k]), f"export after make_resident: {k}"
    ref = [{k: p[k].copy() for k in PKEYS} for p in parts_np]
    En, Bn = E.cpu().numpy(), B.cpu().numpy()
    leavers = 0
    for step in range(steps):
        rho, J, M = alloc_moments(cfg.nodes, nsp)
        if mode == "fused":
            ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
        elif mode == "split":
            ctx.moments_all(B, cfg.dt, rho, J, M)
            ctx.push_all(E, B, cfg.dt, cfg.theta)
        else:
            for s in range(nsp):
                ctx.push_and_moments(s, E, B, cfg.dt, cfg.theta, rho[s], J[s], M,
                                     accumulate=(pk.ACC_M_ONLY if s else pk.ACC_NONE))
        torch.cuda.synchronize()
        assert ctx.stray_count() == 0
        leavers += ctx.leaver_count()
        total = oracle.Moments(cfg.nodes)
        for s, sp in enumerate(cfg.species):
            m = oracle.Moments(cfg.nodes)
            oracle.step(grid_of(cfg), sp.qom, cfg.dt, ref[s], En, Bn, m)
            assert_moments_close(rho[s], J[s], None, m, f"resident step {step} species {s}")
            total.M += m.M
            total.M_abs += m.M_abs
        assert_moments_close(None, None, M, total, f"resident step {step}")
        for s in range(nsp):
            if n_s[s] == 0:
                continue
            got = _by_id(_export(ctx, s, n_s[s]), q0[s])
            assert np.array_equal(_ids(got["q"], q0[s]), np.arange(n_s[s])), "particle set not conserved"
            assert_particles_close(got, ref[s], cfg, f"resident step {step} species {s}")
            ref[s] = got                       # restart the oracle from the library's state: per-step bound
    assert ctx.resort_count() == 0
    if expect_relayout is True:
        assert ctx.relayout_count() > 0
    elif expect_relayout is False:
        assert ctx.relayout_count() == 0
    ctx.close()
    return leavers


def _tagged_parts(cfg):
    parts_np = []
    for s, sp in enumerate(cfg.species):
        p = to_numpy(wl.gen_species(cfg, s))
        p["q"] = _tag_ids(p["q"], sp.q_sign * cfg.q_abs)
        parts_np.append(p)
    return parts_np


@pytest.mark.parametrize("mode", ["fused", "split", "single"])
def test_resident_eleven_steps_match_oracle(mode):
    """Config 1's protocol (one step + 10 more, fields fixed) on a 10x8x12 box with resident species."""
    cfg = wl.config(1, (10, 8, 12))
    E, B = wl.gen_fields(cfg)
    # (the fixed random E of the recipe bunches the electrons: after ~5 steps single cells outgrow a slack of 25 % and the
    # species is laid out afresh once or twice -- part of what is tested; slack 1.0 below never needs it)
    leavers = _resident_run(cfg, cfg.steps, 0.25, mode, E.cuda(), B.cuda(), _tagged_parts(cfg))
    assert leavers > 100                         # particles did change cells, and were moved to their new segments


def test_resident_with_ample_slack_never_lays_out_again():
    cfg = wl.config(1, (10, 8, 12))
    E, B = wl.gen_fields(cfg)
    _resident_run(cfg, cfg.steps, 1.0, "fused", E.cuda(), B.cuda(), _tagged_parts(cfg), expect_relayout=False)


def test_resident_harris_sheet_and_shuffled_input():
    cfg = wl.config(3, (6, 48, 6))
    E, B = wl.gen_fields(cfg)
    parts_np = _tagged_parts(cfg)
    rng = np.random.default_rng(5)
    for p in parts_np:                           # arbitrary input order: make_resident sorts first
        perm = rng.permutation(p["x"].shape[0])
        for k in PKEYS:
            p[k] = p[k][perm]
        # ids follow the particles: re-tag in the new order so that _by_id / arange checks stay simple
    for s, sp in enumerate(cfg.species):
        parts_np[s]["q"] = _tag_ids(parts_np[s]["q"], sp.q_sign * cfg.q_abs)
    _resident_run(cfg, 4, 0.25, "fused", E.cuda(), B.cuda(), parts_np)


@pytest.mark.parametrize("resort_fraction", [0.0, 100.0], ids=["fresh_layout", "homeless_forever"])
def test_resident_full_segments(resort_fraction):
    """Hot particles (a quarter of them change cell per step) and segments with next to no slack: arrivals find their new
    cell full and go to the overflow list.  Every later pass deposits and pushes those homeless particles one warp each
    and tries again for a slot; with resort_fraction = 0 any overflow makes the next call lay the species out afresh,
    with 100 it never does.  Same parity either way (diagnostics included)."""
    base = wl.config(0, (6, 6, 6))
    hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.0, 0.5)))
    cfg = dataclasses.replace(base, dt=0.2, ppc=40, species=hot)
    E, B = wl.gen_fields(cfg)
    leavers = _resident_run(cfg, 5, 0.0, "fused", E.cuda(), B.cuda(), _tagged_parts(cfg),
                            expect_relayout=(resort_fraction == 0.0), resort_fraction=resort_fraction)
    assert leavers > 1000
    _resident_run(cfg, 3, 0.0, "split", E.cuda(), B.cuda(), _tagged_parts(cfg), resort_fraction=resort_fraction)


def test_resident_ragged_random_grid_three_species():
    """Anisotropic 4x5x3 grid, three species (one neutral, one empty), random positions incl. node / face / L-ulp."""
    grid = (4, 5, 3, 0.7, 1.3, 0.9)
    base = wl.config(0)
    qoms = [-7.0, 0.0, 2.0]
    species = tuple(dataclasses.replace(base.species[0], qom=q, q_sign=1.0) for q in qoms)
    cfg = dataclasses.replace(base, nx=4, ny=5, nz=3, dx=0.7, dy=1.3, dz=0.9, dt=0.3, species=species, q_abs=1.0,
                              name="ragged")
    rng = np.random.default_rng(21)
    parts_np = []
    for s, n in enumerate([3000, 700, 0]):
        p = rand_particles(rng, n, grid, vscale=0.3)
        if n >= 206:
            Lx, Ly, Lz = cfg.lengths
            p["x"][200:206] = [0.0, 1.4, np.nextafter(Lx, 0), 0.7, 2.1, 0.35]
            p["y"][200:206] = [0.0, 2.6, np.nextafter(Ly, 0), 0.1, 3.9, 6.4999]
            p["z"][200:206] = [0.0, 0.9, np.nextafter(Lz, 0), 1.8, 0.45, 2.6999]
        p["q"] = _tag_ids(p["q"], 1.0)
        parts_np.append(p)
    En, Bn = rand_fields(rng, grid, escale=0.5, bscale=3.0)
    _resident_run(cfg, 3, 0.25, "fused", torch.from_numpy(En).cuda(), torch.from_numpy(Bn).cuda(), parts_np)


def test_resident_and_dense_species_cannot_share_a_call():
    cfg = wl.config(0, (4, 4, 4))
    E, B, parts = gen_all(cfg)
    parts_cuda = [to_cuda(p) for p in parts]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    ctx.make_resident(0)
    rho, J, M = alloc_moments(cfg.nodes, 2)
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.sort_particles(0)
    ctx.push_and_moments(0, E, B, cfg.dt, cfg.theta, rho[0], J[0], M)            # per-species calls are fine
    ctx.push_and_moments(1, E, B, cfg.dt, cfg.theta, rho[1], J[1], M, accumulate=pk.ACC_M_ONLY)
    torch.cuda.synchronize()
    # a fresh load makes the species dense again
    ctx.load_particles(0, cfg.species[0].qom, to_cuda(parts[0]), sorted=True)
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
    torch.cuda.synchronize()
    ctx.close()


def test_resident_overflow_undoes_the_push_and_loses_nobody():
    """Segments with next to no slack, hot particles and an overflow list of FOUR entries: the push cannot place its
    leavers.  The next call must report ECSIM_ERR_OVERFLOW with the species back at its pre-push state, bit for bit, and
    every particle still there; with room in the list again the repeated push then equals the oracle's step, and the
    moments the fused call deposited (from the pre-push state) were right all along."""
    base = wl.config(0, (6, 6, 6))
    hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.0, 0.5)))
    cfg = dataclasses.replace(base, dt=0.2, ppc=40, species=hot)
    E, B = wl.gen_fields(cfg)
    E_c, B_c = E.cuda(), B.cuda()
    sp = cfg.species[0]
    q0 = sp.q_sign * cfg.q_abs
    p = to_numpy(wl.gen_species(cfg, 0))
    p["q"] = _tag_ids(p["q"], q0)
    n = p["x"].shape[0]
    ctx = make_ctx(cfg, n, n_species=1)
    ctx.load_particles(0, sp.qom, to_cuda(from_numpy(p)), sorted=False)
    ctx.make_resident(0, 0.0)
    ctx.set_overflow_capacity(0, 4)
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.set_overflow_capacity(0, 0)
    before = _by_id(_export(ctx, 0, n), q0)
    for k in PKEYS:
        assert np.array_equal(before[k], p[k])
    rho, J, M = alloc_moments(cfg.nodes, 1)
    ctx.push_and_moments(0, E_c, B_c, cfg.dt, cfg.theta, rho[0], J[0], M)      # enqueued; the overflow is found later
    torch.cuda.synchronize()
    with pytest.raises(pk.EcsimError, match="undone"):
        _export(ctx, 0, n)
    after = _by_id(_export(ctx, 0, n), q0)                                      # the call after the error works again
    assert np.array_equal(_ids(after["q"], q0), np.arange(n)), "a particle was lost or duplicated"
    for k in PKEYS:
        assert np.array_equal(after[k], before[k]), f"{k}: not the pre-push state"
    ref = {k: before[k].copy() for k in PKEYS}
    m = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), sp.qom, cfg.dt, ref, E.numpy(), B.numpy(), m)
    assert_moments_close(rho[0], J[0], M, m, "moments of the call whose push was undone")
    ctx.set_overflow_capacity(0, 65536)                                         # what make_resident carved
    ctx.push(0, E_c, B_c, cfg.dt, cfg.theta)
    got = _by_id(_export(ctx, 0, n), q0)
    assert np.array_equal(_ids(got["q"], q0), np.arange(n))
    assert_particles_close(got, ref, cfg, "repeated push")
    ctx.close()
