"""-m gpu parity of SURVEY §8(f)4, first half: reduced dimensionality (PAPER.md L123 fixPosition; reading R25).
ecsim_set_fixed_axes pins the inactive coordinates in every push; several consecutive steps of 2-D and 1-D runs are
compared with the oracle (oracle.step followed by oracle.fix_position), dense and resident species, fused / split calls
and the atomic variant."""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import alloc_moments, assert_moments_close, assert_particles_close, from_numpy, make_ctx, to_cuda
from util import PKEYS, grid_of, to_numpy

pytestmark = pytest.mark.gpu


def _ids(q, q0):
    return np.rint((q / q0 - 1.0) * 2.0 ** 30).astype(np.int64)


@pytest.mark.parametrize("kind", ["dense", "resident", "atomic", "split"])
@pytest.mark.parametrize("mask", [4, 6], ids=["2d_xy", "1d_x"])
def test_reduced_dimension_steps_match_oracle(mask, kind):
    cfg = wl.config(1, (12, 10, 3))
    pos = (0.0, 4.0 * cfg.dy, 1.0 * cfg.dz)                      # node line y = 4, node plane z = 1
    E, B = wl.gen_fields(cfg)
    En, Bn = E.numpy(), B.numpy()
    ref, q0 = [], []
    for s, sp in enumerate(cfg.species):
        p = to_numpy(wl.gen_species(cfg, s))
        q0.append(sp.q_sign * cfg.q_abs)
        p["q"] = q0[s] * (1.0 + np.arange(p["q"].shape[0]) * 2.0 ** -30)
        ref.append(p)
    pcs = [to_cuda(from_numpy(p)) for p in ref]
    for p in ref:
        oracle.fix_position(p, mask, *pos)
    ctx = make_ctx(cfg, max(p["x"].shape[0] for p in ref), pk.VARIANT_ATOMIC if kind == "atomic" else pk.VARIANT_FUSED)
    ctx.set_fixed_axes(mask, *pos)                                # before the load: the load pins
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, pcs[s], sorted=False)
        if kind == "resident":
            ctx.make_resident(s)
    E_c, B_c = E.cuda(), B.cuda()
    for step in range(4):
        rho, J, M = alloc_moments(cfg.nodes, 2)
        if kind == "split":
            ctx.moments_all(B_c, cfg.dt, rho, J, M)
            ctx.push_all(E_c, B_c, cfg.dt, cfg.theta)
        else:
            ctx.push_and_moments_all(E_c, B_c, cfg.dt, cfg.theta, rho, J, M)
        torch.cuda.synchronize()
        total = oracle.Moments(cfg.nodes)
        for s, sp in enumerate(cfg.species):
            m = oracle.Moments(cfg.nodes)
            oracle.step(grid_of(cfg), sp.qom, cfg.dt, ref[s], En, Bn, m)
            oracle.fix_position(ref[s], mask, *pos)
            assert_moments_close(rho[s], J[s], None, m, f"step {step} species {s}")
            total.M += m.M
            total.M_abs += m.M_abs
        assert_moments_close(None, None, M, total, f"step {step}")
        # nothing is deposited off the plane / line
        M7 = M.view(cfg.nx, cfg.ny, cfg.nz, 27, 9)
        assert float(M7[:, :, [0, 2]].abs().max()) == 0.0
        for s in range(2):
            n = ref[s]["x"].shape[0]
            out = {k: torch.empty(n, dtype=torch.float64, device="cuda") for k in PKEYS}
            ctx.export_particles(s, out)
            torch.cuda.synchronize()
            got = {k: out[k].cpu().numpy() for k in PKEYS}
            order = np.argsort(_ids(got["q"], q0[s]))
            got = {k: got[k][order] for k in PKEYS}
            assert np.array_equal(_ids(got["q"], q0[s]), np.arange(n))
            assert np.all(got["z"] == pos[2])
            if mask & 2:
                assert np.all(got["y"] == pos[1])
            assert_particles_close(got, ref[s], cfg, f"step {step} species {s}")
            ref[s] = got
    ctx.close()


def test_fixed_axes_set_after_the_load_and_switched_off():
    cfg = wl.config(0, (6, 6, 4))
    E, B = wl.gen_fields(cfg)
    p = to_numpy(wl.gen_species(cfg, 0))
    pc = to_cuda(from_numpy(p))
    ctx = make_ctx(cfg, p["x"].shape[0], n_species=1)
    ctx.load_particles(0, cfg.species[0].qom, pc, sorted=True)
    ctx.set_fixed_axes(4, 0.0, 0.0, 2.0)                          # pins the loaded species now
    torch.cuda.synchronize()
    assert bool((pc["z"] == 2.0).all())
    oracle.fix_position(p, 4, 0.0, 0.0, 2.0)
    rho, J, M = alloc_moments(cfg.nodes, 1)
    ctx.push_and_moments(0, E.cuda(), B.cuda(), cfg.dt, cfg.theta, rho[0], J[0], M)
    torch.cuda.synchronize()
    m = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), cfg.species[0].qom, cfg.dt, p, E.numpy(), B.numpy(), m)
    oracle.fix_position(p, 4, 0.0, 0.0, 2.0)
    assert_moments_close(rho[0], J[0], M, m, "pinned after load")
    with pytest.raises(pk.EcsimError, match="invalid"):
        ctx.set_fixed_axes(4, 0.0, 0.0, 99.0)                     # outside the box
    ctx.set_fixed_axes(0)                                         # 3-D again: z moves
    ctx.push_and_moments(0, E.cuda(), B.cuda(), cfg.dt, cfg.theta, rho[0], J[0], M)
    torch.cuda.synchronize()
    assert not bool((pc["z"] == 2.0).all())
    ctx.close()


def test_host_step_with_fixed_axes_pins_what_it_uploads():
    """The host-buffer entry while axes are pinned: the particles arrive unpinned in HOST memory, so the pinning has to
    happen after the upload.  The pipelined form (which loads before it uploads) must not be taken; forced on, the call
    still goes through the serial path and equals oracle.fix_position + oracle.step + oracle.fix_position."""
    cfg = wl.config(0, (8, 6, 4))
    E, B = wl.gen_fields(cfg)
    part = wl.gen_species(cfg, 0, shuffle=False)                 # cell-sorted, z anywhere in the box
    pn = to_numpy(part)
    host = {k: part[k].clone().pin_memory() for k in PKEYS}
    ctx = pk.Ecsim(*grid_of(cfg), 1)
    ctx.set_workspace(part["n"], host_step=True)
    ctx.set_host_pipeline(2)                                     # "pipeline whatever the size"
    pz = 2.0 * cfg.dz
    ctx.set_fixed_axes(4, 0.0, 0.0, pz)
    rho = torch.full((cfg.nodes,), float("nan"), dtype=torch.float64).pin_memory()
    J = torch.full((3, cfg.nodes), float("nan"), dtype=torch.float64).pin_memory()
    M = torch.full((cfg.nodes, 27, 3, 3), float("nan"), dtype=torch.float64).pin_memory()
    ctx.push_and_moments_host(cfg.species[0].qom, True, host, E.contiguous(), B.contiguous(), cfg.dt, cfg.theta, rho, J, M)
    assert ctx.host_pipelined_count() == 0
    oracle.fix_position(pn, 4, 0.0, 0.0, pz)
    m = oracle.Moments(cfg.nodes)
    oracle.step(grid_of(cfg), cfg.species[0].qom, cfg.dt, pn, E.numpy(), B.numpy(), m)
    oracle.fix_position(pn, 4, 0.0, 0.0, pz)
    assert_moments_close(rho, J, M, m, "host step, z pinned")
    assert bool((host["z"] == pz).all())
    assert_particles_close(host, pn, cfg, "host step, z pinned")
    M7 = M.view(cfg.nx, cfg.ny, cfg.nz, 27, 9)
    assert float(M7[:, :, [0, 1, 3]].abs().max()) == 0.0         # nothing deposited off the node plane k = 2
    ctx.close()


def test_fixed_axes_on_a_resident_species_pin_its_homeless_particles_too():
    """A resident species with full segments keeps some particles in its overflow list.  ecsim_set_fixed_axes must pin
    those as well: the layout that follows puts them back into segments, and anything it missed would stay off the
    plane until its next push."""
    base = wl.config(0, (6, 6, 6))
    hot = tuple(dataclasses.replace(sp, vth=v) for sp, v in zip(base.species, (1.0, 0.5)))
    cfg = dataclasses.replace(base, dt=0.2, ppc=40, species=hot)
    E, B = wl.gen_fields(cfg)
    E_c, B_c = E.cuda(), B.cuda()
    p = to_numpy(wl.gen_species(cfg, 0))
    n = p["x"].shape[0]
    q0 = cfg.species[0].q_sign * cfg.q_abs
    p["q"] = q0 * (1.0 + np.arange(n) * 2.0 ** -30)
    ctx = make_ctx(cfg, n, n_species=1)
    ctx.set_resort_fraction(100.0)                               # never lay out afresh: homeless particles stay homeless
    ctx.load_particles(0, cfg.species[0].qom, to_cuda(from_numpy(p)), sorted=False)
    ctx.make_resident(0, 0.0)                                    # no slack: arrivals find their cell full
    for _ in range(3):
        ctx.push(0, E_c, B_c, cfg.dt, cfg.theta)
    assert ctx.relayout_count() == 0
    pz = 3.0 * cfg.dz
    ctx.set_fixed_axes(4, 0.0, 0.0, pz)
    out = {k: torch.empty(n, dtype=torch.float64, device="cuda") for k in PKEYS}
    ctx.export_particles(0, out)
    torch.cuda.synchronize()
    assert np.array_equal(np.sort(_ids(out["q"].cpu().numpy(), q0)), np.arange(n))      # nobody lost
    assert bool((out["z"] == pz).all()), f"{int((out['z'] != pz).sum())} particle(s) left off the plane"
    rho = torch.full((cfg.nodes,), float("nan"), dtype=torch.float64, device="cuda")
    ctx.diagnostics(0, rho, None, None, None)
    torch.cuda.synchronize()
    r = rho.view(cfg.nx, cfg.ny, cfg.nz)
    assert float(r[:, :, [0, 1, 2, 4, 5]].abs().max()) == 0.0
    ctx.close()
