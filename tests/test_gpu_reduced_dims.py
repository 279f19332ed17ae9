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
