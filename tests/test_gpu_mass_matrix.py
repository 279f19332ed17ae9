"""-m gpu parity of SURVEY §8(f)2: the paper's 14-of-27 symmetric mass-matrix storage and the
operator sum_N' M_NN' E_N' of the field equations (Eq. 4-5) as a stencil mat-vec on the device.

  * ECSIM_M_14: the deposit writes M14[node][14][3][3] = slots 13..26 of the oracle's M[node][27][3][3], element by
    element within 1e-10 of the per-scalar |addend| sums; the 13 slots that are not stored follow from the mirror rule;
  * ecsim_apply_M on both layouts == oracle.apply_M (which is pinned against the dense all-pairs einsum in
    tests/test_oracle_pins.py), within 1e-12 of sum |M||E|;
  * ECsim's discrete energy identity on the DEVICE arrays of one whole step of configs[0] (north-star invariant):
        sum_g (Jhat_g + sum_g' M_gg' E_g') . E_g V dt  =  sum_p (m_p/2)(|v'|^2 - |v|^2),   m_p = q_p / (q/m)
    every term produced by the library's kernels (ecsim_push_and_moments_all, ecsim_apply_M), reduced with torch.
"""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from gpu_util import MOM_TOL, alloc_moments, gen_all, make_ctx, oracle_run, to_cuda
from util import PKEYS, grid_of, to_numpy

pytestmark = pytest.mark.gpu


def _step_both_layouts(cfg, variant_calls="all"):
    E, B, parts = gen_all(cfg, shuffle=False)
    nsp = len(cfg.species)
    out = {}
    for layout in (pk.M_27, pk.M_14):
        parts_cuda = [to_cuda(p) for p in parts]
        ctx = make_ctx(cfg, max(p["n"] for p in parts))
        ctx.set_m_layout(layout)
        for s, sp in enumerate(cfg.species):
            ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
        rho = torch.full((nsp, cfg.nodes), float("nan"), dtype=torch.float64, device="cuda")
        J = torch.full((nsp, 3, cfg.nodes), float("nan"), dtype=torch.float64, device="cuda")
        M = torch.full((cfg.nodes, 27 if layout == pk.M_27 else 14, 3, 3), float("nan"), dtype=torch.float64, device="cuda")
        if variant_calls == "all":
            ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
        else:
            for s in range(nsp):
                ctx.push_and_moments(s, E, B, cfg.dt, cfg.theta, rho[s], J[s], M,
                                     accumulate=(pk.ACC_M_ONLY if s else pk.ACC_NONE))
        torch.cuda.synchronize()
        out[layout] = (ctx, rho, J, M, parts_cuda)
    return E, B, parts, out


@pytest.mark.parametrize("case", [(0, None, "all"), (3, (5, 48, 4), "single"), (2, (7, 6, 5), "all")], ids=["cfg0", "cfg3", "cfg2"])
def test_symmetric_storage_matches_oracle_and_mirror_rule(case):
    idx, scale, calls = case
    cfg = wl.config(idx, scale)
    E, B, parts, out = _step_both_layouts(cfg, calls)
    parts_np = [to_numpy(p) for p in parts]
    (total, per_species), = oracle_run(cfg, parts_np, E, B)
    M14 = out[pk.M_14][3].cpu().numpy()
    M27 = out[pk.M_27][3].cpu().numpy()
    assert np.all(np.isfinite(M14))
    # stored slots: 13..26
    err = np.abs(M14 - total.M[:, 13:])
    assert np.all(err <= MOM_TOL * total.M_abs[:, 13:]), f"worst {err.max():.3e}"
    assert np.array_equal(M14, M27[:, 13:])                         # same arithmetic, same order: bitwise
    # the 13 slots that are not stored: M[g][o] = M[g + off(o)][26 - o]   (L73; R11: per component, no transpose)
    M5 = M14.reshape(cfg.nx, cfg.ny, cfg.nz, 14, 3, 3)
    T5 = total.M.reshape(cfg.nx, cfg.ny, cfg.nz, 27, 3, 3)
    A5 = total.M_abs.reshape(cfg.nx, cfg.ny, cfg.nz, 27, 3, 3)
    for o in range(13):
        di, dj, dk = o // 9 - 1, (o // 3) % 3 - 1, o % 3 - 1
        rebuilt = np.roll(M5[:, :, :, 13 - o], shift=(-di, -dj, -dk), axis=(0, 1, 2))   # value at g + off(o), slot 26-o
        assert np.all(np.abs(rebuilt - T5[:, :, :, o]) <= MOM_TOL * A5[:, :, :, o]), f"slot {o}"
    for layout in out:
        out[layout][0].close()


@pytest.mark.parametrize("case", [(0, None), (3, (5, 48, 4)), (2, (3, 2, 4))], ids=["cfg0", "cfg3", "tiny_2wide"])
def test_apply_M_matches_oracle_on_both_layouts(case):
    idx, scale = case
    cfg = wl.config(idx, scale)
    E, B, parts, out = _step_both_layouts(cfg)
    rng = np.random.default_rng(3)
    X = rng.standard_normal((3, cfg.nodes))                         # any node vector, not only E
    Xc = torch.from_numpy(X).cuda()
    M27 = out[pk.M_27][3].cpu().numpy()
    ref = oracle.apply_M(grid_of(cfg), np.ascontiguousarray(M27), X)
    # normaliser: sum |M||X| per output
    ref_abs = oracle.apply_M(grid_of(cfg), np.abs(M27), np.abs(X))
    for layout in (pk.M_27, pk.M_14):
        ctx, _, _, M, _ = out[layout]
        got = torch.full((3, cfg.nodes), float("nan"), dtype=torch.float64, device="cuda")
        ctx.apply_M(M, Xc, got)
        torch.cuda.synchronize()
        g = got.cpu().numpy()
        assert np.all(np.isfinite(g))
        assert np.all(np.abs(g - ref) <= 1e-12 * ref_abs + 1e-300), f"layout {layout}: worst {np.abs(g - ref).max():.3e}"
        ctx.apply_M(M, Xc, got, accumulate=True)                   # out += : twice the operator
        torch.cuda.synchronize()
        assert np.all(np.abs(got.cpu().numpy() - 2 * ref) <= 2e-12 * ref_abs + 1e-300)
    for layout in out:
        out[layout][0].close()


@pytest.mark.parametrize("layout", [pk.M_27, pk.M_14], ids=["27", "14"])
def test_energy_identity_on_device(layout):
    """sum_g (Jhat_g + (M E)_g) . E_g V dt = sum_p (m_p/2)(|v'|^2 - |v|^2) on configs[0], all on device arrays.
    (Per particle (m/2)(|v'|^2 - |v|^2) = q dt vbar.E_p, and sum_p q vbar.E_p = sum_g (Jhat + M E).E V: the two
    north-star identities chained; theta = 1/2: E^{n+theta} is the E the particles feel.)"""
    cfg = wl.config(0)
    E, B, parts = gen_all(cfg)
    nsp = len(cfg.species)
    parts_cuda = [to_cuda(p) for p in parts]
    v0 = [{k: parts_cuda[s][k].clone() for k in "uvw"} for s in range(nsp)]
    ctx = make_ctx(cfg, max(p["n"] for p in parts))
    ctx.set_m_layout(layout)
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts_cuda[s], sorted=True)
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64, device="cuda")
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64, device="cuda")
    M = torch.empty(cfg.nodes, 27 if layout == pk.M_27 else 14, 3, 3, dtype=torch.float64, device="cuda")
    ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
    ME = torch.empty(3, cfg.nodes, dtype=torch.float64, device="cuda")
    ctx.apply_M(M, E, ME)
    torch.cuda.synchronize()
    V = cfg.dx * cfg.dy * cfg.dz
    lhs = float(((J.sum(0) + ME) * E).sum()) * V * cfg.dt
    rhs = 0.0
    scale = 0.0
    for s, sp in enumerate(cfg.species):
        m = parts_cuda[s]["q"] / sp.qom
        ke1 = sum(parts_cuda[s][k] ** 2 for k in "uvw")
        ke0 = sum(v0[s][k] ** 2 for k in "uvw")
        rhs += float((0.5 * m * (ke1 - ke0)).sum())
        scale += float((0.5 * m.abs() * (ke1 + ke0)).sum())
    assert abs(lhs - rhs) <= 1e-12 * scale, (lhs, rhs, scale)
    assert abs(rhs) > 1e-6 * scale                                   # the identity is not trivially 0 = 0
    ctx.close()
