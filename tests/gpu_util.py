"""Helpers of the -m gpu parity tests: run libecpush through its C ABI (Python binding) and the
CPU oracle on the SAME generated inputs and compare element by element.

Tolerances (BASELINE.json north_star):
    positions   periodic |dx| / L            <= 1e-13
    velocities  |dv|_2 / |v_oracle|_2        <= 1e-13 per particle
    rho, Jhat, M   |d| <= 1e-10 * (sum of |addends| of that scalar, from the oracle)
    cell ids, per-cell counts                 bit-exact
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
import paper_2603_16624_b200 as pk
import workloads as wl
from util import PKEYS, grid_of, periodic_absdiff, to_numpy

POS_TOL = 1e-13
VEL_TOL = 1e-13
MOM_TOL = 1e-10


def to_cuda(part: dict) -> dict:
    return {k: part[k].detach().to("cuda", copy=True).contiguous() for k in PKEYS}


def from_numpy(part: dict) -> dict:
    return {k: torch.from_numpy(np.ascontiguousarray(part[k])) for k in PKEYS}


def make_ctx(cfg, n_max, variant=pk.VARIANT_FUSED, n_species=None, host_step=False):
    ctx = pk.Ecsim(*grid_of(cfg), n_species if n_species is not None else len(cfg.species))
    ctx.set_workspace(n_max, host_step=host_step)
    ctx.set_variant(variant)
    return ctx


def alloc_moments(nodes, n_species=1):
    rho = torch.full((n_species, nodes), float("nan"), dtype=torch.float64, device="cuda")
    J = torch.full((n_species, 3, nodes), float("nan"), dtype=torch.float64, device="cuda")
    M = torch.full((nodes, 27, 3, 3), float("nan"), dtype=torch.float64, device="cuda")
    return rho, J, M


def assert_particles_close(gpu: dict, ref: dict, cfg, what=""):
    L = cfg.lengths
    for c, k in enumerate("xyz"):
        g = gpu[k].cpu().numpy() if torch.is_tensor(gpu[k]) else gpu[k]
        assert np.all((g >= 0.0) & (g < L[c])), f"{what}: {k} outside [0,L)"
        d = periodic_absdiff(g, ref[k], L[c]) / L[c]
        assert d.max() <= POS_TOL, f"{what}: position {k} off by {d.max():.3e} (relative to L)"
    gv = np.stack([(gpu[k].cpu().numpy() if torch.is_tensor(gpu[k]) else gpu[k]) for k in "uvw"], -1)
    rv = np.stack([ref[k] for k in "uvw"], -1)
    num = np.linalg.norm(gv - rv, axis=-1)
    den = np.linalg.norm(rv, axis=-1)
    rel = num / np.maximum(den, 1e-300)
    assert rel.max() <= VEL_TOL, f"{what}: velocity off by {rel.max():.3e}"


def assert_moments_close(rho, J, M, mom: "oracle.Moments", what=""):
    """rho [nodes], J [3][nodes], M [nodes][27][3][3] (torch cuda or numpy) against an oracle.Moments
    carrying the |addend| sums."""
    def np_(t):
        return t.detach().cpu().numpy() if torch.is_tensor(t) else t
    for name, got, ref, norm in (("rho", rho, mom.rho, mom.rho_abs), ("J", J, mom.J, mom.J_abs),
                                 ("M", M, mom.M, mom.M_abs)):
        if got is None:
            continue
        g = np_(got).reshape(ref.shape)
        assert np.all(np.isfinite(g)), f"{what}: {name} has non-finite entries"
        err = np.abs(g - ref)
        bound = MOM_TOL * norm
        bad = err > bound
        if bad.any():
            idx = np.unravel_index(np.argmax(err - bound), err.shape)
            raise AssertionError(f"{what}: {name}{idx} = {g[idx]!r} vs oracle {ref[idx]!r}; |d| = {err[idx]:.3e} > "
                                 f"1e-10 * {norm[idx]:.3e}; {int(bad.sum())} entries out of tolerance")


def oracle_run(cfg, parts_np, E, B, steps=1):
    """Oracle on numpy copies: returns (list of per-step Moments summed over species with per-species rho/J,
    final particles).  parts_np: list over species of dicts (updated in place)."""
    grid = grid_of(cfg)
    out = []
    En, Bn = E.cpu().numpy(), B.cpu().numpy()
    for _ in range(steps):
        per_species = []
        total = oracle.Moments(cfg.nodes)
        for s, sp in enumerate(cfg.species):
            m = oracle.Moments(cfg.nodes)
            oracle.step(grid, sp.qom, cfg.dt, parts_np[s], En, Bn, m)
            per_species.append(m)
            total.M += m.M
            total.M_abs += m.M_abs
            total.rho += m.rho
            total.rho_abs += m.rho_abs
            total.J += m.J
            total.J_abs += m.J_abs
        out.append((total, per_species))
    return out


def gen_all(cfg, shuffle=None):
    """(E, B on cuda, list of generated species dicts on CPU)."""
    E, B = wl.gen_fields(cfg)
    parts = [wl.gen_species(cfg, s, shuffle=shuffle) for s in range(len(cfg.species))]
    return E.cuda(), B.cuda(), parts
