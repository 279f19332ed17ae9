"""Shared driver of the slab-decomposition tests: a few steps of a domain-decomposed run compared with
the single-domain oracle.  The per-slab compute engine is a callback: the CPU oracle on the slab's local grid in the
gloo / LocalRing tests (this file imports `oracle`: test infrastructure), libecpush in the -m gpu test."""
from __future__ import annotations

import numpy as np
import torch

import oracle
import workloads as wl
from paper_2603_16624_b200.slabs import PKEYS, SlabGrid
from util import grid_of, periodic_absdiff


def tagged_global_particles(cfg):
    parts = []
    for s, sp in enumerate(cfg.species):
        p = wl.gen_species(cfg, s)
        q0 = sp.q_sign * cfg.q_abs
        d = {k: p[k].clone() for k in PKEYS}
        d["q"] = q0 * (1.0 + torch.arange(d["q"].numel(), dtype=torch.float64) * 2.0 ** -30)
        parts.append(d)
    return parts


def ids_of(q, q0):
    return np.rint((np.asarray(q) / q0 - 1.0) * 2.0 ** 30).astype(np.int64)


def oracle_engine(grid: SlabGrid, cfg, parts_l, E_l, B_l):
    """One step of every species of one slab on its local (periodic, nxl + 2 planes) grid with the CPU oracle.
    Returns rho [nsp][nodes_l], J [nsp][3][nodes_l], M [nodes_l][243] (torch, CPU); parts_l updated in place."""
    nsp = len(cfg.species)
    nl = grid.local_nodes
    rho = torch.zeros(nsp, nl, dtype=torch.float64)
    J = torch.zeros(nsp, 3, nl, dtype=torch.float64)
    M = torch.zeros(nl, 243, dtype=torch.float64)
    En, Bn = E_l.numpy(), B_l.numpy()
    for s, sp in enumerate(cfg.species):
        m = oracle.Moments(nl, with_abs=False)
        pn = {k: parts_l[s][k].numpy() for k in PKEYS}           # shares memory with the torch tensors
        oracle.step(grid.local_dims, sp.qom, cfg.dt, pn, En, Bn, m)
        rho[s] = torch.from_numpy(m.rho)
        J[s] = torch.from_numpy(m.J)
        M += torch.from_numpy(m.M.reshape(nl, 243))
    return rho, J, M


def global_reference_step(cfg, ref_parts, E, B):
    """The same step on the undecomposed grid: per-species Moments (with |addend| sums) and their M total."""
    total = oracle.Moments(cfg.nodes)
    per = []
    for s, sp in enumerate(cfg.species):
        m = oracle.Moments(cfg.nodes)
        oracle.step(grid_of(cfg), sp.qom, cfg.dt, ref_parts[s], E.numpy(), B.numpy(), m)
        per.append(m)
        total.M += m.M
        total.M_abs += m.M_abs
    return per, total


def check_against_global(cfg, grids, owned_rho, owned_J, owned_M, parts_global, ref_parts, per, total, what):
    """owned_*: per rank, the owned node planes; parts_global: per rank per species, particles in global coordinates."""
    nsp = len(cfg.species)
    rho = torch.cat(owned_rho, dim=1).numpy()                     # [nsp][nodes]: slabs are consecutive x-planes
    J = torch.cat(owned_J, dim=2).numpy()
    M = torch.cat(owned_M, dim=0).numpy().reshape(cfg.nodes, 27, 3, 3)
    for s in range(nsp):
        assert np.all(np.abs(rho[s] - per[s].rho) <= 1e-10 * per[s].rho_abs), f"{what}: rho species {s}"
        assert np.all(np.abs(J[s] - per[s].J) <= 1e-10 * per[s].J_abs), f"{what}: Jhat species {s}"
    assert np.all(np.abs(M - total.M) <= 1e-10 * total.M_abs), f"{what}: M"
    L = cfg.lengths
    for s, sp in enumerate(cfg.species):
        q0 = sp.q_sign * cfg.q_abs
        got = {k: np.concatenate([np.asarray(parts_global[r][s][k]) for r in range(len(grids))]) for k in PKEYS}
        order = np.argsort(ids_of(got["q"], q0))
        got = {k: got[k][order] for k in PKEYS}
        n = ref_parts[s]["x"].shape[0]
        assert np.array_equal(ids_of(got["q"], q0), np.arange(n)), f"{what}: particle set of species {s} not conserved"
        for c, k in enumerate("xyz"):
            assert (periodic_absdiff(got[k], ref_parts[s][k], L[c]) / L[c]).max() <= 1e-13, f"{what}: {k}"
        for k in "uvw":
            assert np.abs(got[k] - ref_parts[s][k]).max() <= 1e-13 * max(np.abs(ref_parts[s][k]).max(), 1e-300), f"{what}: {k}"
        # every particle is in the slab that owns its cell
        for r, g in enumerate(grids):
            xg = np.asarray(parts_global[r][s]["x"])
            ci = np.minimum(np.floor(xg / cfg.dx), cfg.nx - 1)
            assert np.all((ci >= g.i0) & (ci < g.i1)), f"{what}: rank {r} holds a particle outside its slab"
        ref_parts[s] = got                                       # restart the reference from the decomposed state
    return got
