"""Pins of oracle.diagnostics (charge density, un-rotated charge current, pressure tensor, heat
flux; readings R22-R24 of DESIGN.md) against things other than itself.  CPU only.

The paper prints no formula and no number for the diagnostics: "absolute values unpinned by the paper"; what pins
the oracle are (i) the dense hat-function definition with no cell / corner logic (oracle/dense.hat_weights + plain
einsums), (ii) closed forms: one particle on a node, a cold beam (every particle the same velocity => J = rho v0,
P = rho v0 v0^T, Q = rho |v0|^2/2 v0 with rho pinned in test_oracle_pins.py), (iii) global sums, (iv) the tie to the
hot-path oracle: rho is the same rho, and with B = 0 (alpha = I) the un-rotated current IS Jhat, (v) translation.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from oracle import dense
from util import rand_fields, rand_particles

PAIRS = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]      # P components xx, xy, xz, yy, yz, zz


def _run(grid, p):
    d = oracle.Diagnostics(grid[0] * grid[1] * grid[2])
    oracle.diagnostics(grid, p, d)
    return d


@pytest.mark.parametrize("grid", [(3, 4, 5, 0.7, 1.3, 0.9), (5, 3, 3, 1.0, 0.5, 2.0), (2, 2, 2, 1.0, 1.0, 1.0)])
def test_dense_hat_function_brute_force(grid):
    rng = np.random.default_rng(7)
    p = rand_particles(rng, 300, grid, vscale=0.8)
    d = _run(grid, p)
    V = grid[3] * grid[4] * grid[5]
    if min(grid[:3]) >= 3:
        W = dense.hat_weights(grid, p["x"], p["y"], p["z"])        # [p, g], no cell logic
    else:
        # two nodes per axis: the minimum-image hat function double counts; build W from both images explicitly
        W = _weights_two_images(grid, p)
    v = np.stack([p["u"], p["v"], p["w"]], -1)
    qW = p["q"][:, None] * W / V
    assert np.allclose(d.rho, qW.sum(0), rtol=0, atol=1e-13 * np.abs(qW).sum(0).max())
    for c in range(3):
        ref = (qW * v[:, c:c + 1]).sum(0)
        assert np.allclose(d.J[c], ref, rtol=0, atol=1e-13 * d.J_abs[c].max())
        refq = (qW * (0.5 * (v * v).sum(-1) * v[:, c])[:, None]).sum(0)
        assert np.allclose(d.Q[c], refq, rtol=0, atol=1e-13 * d.Q_abs[c].max())
    for k, (i, j) in enumerate(PAIRS):
        ref = (qW * (v[:, i] * v[:, j])[:, None]).sum(0)
        assert np.allclose(d.P[k], ref, rtol=0, atol=1e-13 * d.P_abs[k].max())


def _weights_two_images(grid, p):
    nx, ny, nz, dx, dy, dz = grid

    def axis(pos, n, d):
        X = np.arange(n) * d
        L = n * d
        w = np.zeros((pos.shape[0], n))
        for shift in (-L, 0.0, L):
            w += np.maximum(0.0, 1.0 - np.abs(pos[:, None] - X[None, :] + shift) / d)
        return w
    wx, wy, wz = axis(p["x"], nx, dx), axis(p["y"], ny, dy), axis(p["z"], nz, dz)
    return (wx[:, :, None, None] * wy[:, None, :, None] * wz[:, None, None, :]).reshape(p["x"].shape[0], -1)


def test_one_particle_on_a_node():
    grid = (4, 3, 5, 0.5, 2.0, 1.0)
    V = 0.5 * 2.0 * 1.0
    i, j, k = 2, 1, 4
    p = dict(x=np.array([i * 0.5]), y=np.array([j * 2.0]), z=np.array([k * 1.0]), u=np.array([0.3]),
             v=np.array([-0.7]), w=np.array([1.1]), q=np.array([-0.25]))
    d = _run(grid, p)
    g = (i * 3 + j) * 5 + k
    vel = np.array([0.3, -0.7, 1.1])
    assert d.rho[g] == -0.25 / V and np.count_nonzero(d.rho) == 1
    assert np.allclose(d.J[:, g], -0.25 / V * vel, rtol=1e-15, atol=0)
    assert np.allclose(d.P[:, g], [-0.25 / V * vel[a] * vel[b] for a, b in PAIRS], rtol=1e-15, atol=0)
    assert np.allclose(d.Q[:, g], -0.25 / V * 0.5 * (vel @ vel) * vel, rtol=1e-15, atol=0)
    mask = np.ones(60, bool)
    mask[g] = False
    assert not d.J[:, mask].any() and not d.P[:, mask].any() and not d.Q[:, mask].any()


def test_cold_beam_closed_form_and_global_sums():
    grid = (5, 4, 3, 1.0, 0.8, 1.25)
    V = 1.0
    rng = np.random.default_rng(11)
    p = rand_particles(rng, 2000, grid)
    v0 = np.array([0.4, -1.2, 0.05])
    p["u"][:], p["v"][:], p["w"][:] = v0
    d = _run(grid, p)
    tol = 1e-13 * d.rho_abs.max()
    for c in range(3):
        assert np.allclose(d.J[c], d.rho * v0[c], rtol=0, atol=tol * abs(v0[c]))
        assert np.allclose(d.Q[c], d.rho * 0.5 * (v0 @ v0) * v0[c], rtol=0, atol=tol)
    for k, (i, j) in enumerate(PAIRS):
        assert np.allclose(d.P[k], d.rho * v0[i] * v0[j], rtol=0, atol=tol * 2)
    # global sums with thermal velocities: sum_g X_g V = sum_p q_p x_p
    p = rand_particles(rng, 2000, grid, vscale=0.7)
    d = _run(grid, p)
    v = np.stack([p["u"], p["v"], p["w"]], -1)
    assert abs(d.rho.sum() * V - p["q"].sum()) <= 1e-13 * np.abs(p["q"]).sum()
    for c in range(3):
        assert abs(d.J[c].sum() * V - (p["q"] * v[:, c]).sum()) <= 1e-13 * (np.abs(p["q"] * v[:, c])).sum()
        e = p["q"] * 0.5 * (v * v).sum(-1) * v[:, c]
        assert abs(d.Q[c].sum() * V - e.sum()) <= 1e-13 * np.abs(e).sum()
    for k, (i, j) in enumerate(PAIRS):
        e = p["q"] * v[:, i] * v[:, j]
        assert abs(d.P[k].sum() * V - e.sum()) <= 1e-13 * np.abs(e).sum()


def test_tie_to_the_hot_path_oracle():
    """rho is the hot path's rho bit for bit; with B = 0 (alpha = I, Eq. 2) the un-rotated current equals Jhat."""
    grid = (4, 5, 3, 0.7, 1.3, 0.9)
    nodes = 60
    rng = np.random.default_rng(13)
    p = rand_particles(rng, 500, grid, vscale=0.5)
    E, _ = rand_fields(rng, grid)
    B0 = np.zeros((3, nodes))
    m = oracle.Moments(nodes)
    oracle.step(grid, -3.0, 0.1, {k: v.copy() for k, v in p.items()}, E, B0, m, push=False)
    d = _run(grid, p)
    assert np.array_equal(d.rho, m.rho)
    assert np.allclose(d.J, m.J, rtol=0, atol=1e-15 * m.J_abs.max())
    # with B != 0 the two currents differ (the diagnostic one "excludes the effect of velocity rotation", L147)
    _, B = rand_fields(rng, grid)
    m2 = oracle.Moments(nodes)
    oracle.step(grid, -3.0, 0.1, {k: v.copy() for k, v in p.items()}, E, B, m2, push=False)
    assert np.abs(d.J - m2.J).max() > 1e-3 * np.abs(d.J).max()


def test_translation_by_whole_cells_rolls_the_outputs():
    grid = (4, 3, 5, 0.7, 1.3, 0.9)
    rng = np.random.default_rng(17)
    p = rand_particles(rng, 400, grid, vscale=0.5)
    # positions on a binary grid inside the cell so that shifting by whole cells is exact in floating point
    for k, (n, dd) in zip("xyz", ((4, 0.7), (3, 1.3), (5, 0.9))):
        cell = np.floor(p[k] / dd)
        frac = np.round((p[k] / dd - cell) * 64) / 64
        p[k] = (np.minimum(cell, n - 1) + np.minimum(frac, 63 / 64)) * dd
    d0 = _run(grid, p)
    sh = (1, 2, 3)
    p2 = {k: v.copy() for k, v in p.items()}
    for k, (n, dd), s in zip("xyz", ((4, 0.7), (3, 1.3), (5, 0.9)), sh):
        cell = np.floor(p[k] / dd + 1e-9)
        frac = p[k] / dd - cell
        p2[k] = (((cell + s) % n) + frac) * dd
    d1 = _run(grid, p2)
    for a, b in ((d0.rho, d1.rho),):
        assert np.allclose(np.roll(a.reshape(4, 3, 5), sh, (0, 1, 2)), b.reshape(4, 3, 5), rtol=0, atol=1e-13 * d0.rho_abs.max())
    for a, b, ab in ((d0.J, d1.J, d0.J_abs), (d0.P, d1.P, d0.P_abs), (d0.Q, d1.Q, d0.Q_abs)):
        ra = np.roll(a.reshape(-1, 4, 3, 5), sh, (1, 2, 3))
        assert np.allclose(ra, b.reshape(-1, 4, 3, 5), rtol=0, atol=1e-13 * ab.max())
