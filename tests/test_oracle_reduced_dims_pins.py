"""Pins of the reduced-dimension reading (PAPER.md L123 fixPosition; R25), CPU only: with the particles pinned
to a node plane (2-D) or a node line (1-D) the 3-D oracle must reproduce an INDEPENDENT lower-dimensional computation --
the dense hat-function definition (oracle/dense.py, no cell / corner / slot logic) on a grid with ONE node along every
pinned axis -- on that plane / line, and deposit nothing anywhere else ("necessary to ensure the correctness of the mass
matrix calculations in case of reduced simulation dimensions")."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from oracle import dense
from util import rand_fields, rand_particles


@pytest.mark.parametrize("mask,grid", [(4, (4, 5, 3, 0.7, 1.3, 0.9)), (6, (5, 3, 4, 1.0, 0.5, 2.0)), (1, (3, 4, 5, 0.8, 1.1, 0.6))],
                         ids=["2d_xy", "1d_x", "2d_yz"])
def test_pinned_run_equals_lower_dimensional_dense_definition(mask, grid):
    nx, ny, nz, dx, dy, dz = grid
    n3 = (nx, ny, nz)
    d3 = (dx, dy, dz)
    rng = np.random.default_rng(41)
    p = rand_particles(rng, 120, grid, vscale=0.5)
    E, B = rand_fields(rng, grid, escale=0.3, bscale=1.5)
    k0 = [1, 2, 1]                                              # the node plane / line the pinned axes sit on
    pos = [k0[a] * d3[a] for a in range(3)]
    oracle.fix_position(p, mask, *pos)
    qom, dt = -3.0, 0.1
    nodes = nx * ny * nz
    m = oracle.Moments(nodes)
    p3 = {k: v.copy() for k, v in p.items()}
    vbar = oracle.step(grid, qom, dt, p3, E, B, m, want_vbar=True)
    oracle.fix_position(p3, mask, *pos)
    # the lower-dimensional problem: one node along every pinned axis, fields = the plane / line the particles sit on
    nl = [1 if (mask >> a) & 1 else n3[a] for a in range(3)]
    gl = (nl[0], nl[1], nl[2], dx, dy, dz)
    sel = np.ix_(*[[k0[a]] if (mask >> a) & 1 else range(n3[a]) for a in range(3)])
    El = np.stack([E[c].reshape(n3)[sel].reshape(-1) for c in range(3)])
    Bl = np.stack([B[c].reshape(n3)[sel].reshape(-1) for c in range(3)])
    pl = {k: v.copy() for k, v in p.items()}
    for a, key in enumerate("xyz"):
        if (mask >> a) & 1:
            pl[key] = np.zeros_like(pl[key])                    # on the single node of that axis
    ref = dense.dense_step(gl, qom, dt, pl, El, Bl)
    # (i) rho, Jhat on the plane equal the lower-dimensional ones; zero elsewhere
    on = np.zeros(n3, bool)
    on[sel] = True
    on = on.reshape(-1)
    assert np.allclose(m.rho[on], ref["rho"], rtol=0, atol=1e-13 * np.abs(m.rho_abs).max())
    assert np.allclose(m.J[:, on], ref["J"], rtol=0, atol=1e-13 * np.abs(m.J_abs).max())
    assert not m.rho[~on].any() and not m.J[:, ~on].any() and not m.M[~on].any()
    # (ii) mass matrices: every slot that leaves the plane is empty; in-plane slots equal the dense M_gg'
    Md = ref["M"]                                               # [g, g', 3, 3] on the lower-dimensional grid
    idx_l = np.arange(nl[0] * nl[1] * nl[2]).reshape(nl)
    scale = np.abs(m.M_abs).max()
    checked = 0
    for o in range(27):
        off = (o // 9 - 1, (o // 3) % 3 - 1, o % 3 - 1)
        leaves = any(off[a] != 0 and (mask >> a) & 1 for a in range(3))
        Mo = m.M[on][:, o]                                      # [plane nodes, 3, 3]
        if leaves:
            assert not Mo.any(), f"slot {o} leaves the plane but holds mass"
            continue
        # neighbour g' = g + off on the lower-dimensional periodic grid; an axis with < 3 nodes folds several offsets onto
        # one pair (dense cannot separate them): compare only when every active axis has >= 3 nodes
        if any(nl[a] < 3 and not (mask >> a) & 1 for a in range(3)):
            continue
        g2 = np.roll(idx_l, shift=tuple(-off[a] if nl[a] > 1 else 0 for a in range(3)), axis=(0, 1, 2)).reshape(-1)
        assert np.allclose(Mo, Md[np.arange(g2.size), g2], rtol=0, atol=1e-13 * scale), f"slot {o}"
        checked += 1
    assert checked == (9 if bin(mask).count("1") == 1 else 3)
    # (iii) the push: velocities (all three components evolve) and the free coordinates; pinned coordinates stay
    assert np.allclose(vbar.T, ref["vbar"], rtol=0, atol=1e-14)
    for a, key in enumerate("xyz"):
        if (mask >> a) & 1:
            assert np.all(p3[key] == pos[a])
