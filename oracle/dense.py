"""Dense hat-function brute force of the hot path -- TEST INFRASTRUCTURE (tiny grids only).

The definition with no cell, corner or neighbour-slot logic at all (PAPER.md
L49 "linear interpolation function between the particle p ... and the node N"):

    S(t)   = max(0, 1 - |t|)
    W_pg   = prod_d S( minimum_image(x_pd - X_gd) / Delta_d )          for EVERY node g
    F_p    = sum_g W_pg F_g                                            (F = E^{n+theta}, B^n)
    alpha  = (I - [b]x + b b^T) / (1 + |b|^2),  b = beta B_p           (Eq. 2)
    rho_g  = sum_p q_p W_pg / V;   J_g = sum_p q_p W_pg alpha_p v_p / V            (Eq. 1)
    M_gg'  = sum_p q_p beta W_pg W_pg' alpha_p / V   for ALL node pairs (g, g')    (Eq. 3)
    vbar   = alpha (v + beta E_p);  v' = 2 vbar - v;  x' = x + dt v'               (Eq. 6-8)

O(P * nodes^2) memory/time: grids of <= ~5^3 nodes, needs >= 3 nodes per axis to be comparable
with 27-slot storage.
"""
from __future__ import annotations

import numpy as np


def hat_weights(grid, x, y, z):
    """W[p, g] for every node g = (i*ny + j)*nz + k."""
    nx, ny, nz, dx, dy, dz = grid

    def axis(pos, n, d):
        L = n * d
        X = np.arange(n) * d
        r = pos[:, None] - X[None, :]
        r = r - L * np.round(r / L)          # minimum image
        return np.maximum(0.0, 1.0 - np.abs(r) / d)

    wx, wy, wz = axis(x, nx, dx), axis(y, ny, dy), axis(z, nz, dz)
    W = wx[:, :, None, None] * wy[:, None, :, None] * wz[:, None, None, :]
    return W.reshape(x.shape[0], nx * ny * nz)


def cross_matrix(b):
    """[b]x with [b]x v = b x v, batched over the leading axis."""
    Z = np.zeros(b.shape[0])
    return np.stack([np.stack([Z, -b[:, 2], b[:, 1]], -1),
                     np.stack([b[:, 2], Z, -b[:, 0]], -1),
                     np.stack([-b[:, 1], b[:, 0], Z], -1)], -2)


def dense_step(grid, qom, dt, part, E, B):
    """Returns dict(rho[g], J[3,g], Mdense[g,g',3,3], vbar[p,3], vnew[p,3], xnew[p,3] unwrapped)."""
    nx, ny, nz, dx, dy, dz = grid
    V = dx * dy * dz
    beta = qom * dt / 2.0
    W = hat_weights(grid, part["x"], part["y"], part["z"])            # [p, g]
    Ep = W @ E.T                                                      # [p, 3]
    Bp = W @ B.T
    b = beta * Bp
    eye = np.eye(3)[None]
    alpha = (eye - cross_matrix(b) + b[:, :, None] * b[:, None, :]) / (1.0 + (b * b).sum(-1))[:, None, None]
    v = np.stack([part["u"], part["v"], part["w"]], -1)
    q = part["q"]
    vhat = np.einsum("pij,pj->pi", alpha, v)
    rho = (q[:, None] * W).sum(0) / V
    J = np.einsum("p,pg,pi->ig", q, W, vhat) / V
    Md = np.einsum("p,pg,ph,pij->ghij", q * beta, W, W, alpha) / V
    vbar = np.einsum("pij,pj->pi", alpha, v + beta * Ep)
    vnew = 2.0 * vbar - v
    xnew = np.stack([part["x"], part["y"], part["z"]], -1) + dt * vnew
    return dict(rho=rho, J=J, M=Md, vbar=vbar, vnew=vnew, xnew=xnew, alpha=alpha, Ep=Ep, Bp=Bp, W=W)


def stencil_to_dense(grid, M):
    """Expand M[g][27][3][3] to dense [g][g'][3][3] (needs >= 3 nodes per axis)."""
    nx, ny, nz = grid[:3]
    nodes = nx * ny * nz
    out = np.zeros((nodes, nodes, 3, 3))
    for i in range(nx):
        for j in range(ny):
            for k in range(nz):
                g = (i * ny + j) * nz + k
                for di in (-1, 0, 1):
                    for dj in (-1, 0, 1):
                        for dk in (-1, 0, 1):
                            o = (di + 1) * 9 + (dj + 1) * 3 + (dk + 1)
                            g2 = (((i + di) % nx) * ny + (j + dj) % ny) * nz + (k + dk) % nz
                            out[g, g2] += M[g, o]
    return out
