"""Dense N x N brute force used ONLY to pin the oracle (and, through it, the GPU
path): periodic stencils with np.roll, dense RK4 of the same right-hand side, and
a dense TT-SVD that works on the full tensor.  Independent of oracle/ (no imports
from it) so that a mistake there cannot hide here.

Fields are F[x][y] on x_j = y_j = j/N; dx = 1/N (reading 2).
"""
from __future__ import annotations

import numpy as np


def ddx(F, dx):
    """PAPER.md:87 Eq. 6: (F[x+1] - F[x-1]) / (2 dx), periodic."""
    return (np.roll(F, -1, axis=0) - np.roll(F, 1, axis=0)) / (2.0 * dx)


def ddy(F, dx):
    return (np.roll(F, -1, axis=1) - np.roll(F, 1, axis=1)) / (2.0 * dx)


def lap5(F, dx):
    """Compact 5-point Laplacian."""
    return (np.roll(F, -1, 0) + np.roll(F, 1, 0) + np.roll(F, -1, 1) + np.roll(F, 1, 1) - 4.0 * F) / dx**2


def convection_skew(ux, uy, dx):
    """PAPER.md:432-435 Eq. B2: 1/2 (u_j d_j u_i + d_j (u_j u_i)), summed over j."""
    cx = 0.5 * (ux * ddx(ux, dx) + uy * ddy(ux, dx) + ddx(ux * ux, dx) + ddy(uy * ux, dx))
    cy = 0.5 * (ux * ddx(uy, dx) + uy * ddy(uy, dx) + ddx(ux * uy, dx) + ddy(uy * uy, dx))
    return cx, cy


def rhs_dense(ux, uy, Re, dx, skew=False):
    """PAPER.md:49-53 Eq. 2 without pressure; convective form, or the skew-symmetric form of Eq. B2."""
    if skew:
        cx, cy = convection_skew(ux, uy, dx)
        return -cx + lap5(ux, dx) / Re, -cy + lap5(uy, dx) / Re
    fx = -(ux * ddx(ux, dx) + uy * ddy(ux, dx)) + lap5(ux, dx) / Re
    fy = -(ux * ddx(uy, dx) + uy * ddy(uy, dx)) + lap5(uy, dx) / Re
    return fx, fy


def rk4_dense(ux, uy, Re, dt, dx, skew=False):
    """PAPER.md:126 Eq. 11."""
    k1 = rhs_dense(ux, uy, Re, dx, skew)
    k2 = rhs_dense(ux + dt / 2 * k1[0], uy + dt / 2 * k1[1], Re, dx, skew)
    k3 = rhs_dense(ux + dt / 2 * k2[0], uy + dt / 2 * k2[1], Re, dx, skew)
    k4 = rhs_dense(ux + dt * k3[0], uy + dt * k3[1], Re, dx, skew)
    return (ux + dt / 6 * (k1[0] + 2 * k2[0] + 2 * k3[0] + k4[0]),
            uy + dt / 6 * (k1[1] + 2 * k2[1] + 2 * k3[1] + k4[1]))


def interleave_index(n):
    """perm[p] = flat index x*N + y of the grid point whose quantics multi-index
    (w_1..w_n), w_k = 2 x_bit_k + y_bit_k (bit 1 = msb), has flat position p.
    Written with integer bit loops, not reshapes (independent of the oracle)."""
    N = 1 << n
    perm = np.empty(N * N, dtype=np.int64)
    for p in range(N * N):
        x = y = 0
        for k in range(n):
            w = (p >> (2 * (n - 1 - k))) & 3
            x = (x << 1) | (w >> 1)
            y = (y << 1) | (w & 1)
        perm[p] = x * N + y
    return perm


def quantics_vector(F):
    n = int(np.log2(F.shape[0]))
    return F.reshape(-1)[interleave_index(n)]


def from_quantics_vector(v, n):
    N = 1 << n
    out = np.empty(N * N)
    out[interleave_index(n)] = v
    return out.reshape(N, N)


def schmidt_dense(F, bond):
    """Singular values of the bipartition (sites 1..bond | bond+1..n) of the dense
    quantics tensor."""
    n = int(np.log2(F.shape[0]))
    v = quantics_vector(F)
    return np.linalg.svd(v.reshape(4**bond, 4 ** (n - bond)), compute_uv=False)


def best_rank_error_bound(F, chi):
    """sqrt(sum over bonds of the squared discarded Schmidt weight): upper bound
    on the TT-SVD error, and each single term a lower bound."""
    n = int(np.log2(F.shape[0]))
    tot = 0.0
    worst = 0.0
    for b in range(1, n):
        s = schmidt_dense(F, b)
        t = float(np.sum(s[chi:] ** 2))
        tot += t
        worst = max(worst, t)
    return np.sqrt(worst), np.sqrt(tot)
