"""CPU ORACLE (TEST INFRASTRUCTURE, NOT PRODUCT CODE), 3D part: the quantics encoding with physical
dimension d = 8 and the finite-difference MPOs on a 2^n x 2^n x 2^n periodic grid (SURVEY.md section 8f next-4,
first half; "the methods outlined here can be generalized to 3D"; reading 26).

Plain NumPy fp64, same rules as oracle/qtt_oracle.py (whose apply_mpo, hadamard, lincomb, round_mps, round_product,
dot and diff_norm take the physical dimension from the core shapes and are used as they are); shares no code with
the CUDA path.  Only tests/ may import this module.

Data model: a field F[x][y][z], N = 2**n points per direction, becomes an n-site MPS whose site k carries
omega_k = 4 x_bit_k + 2 y_bit_k + z_bit_k (Eq. 3 with one more coordinate: the bits of one length
scale share a site), bit 1 the most significant.  Cores (r_{k-1}, 8, r_k); MPO cores (D_{k-1}, 8, 8, D_k) indexed
[alpha_{k-1}][omega (output)][omega' (input)][alpha_k].

  P1  encode3 / decode3            PAPER.md:59-67 Eq. 3 (three coordinates)
  P2  from_dense3 / to_dense3      PAPER.md:67-72 Eq. 4 (R->L TT-SVD, the rank rule of O6)
  P3  mpo_stencil3, mpo_d3, mpo_laplacian3    PAPER.md:391-424 App. A (the carry automaton of Table II on the bit of
                                   the shifted coordinate; "same logic"); 7-point Laplacian of bond 7
  P4  rhs3 / rk4_step3             PAPER.md:49-53 Eq. 2 without pressure, three components; Eq. 11

Pins (tests/test_oracle_3d.py): encode3 against index arithmetic written out bit by bit; from_dense3/to_dense3 round
trip and the dense TT-SVD error identity; every MPO against np.roll stencils on the dense cube; separable fields
(bond 1 and 2 closed forms); the 2D operators of O10 embedded in 3D (a field constant in z); rk4_step3 against a
dense RK4 of the same stencils.
"""
from __future__ import annotations

import math
import numpy as np

from . import qtt_oracle as o2

D3 = 8  # physical dimension 2^3 (PAPER.md:407 with three coordinates)


# --------------------------------------------------------------------------- P1
def encode3(F: np.ndarray) -> np.ndarray:
    """Dense F[x][y][z] (N^3) -> tensor U[w_1]...[w_n], w_k = 4 x_bit_k + 2 y_bit_k + z_bit_k, bit 1 most significant."""
    N = F.shape[0]
    n = int(round(math.log2(N)))
    assert F.shape == (N, N, N) and (1 << n) == N
    T = np.asarray(F, dtype=np.float64).reshape((2,) * (3 * n))  # x bits msb..lsb, y bits, z bits
    perm = []
    for k in range(n):
        perm += [k, n + k, 2 * n + k]
    return T.transpose(perm).reshape((D3,) * n)


def decode3(U: np.ndarray) -> np.ndarray:
    """Inverse of :func:`encode3`."""
    n = U.ndim
    N = 1 << n
    T = U.reshape((2, 2, 2) * n)  # x1 y1 z1 x2 y2 z2 ...
    perm = [3 * k for k in range(n)] + [3 * k + 1 for k in range(n)] + [3 * k + 2 for k in range(n)]
    return T.transpose(perm).reshape(N, N, N)


# --------------------------------------------------------------------------- P2
def from_dense3(F: np.ndarray, chi_max: int = 1 << 30, eps: float = 0.0):
    """TT-SVD right-to-left (Eq. 4; the steps of O2 with d = 8): for k = n..2, SVD of the
    8^{k-1} x (8 r_k) unfolding, rank by the rule of O6, core_k = V^T, carry U S; core_1 = carry."""
    U = encode3(F)
    n = U.ndim
    nrm = float(np.linalg.norm(U))
    delta = eps * nrm / math.sqrt(max(n - 1, 1)) if eps > 0 else None
    cores = [None] * n
    carry = U.reshape(-1, 1)
    r = 1
    for k in range(n, 1, -1):
        M = carry.reshape(D3 ** (k - 1), D3 * r)
        Um, s, Vt = np.linalg.svd(M, full_matrices=False)
        rk = o2._rank_rule(s, chi_max, delta)
        cores[k - 1] = Vt[:rk].reshape(rk, D3, r)
        carry = Um[:, :rk] * s[:rk]
        r = rk
    cores[0] = carry.reshape(1, D3, r)
    return cores


def to_dense3(cores) -> np.ndarray:
    """MPS -> dense F[x][y][z]."""
    return decode3(o2.to_tensor(cores))


# --------------------------------------------------------------------------- P3
def mpo_stencil3(n: int, direction: int, coeffs):
    """(O F)[.., x_dir, ..] = sum_{k=-K..K} coeffs[k + K] F[.., x_dir + k, ..] (periodic) as an MPO of bond 2K + 1:
    the construction of App. A as in O10's mpo_stencil -- bond index = carry + K of the addition
    x_dir + k, travelling from the least- to the most-significant site; at a site with output bit b of the shifted
    coordinate and incoming carry c the input bit is (b + c) mod 2, the outgoing carry floor((b + c) / 2); the other
    two bits pass unchanged.  direction 1, 2, 3 = x, y, z = bit 2, 1, 0 of omega.  L = ones, R = coeffs."""
    coeffs = np.asarray(coeffs, dtype=np.float64)
    assert direction in (1, 2, 3) and len(coeffs) % 2 == 1 and n >= 2
    K = (len(coeffs) - 1) // 2
    D = 2 * K + 1
    pos = 3 - direction
    C = np.zeros((D, D3, D3, D))
    for cin in range(-K, K + 1):
        for w in range(D3):
            b = (w >> pos) & 1
            s = b + cin
            bin_ = s % 2
            cout = (s - bin_) // 2
            wp = (w & ~(1 << pos)) | (bin_ << pos)
            C[cout + K, w, wp, cin + K] = 1.0
    cores = [C.copy() for _ in range(n)]
    cores[0] = np.einsum("a,awvb->wvb", np.ones(D), C)[None]
    cores[-1] = np.einsum("awvb,b->awv", C, coeffs)[..., None]
    return cores


def _channel_core3(channels):
    """Bulk core of Table II for a list of channels (coordinate j, shift s = +-1); channel 0 = identity.
    A channel c > 0 at a site flips the bit of its coordinate (input bit = output bit + s mod 2) and stays in c when the
    addition carries on to the more significant site (s = +1: output bit 1; s = -1: output bit 0), else falls to channel 0
    -- the entries alpha_{m+1} = 1, 2 of Table II, with the bit of coordinate j in place of the x bit."""
    D = 1 + len(channels)
    C = np.zeros((D, D3, D3, D))
    for w in range(D3):
        C[0, w, w, 0] = 1.0
    for c, (j, shift) in enumerate(channels, start=1):
        pos = 3 - j
        for w in range(D3):
            b = (w >> pos) & 1
            wp = w ^ (1 << pos)
            onward = (b == 1) if shift > 0 else (b == 0)
            C[c if onward else 0, w, wp, c] = 1.0
    return C


def _fold3(C, n, R):
    cores = [C.copy() for _ in range(n)]
    cores[0] = np.einsum("a,awvb->wvb", np.ones(C.shape[0]), C)[None]   # L = ones on the most-significant end
    cores[-1] = np.einsum("awvb,b->awv", C, np.asarray(R, dtype=np.float64))[..., None]  # R on the least-significant end
    return cores


def mpo_d3(n: int, direction: int, dx: float):
    """Central difference along one direction (PAPER.md:395-404 Eq. A1-A3): (F[x+1] - F[x-1]) / (2 dx), bond 3, channels
    identity / +1 / -1 as in Table II, L = (1,1,1), R = (0, 1, -1) / (2 dx)."""
    assert direction in (1, 2, 3) and n >= 2
    return _fold3(_channel_core3([(direction, +1), (direction, -1)]), n, np.array([0.0, 1.0, -1.0]) / (2.0 * dx))


def mpo_laplacian3(n: int, dx: float):
    """7-point Laplacian, bond 7 (reading 3 with three coordinates): channel 0 = identity, channels 2j-1 / 2j = shift
    by +1 / -1 along direction j; L = ones, R = (-6, 1, 1, 1, 1, 1, 1) / dx^2."""
    assert n >= 2
    ch = [(j, s) for j in (1, 2, 3) for s in (+1, -1)]
    return _fold3(_channel_core3(ch), n, np.array([-6.0, 1, 1, 1, 1, 1, 1]) / dx**2)


# --------------------------------------------------------------------------- P4
def rhs3(u, Dj, Lap, Re, chi_max, eps=0.0, chi_work=None):
    """f_i = -sum_{j=1..3} u_j (.) D_j u_i + (1/Re) Lap u_i, i = 1..3 (Eq. 2 without pressure, convective
    form, reading 4), one rounding after every apply, product and sum (reading 7)."""
    f = []
    for i in range(3):
        g = [o2.round_mps(o2.apply_mpo(Dj[j], u[i]), chi_max, eps) for j in range(3)]
        lap = o2.round_mps(o2.apply_mpo(Lap, u[i]), chi_max, eps)
        c = [o2.round_product(u[j], g[j], chi_max, eps, chi_work) for j in range(3)]
        f.append(o2.round_mps(o2.lincomb([(-1.0, c[0]), (-1.0, c[1]), (-1.0, c[2]), (1.0 / Re, lap)]), chi_max, eps))
    return f


def rk4_step3(u, Dj, Lap, Re, dt, chi_max, eps=0.0, chi_work=None):
    """Classical RK4 (Eq. 11) on the MPS triple; roundings and the final 5-term sum as in O9."""
    def stage(k, h):
        return [o2.round_mps(o2.lincomb([(1.0, u[i]), (h, k[i])]), chi_max, eps) for i in range(3)]

    k1 = rhs3(u, Dj, Lap, Re, chi_max, eps, chi_work)
    k2 = rhs3(stage(k1, dt / 2), Dj, Lap, Re, chi_max, eps, chi_work)
    k3 = rhs3(stage(k2, dt / 2), Dj, Lap, Re, chi_max, eps, chi_work)
    k4 = rhs3(stage(k3, dt), Dj, Lap, Re, chi_max, eps, chi_work)
    return [
        o2.round_mps(
            o2.lincomb([(1.0, u[i]), (dt / 6, k1[i]), (dt / 3, k2[i]), (dt / 3, k3[i]), (dt / 6, k4[i])]), chi_max, eps)
        for i in range(3)
    ]
