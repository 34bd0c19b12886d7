"""Pins of the 3D (d = 8) oracle (oracle/qtt_oracle_3d.py, reading 26) against
what the mathematics fixes: index arithmetic written out bit by bit, np.roll stencils on the dense cube, separable
closed forms, the 2D operators embedded in 3D, the TT-SVD error identity and a dense RK4 of the same stencils."""
import numpy as np
import pytest

from oracle import qtt_oracle as o2
from oracle import qtt_oracle_3d as o3
from qtt_inputs import fields


def _rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def test_encode3_bit_by_bit():
    n = 3
    N = 1 << n
    F = np.random.default_rng(1).standard_normal((N, N, N))
    U = o3.encode3(F)
    assert U.shape == (8,) * n
    for x in range(N):
        for y in range(N):
            for z in range(N):
                w = []
                for k in range(n):  # bit 1 = most significant
                    sh = n - 1 - k
                    w.append(4 * ((x >> sh) & 1) + 2 * ((y >> sh) & 1) + ((z >> sh) & 1))
                assert U[tuple(w)] == F[x, y, z]
    assert np.array_equal(o3.decode3(U), F)


def test_from_dense3_exact_and_truncation_identity():
    n = 3
    F = np.random.default_rng(2).standard_normal((8, 8, 8))
    A = o3.from_dense3(F)
    assert [c.shape[1] for c in A] == [8] * n
    assert o2.bonds(A) == [1, 8, 8, 1]
    assert _rel(o3.to_dense3(A), F) < 1e-13
    # truncated: the error is bounded by the root-sum-square of the discarded singular values of the unfoldings and
    # is at least the best rank-chi error of every unfolding (Eckart-Young)
    chi = 3
    B = o3.from_dense3(F, chi)
    assert max(o2.bonds(B)) == chi
    err = np.linalg.norm(o3.to_dense3(B) - F)
    U = o3.encode3(F)
    tails = []
    for k in range(1, n):
        s = np.linalg.svd(U.reshape(8**k, -1), compute_uv=False)
        tails.append(np.sqrt(np.sum(s[chi:] ** 2)))
    assert err >= max(tails) * (1 - 1e-12)
    assert err <= np.sqrt(np.sum(np.square(tails))) * (1 + 1e-12)


def test_separable_fields_have_the_closed_form_bonds():
    n = 4
    N = 1 << n
    t = 2 * np.pi * np.arange(N) / N
    X, Y, Z = np.meshgrid(t, t, t, indexing="ij")
    # a product of one-coordinate exponentials has bond 1; sin(X + Y + Z) bond 2; the Taylor-Green component bond <= 8
    for F, r in ((np.exp(0.3 * X / (2 * np.pi)) * np.exp(-0.2 * Y) * np.exp(0.1 * Z), 1), (np.sin(X + Y + Z), 2)):
        A = o3.from_dense3(F, eps=1e-12)
        assert max(o2.bonds(A)) == r
        assert _rel(o3.to_dense3(A), F) < 1e-11
    u1, _, _ = fields.taylor_green_3d(n, noise=0.0)
    A = o3.from_dense3(u1, eps=1e-12)
    assert max(o2.bonds(A)) <= 8
    assert _rel(o3.to_dense3(A), u1) < 1e-11


@pytest.mark.parametrize("direction", [1, 2, 3])
def test_mpo_d3_is_the_rolled_central_difference(direction):
    n = 3
    N = 1 << n
    dx = 1.0 / N
    F = np.random.default_rng(3 + direction).standard_normal((N, N, N))
    A = o3.from_dense3(F)
    G = o3.to_dense3(o2.apply_mpo(o3.mpo_d3(n, direction, dx), A))
    ax = direction - 1
    ref = (np.roll(F, -1, axis=ax) - np.roll(F, 1, axis=ax)) / (2 * dx)
    assert _rel(G, ref) < 1e-13
    # the same operator built as a stencil MPO (another bond basis: carries -1, 0, +1)
    S = o3.to_dense3(o2.apply_mpo(o3.mpo_stencil3(n, direction, np.array([-1.0, 0.0, 1.0]) / (2 * dx)), A))
    assert _rel(G, S) < 1e-13
    # the bulk core restricted to a field that does not depend on the other two coordinates is Table II verbatim
    if direction == 1:
        C = o3._channel_core3([(1, +1), (1, -1)])
        T2 = np.zeros((3, 4, 4, 3))
        for am, am1, w, wp in o2._TABLE_II:
            T2[am, w, wp, am1] = 1.0
        # omega_3d = 2 * omega_2d + z_bit: take z_bit = 0 on both sides
        assert np.array_equal(C[:, 0::2, 0::2, :], T2)

    idx = [2, 5, 7]
    ip, im = list(idx), list(idx)
    ip[ax] = (idx[ax] + 1) % N
    im[ax] = (idx[ax] - 1) % N
    assert abs(G[tuple(idx)] - (F[tuple(ip)] - F[tuple(im)]) / (2 * dx)) < 1e-11


@pytest.mark.parametrize("direction", [1, 2, 3])
def test_mpo_stencil3_wide_stencils(direction):
    n = 4
    N = 1 << n
    F = np.random.default_rng(7).standard_normal((N, N, N))
    A = o3.from_dense3(F, 64)
    Fd = o3.to_dense3(A)
    c = np.array([0.3, -1.1, 0.0, 2.0, 0.7])  # offsets -2..2, asymmetric on purpose
    G = o3.to_dense3(o2.apply_mpo(o3.mpo_stencil3(n, direction, c), A))
    ref = sum(c[k + 2] * np.roll(Fd, -k, axis=direction - 1) for k in range(-2, 3))
    assert _rel(G, ref) < 1e-13


def test_mpo_laplacian3_is_the_7_point_stencil_and_sums_the_1d_ones():
    n = 3
    N = 1 << n
    dx = 1.0 / N
    F = np.random.default_rng(11).standard_normal((N, N, N))
    A = o3.from_dense3(F)
    L = o3.mpo_laplacian3(n, dx)
    assert [c.shape[0] for c in L] == [1, 7, 7] and L[0].shape[1:3] == (8, 8)
    G = o3.to_dense3(o2.apply_mpo(L, A))
    ref = -6 * F
    for ax in range(3):
        ref = ref + np.roll(F, 1, axis=ax) + np.roll(F, -1, axis=ax)
    assert _rel(G, ref / dx**2) < 1e-13
    # = sum over directions of the 3-point second difference built as a stencil MPO
    S = sum(o3.to_dense3(o2.apply_mpo(o3.mpo_stencil3(n, d, np.array([1.0, -2.0, 1.0]) / dx**2), A)) for d in (1, 2, 3))
    assert _rel(G, S) < 1e-13
    # analytic: a single Fourier mode is an eigenvector with eigenvalue (2 cos(2 pi k dx) - 2) / dx^2 per coordinate
    t = 2 * np.pi * np.arange(N) / N
    X, Y, Z = np.meshgrid(t, t, t, indexing="ij")
    M = np.sin(X) * np.cos(2 * Y) * np.cos(Z)
    lam = sum((2 * np.cos(2 * np.pi * k * dx) - 2) / dx**2 for k in (1, 2, 1))
    GM = o3.to_dense3(o2.apply_mpo(L, o3.from_dense3(M)))
    assert _rel(GM, lam * M) < 1e-12


def test_2d_operators_embedded_in_3d():
    """A field constant in z: D_1, D_2 and the Laplacian act on it as the 2D operators of O10 act on the slice; D_3 kills it."""
    n = 4
    N = 1 << n
    dx = 1.0 / N
    F2 = np.random.default_rng(5).standard_normal((N, N))
    F3 = np.repeat(F2[:, :, None], N, axis=2)
    A2 = o2.from_dense(F2)
    A3 = o3.from_dense3(F3)
    for d3, W2 in ((1, o2.mpo_d1(n, dx)), (2, o2.mpo_d2(n, dx))):
        G3 = o3.to_dense3(o2.apply_mpo(o3.mpo_d3(n, d3, dx), A3))
        G2 = o2.to_dense(o2.apply_mpo(W2, A2))
        assert _rel(G3[:, :, 3], G2) < 1e-12 and _rel(G3[:, :, 0], G3[:, :, 9]) < 1e-12
    assert np.linalg.norm(o3.to_dense3(o2.apply_mpo(o3.mpo_d3(n, 3, dx), A3))) < 1e-9 * np.linalg.norm(F3) / dx
    L3 = o3.to_dense3(o2.apply_mpo(o3.mpo_laplacian3(n, dx), A3))
    L2 = o2.to_dense(o2.apply_mpo(o2.mpo_laplacian(n, dx), A2))
    assert _rel(L3[:, :, 6], L2) < 1e-11


def test_hadamard_round_and_sums_with_d8():
    n = 3
    rng = np.random.default_rng(9)
    F, G = rng.standard_normal((8, 8, 8)), rng.standard_normal((8, 8, 8))
    A, B = o3.from_dense3(F, 5), o3.from_dense3(G, 4)
    Fd, Gd = o3.to_dense3(A), o3.to_dense3(B)
    assert _rel(o3.to_dense3(o2.hadamard(A, B)), Fd * Gd) < 1e-13
    assert _rel(o3.to_dense3(o2.lincomb([(2.0, A), (-0.5, B), (1.0, A)])), 3 * Fd - 0.5 * Gd) < 1e-13
    # exact working bond: the zip-up is round(hadamard); rounding a full-rank representation changes nothing
    P = o2.round_product(A, B, 64, chi_work=10**6)
    assert _rel(o3.to_dense3(P), Fd * Gd) < 1e-12
    Q = o2.round_mps(o2.hadamard(A, B), 64)
    assert o2.diff_norm(P, Q) < 1e-12 * o2.norm(Q)
    # truncating: equals the dense TT-SVD truncation of the product up to the quasi-optimality bound, above Eckart-Young
    chi = 3
    T = o2.round_mps(o2.hadamard(A, B), chi)
    err = np.linalg.norm(o3.to_dense3(T) - Fd * Gd)
    U = o3.encode3(Fd * Gd)
    tails = [np.sqrt(np.sum(np.linalg.svd(U.reshape(8**k, -1), compute_uv=False)[chi:] ** 2)) for k in range(1, n)]
    assert max(tails) * (1 - 1e-12) <= err <= np.sqrt(np.sum(np.square(tails))) * (1 + 1e-12)


def _dense_rhs3(u, Re, dx):
    def d(F, ax):
        return (np.roll(F, -1, axis=ax) - np.roll(F, 1, axis=ax)) / (2 * dx)

    def lap(F):
        return sum(np.roll(F, 1, axis=a) + np.roll(F, -1, axis=a) - 2 * F for a in range(3)) / dx**2

    return [-(u[0] * d(u[i], 0) + u[1] * d(u[i], 1) + u[2] * d(u[i], 2)) + lap(u[i]) / Re for i in range(3)]


def test_rk4_step3_matches_dense_rk4_at_full_bonds():
    n = 3
    N = 1 << n
    dx = 1.0 / N
    Re, dt = 50.0, 1e-3
    u = list(fields.taylor_green_3d(n, seed=0, noise=1e-2))
    U = [o3.from_dense3(f) for f in u]
    Dj = [o3.mpo_d3(n, j, dx) for j in (1, 2, 3)]
    Lap = o3.mpo_laplacian3(n, dx)
    out = o3.rk4_step3(U, Dj, Lap, Re, dt, chi_max=64, chi_work=10**6)
    k1 = _dense_rhs3(u, Re, dx)
    k2 = _dense_rhs3([a + dt / 2 * b for a, b in zip(u, k1)], Re, dx)
    k3 = _dense_rhs3([a + dt / 2 * b for a, b in zip(u, k2)], Re, dx)
    k4 = _dense_rhs3([a + dt * b for a, b in zip(u, k3)], Re, dx)
    for i in range(3):
        ref = u[i] + dt / 6 * (k1[i] + 2 * k2[i] + 2 * k3[i] + k4[i])
        assert _rel(o3.to_dense3(out[i]), ref) < 1e-12
        assert _rel(ref, u[i]) > 1e-6  # the step did something
