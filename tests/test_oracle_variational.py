"""Pins for the oracle's variational stage (Sec. II.C, App. B Eq. B3-B6, B20-B24).

What fixes it other than itself: the DENSE normal equations of the same cost function (the minimiser of Theta over all
fields solves (I + mu h^2 D^T D) v = a - h B, a plain linear solve on a 2^3 / 2^4 grid), finite differences of Theta
(stationarity at the returned centre tensors when the bonds really truncate), the dense operator product, and the
physics the penalty is there for (the divergence goes down as mu goes up)."""
import math

import numpy as np
import pytest

from oracle import qtt_oracle as O
import qtt_inputs as I


def fields(n, seed, k=4):
    N = 1 << n
    rng = np.random.default_rng(seed)
    X, Y = I.grid(n)
    out = []
    for s in range(k):
        F = np.zeros((N, N))
        for kx in range(-2, 3):
            for ky in range(-2, 3):
                F += rng.standard_normal() / (1 + kx * kx + ky * ky) * np.cos(2 * np.pi * (kx * X + ky * Y) + rng.uniform(0, 6.28))
        out.append(F + 0.05 * rng.standard_normal((N, N)))
    return out


def dense_minimiser(a, Bm, D1, D2, h, mu):
    M1, M2 = O.mpo_to_dense(D1), O.mpo_to_dense(D2)
    Dd = np.hstack([M1, M2])
    nn = M1.shape[0]
    A = np.eye(2 * nn) + mu * h * h * Dd.T @ Dd
    g = np.concatenate([O.to_tensor(a[i]).reshape(-1) - h * O.to_tensor(Bm[i]).reshape(-1) for i in range(2)])
    return np.linalg.solve(A, g), A, g


def theta_dense(v, a, Bm, D1, D2, h, mu):
    M1, M2 = O.mpo_to_dense(D1), O.mpo_to_dense(D2)
    t = lambda x: O.to_tensor(x).reshape(-1)
    th = mu * np.linalg.norm(M1 @ t(v[0]) + M2 @ t(v[1])) ** 2
    for i in range(2):
        th += np.linalg.norm((t(v[i]) - t(a[i])) / h + t(Bm[i])) ** 2
    return th


def test_mpo_product_is_the_operator_product():
    n, dx = 4, 1 / 16
    D1, D2 = O.mpo_d1(n, dx), O.mpo_d2(n, dx)
    for A, B in ((D1, D2), (D2, D2), (D1, D1)):
        P = O.mpo_product(A, B)
        assert np.allclose(O.mpo_to_dense(P), O.mpo_to_dense(A) @ O.mpo_to_dense(B), atol=1e-9)
        assert [c.shape[0] for c in P[1:]] == [9] * (n - 1)


def test_cost_function_is_eq_b6_on_dense_fields():
    n, dx, h, mu = 4, 1 / 16, 2e-2, 30.0
    F = fields(n, 0, 6)
    v, a, Bm = [O.from_dense(F[0]), O.from_dense(F[1])], [O.from_dense(F[2]), O.from_dense(F[3])], [O.from_dense(F[4]), O.from_dense(F[5])]
    D1, D2 = O.mpo_d1(n, dx), O.mpo_d2(n, dx)
    from tests import dense_ref as R
    want = mu * np.sum((R.ddx(F[0], dx) + R.ddy(F[1], dx)) ** 2) + sum(np.sum(((F[i] - F[2 + i]) / h + F[4 + i]) ** 2) for i in range(2))
    assert abs(O.variational_cost(v, a, Bm, D1, D2, h, mu) - want) <= 1e-11 * want


@pytest.mark.parametrize("n,mu,h", [(3, 40.0, 2e-2), (4, 50.0, 1e-2), (4, 25e4, 1e-3)])
def test_full_bond_stage_equals_dense_normal_equations(n, mu, h):
    """With untruncated bonds the one-site sweeps reach the minimiser of Theta over ALL fields: the solution of the dense
    normal equations; mu = 25e4 is the paper's penalty."""
    dx = 1.0 / (1 << n)
    F = fields(n, n, 6)
    a, Bm = [O.from_dense(F[0]), O.from_dense(F[1])], [O.from_dense(F[2]), O.from_dense(F[3])]
    v0 = [O.from_dense(F[4]), O.from_dense(F[5])]
    D1, D2 = O.mpo_d1(n, dx), O.mpo_d2(n, dx)
    sol, A, g = dense_minimiser(a, Bm, D1, D2, h, mu)
    info = {}
    V = O.variational_stage(v0, a, Bm, D1, D2, h, mu, max_sweeps=40, sweep_tol=1e-15, cg_maxit=2000, cg_tol=1e-13, info=info)
    got = np.concatenate([O.to_tensor(V[i]).reshape(-1) for i in range(2)])
    assert np.linalg.norm(got - sol) <= 1e-9 * np.linalg.norm(sol)
    assert O.bonds(V[0]) == O.bonds(v0[0])
    # Theta at the minimiser, from the dense definition
    th = theta_dense(V, a, Bm, D1, D2, h, mu)
    assert abs(th - O.variational_cost(V, a, Bm, D1, D2, h, mu)) <= 1e-9 * max(th, 1.0)
    assert th <= theta_dense(v0, a, Bm, D1, D2, h, mu)


def test_truncated_stage_is_stationary_and_decreases_theta():
    """Bonds that really truncate (chi = 3 on a 2^5 grid): the result is no longer the dense minimiser, but Theta must be
    stationary with respect to the centre tensors (Eq. B22), checked by central finite differences of the cost function,
    and no sampled perturbation of any core lowers it."""
    n, chi, mu, h = 5, 3, 200.0, 1e-2
    dx = 1.0 / (1 << n)
    F = fields(n, 7, 6)
    a, Bm = [O.from_dense(F[0], 6), O.from_dense(F[1], 6)], [O.from_dense(F[2], 6), O.from_dense(F[3], 6)]
    v0 = [O.from_dense(F[0], chi), O.from_dense(F[1], chi)]
    D1, D2 = O.mpo_d1(n, dx), O.mpo_d2(n, dx)
    cost = lambda v: O.variational_cost(v, a, Bm, D1, D2, h, mu)
    info = {}
    V = O.variational_stage(v0, a, Bm, D1, D2, h, mu, max_sweeps=60, sweep_tol=1e-14, cg_maxit=500, cg_tol=1e-13, info=info)
    assert max(O.bonds(V[0])) == chi
    t0, t1 = cost(v0), cost(V)
    assert t1 < t0
    # stationarity in the centre tensors (site 1 after a full sweep) of both components
    rng = np.random.default_rng(1)

    def fd_grad(v, i, k, idx, e):
        vp = [[c.copy() for c in v[0]], [c.copy() for c in v[1]]]
        vm = [[c.copy() for c in v[0]], [c.copy() for c in v[1]]]
        vp[i][k][idx] += e
        vm[i][k][idx] -= e
        return (cost(vp) - cost(vm)) / (2 * e)

    scale = max(abs(fd_grad(v0, i, 0, (0, w, 0), 1e-5)) for i in range(2) for w in range(4))
    for i in range(2):
        for _ in range(6):
            idx = (0, int(rng.integers(4)), int(rng.integers(V[i][0].shape[2])))
            assert abs(fd_grad(V, i, 0, idx, 1e-5)) <= 1e-5 * scale
    # local minimum with respect to every core (the cost is quadratic and convex in each single core)
    for _ in range(10):
        i, k = int(rng.integers(2)), int(rng.integers(n))
        vp = [[c.copy() for c in V[0]], [c.copy() for c in V[1]]]
        vp[i][k] = vp[i][k] + 1e-3 * np.linalg.norm(vp[i][k]) * rng.standard_normal(vp[i][k].shape) / math.sqrt(vp[i][k].size)
        assert cost(vp) >= t1 * (1 - 1e-12)


def test_penalty_removes_divergence_and_paper_cg_limits_hold():
    """mu is the incompressibility penalty: the larger mu, the smaller ||D1 v1 + D2 v2||; with the
    paper's solver settings (100 CG iterations, 1e-5) every local solve respects the iteration limit."""
    n, h = 4, 1e-2
    dx = 1.0 / (1 << n)
    F = fields(n, 11, 4)
    a, Bm = [O.from_dense(F[0]), O.from_dense(F[1])], [O.from_dense(0 * F[2]), O.from_dense(0 * F[3])]
    D1, D2 = O.mpo_d1(n, dx), O.mpo_d2(n, dx)
    div = lambda v: np.linalg.norm(O.to_dense(O.apply_mpo(D1, v[0])) + O.to_dense(O.apply_mpo(D2, v[1])))
    d_prev = div(a)
    for mu in (1e2, 1e4, 25e4):
        info = {}
        V = O.variational_stage(a, a, Bm, D1, D2, h, mu, info=info)
        assert max(info["cg_iterations"]) <= 100 and info["sweeps"] <= 20
        d = div(V)
        assert d < d_prev
        d_prev = d
    assert d_prev < 0.2 * div(a)
