"""Pins for oracle O1, O2, O3, O10 (encoding, TT-SVD, MPO apply, FD operators).

Every check compares the oracle with something that is NOT the oracle: the
paper's Table II (tests/golden/table_II.txt), the periodic circulant stencil of
PAPER.md:87 Eq. 6 written with np.roll, closed forms, and integer bit loops.
"""
import os

import numpy as np
import pytest

from oracle import qtt_oracle as O
from tests import dense_ref as R
import qtt_inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


# ------------------------------------------------------------------ O1 encode
@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_encode_matches_bit_loops(n):
    """PAPER.md:59-67 Eq. 3: omega_k = (x^k y^k)_2, bit 1 most significant."""
    N = 1 << n
    F = np.random.default_rng(n).standard_normal((N, N))
    T = O.encode(F)
    assert T.shape == (4,) * n
    assert np.array_equal(T.reshape(-1), R.quantics_vector(F))
    assert np.array_equal(O.decode(T), F)
    # spot check one grid point by hand: x = N-2 (1..10), y = 1 (0..01)
    x, y = N - 2, 1
    idx = tuple(2 * ((x >> (n - 1 - k)) & 1) + ((y >> (n - 1 - k)) & 1) for k in range(n))
    assert T[idx] == F[x, y]


# --------------------------------------------------------------- O2 from_dense
@pytest.mark.parametrize("n", [3, 4, 5, 6])
def test_from_dense_exact_roundtrip_and_bond_profile(n):
    N = 1 << n
    F = np.random.default_rng(10 + n).standard_normal((N, N))
    A = O.from_dense(F)
    assert rel(O.to_dense(A), F) < 1e-13
    b = O.bonds(A)
    # PAPER.md:258 footnote 2: bond l is at most min(d^l, d^(n-l))
    assert b == [min(4**l, 4 ** (n - l)) for l in range(n + 1)]


def test_closed_form_bond_two_for_sin_cos():
    """sin(2 pi x), cos(2 pi y), sin(2 pi (x+y)) have QTT bond 2; sin*cos has 4
    (exponentials are rank 1 in the quantics format)."""
    n = 6
    X, Y = I.grid(n)
    for F, want in ((np.sin(2 * np.pi * X), 2), (np.cos(2 * np.pi * Y), 2),
                    (np.sin(2 * np.pi * (X + Y)), 2), (np.sin(2 * np.pi * X) * np.cos(6 * np.pi * Y), 4)):
        A = O.from_dense(F, eps=1e-12)
        assert max(O.bonds(A)) == want, O.bonds(A)
        assert rel(O.to_dense(A), F) < 1e-11


def test_from_dense_truncation_is_bounded_by_schmidt_tails():
    """TT-SVD error lies between the worst single-bond tail and the root-sum-square
    of all tails (Schmidt values of the DENSE tensor)."""
    F = I.config1_field()
    for chi in (2, 4, 8):
        A = O.from_dense(F, chi_max=chi)
        assert max(O.bonds(A)) <= chi
        err = np.linalg.norm(O.to_dense(A) - F)
        lo, hi = R.best_rank_error_bound(F, chi)
        assert lo * (1 - 1e-12) <= err <= hi * (1 + 1e-12)


def test_from_dense_eps_rule_meets_total_error():
    """PAPER.md:238 Eq. 16: eps = ||u(chi) - u|| / ||u||."""
    F = I.config1_field()
    for eps in (1e-1, 1e-2, 1e-3):
        A = O.from_dense(F, eps=eps)
        assert rel(O.to_dense(A), F) <= eps
    # chi cap wins over eps
    A = O.from_dense(F, chi_max=3, eps=1e-6)
    assert max(O.bonds(A)) <= 3


def test_schmidt_values_match_dense():
    F = I.config1_field()
    A = O.from_dense(F)
    sv = O.schmidt_values(A)
    for b in range(1, 5):
        s_d = R.schmidt_dense(F, b)
        m = min(len(s_d), len(sv[b]))
        assert np.allclose(sv[b][:m], s_d[:m], rtol=0, atol=1e-12 * s_d[0])


# ------------------------------------------------------------- O10 operators
def test_shift_core_is_table_II():
    """Golden: the 12 entries printed in PAPER.md:409-424."""
    rows = [tuple(int(t) for t in ln.split()) for ln in open(os.path.join(GOLD, "table_II.txt"))
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 12
    C = O.shift_core(1)
    assert C.shape == (3, 4, 4, 3)
    assert np.count_nonzero(C) == 12
    for am, am1, w, wp in rows:
        assert C[am, w, wp, am1] == 1.0
    # y-direction core: same logic on the other bit
    C2 = O.shift_core(2)
    assert np.count_nonzero(C2) == 12
    sw = [0, 2, 1, 3]
    for am, am1, w, wp in rows:
        assert C2[am, sw[w], sw[wp], am1] == 1.0


@pytest.mark.parametrize("n", [2, 3, 4])
def test_dense_operator_is_periodic_circulant(n):
    """Dense D_1 == the circulant of PAPER.md:87 Eq. 6 in the quantics ordering; D^T = -D
    (PAPER.md:542); same for D_2 and the 5-point Laplacian."""
    N = 1 << n
    dx = 1.0 / N
    perm = R.interleave_index(n)
    eye = np.eye(N * N)
    for mpo, sten in ((O.mpo_d1(n, dx), R.ddx), (O.mpo_d2(n, dx), R.ddy), (O.mpo_laplacian(n, dx), R.lap5)):
        D = O.mpo_to_dense(mpo)
        # column j of the dense stencil: apply to unit fields
        Dref = np.empty_like(D)
        for j in range(N * N):
            e = np.zeros(N * N)
            e[perm[j]] = 1.0
            Dref[:, j] = sten(e.reshape(N, N), dx).reshape(-1)[perm]
        assert np.array_equal(D, Dref) or np.allclose(D, Dref, rtol=0, atol=1e-12 * np.abs(Dref).max())
        assert eye.shape == D.shape
    D1 = O.mpo_to_dense(O.mpo_d1(n, dx))
    assert np.array_equal(D1.T, -D1)
    L = O.mpo_to_dense(O.mpo_laplacian(n, dx))
    assert np.array_equal(L.T, L)


def test_mpo_bond_dims():
    n = 6
    for mpo, D in ((O.mpo_d1(n, 1 / 64), 3), (O.mpo_d2(n, 1 / 64), 3), (O.mpo_laplacian(n, 1 / 64), 5)):
        b = [1] + [w.shape[3] for w in mpo]
        assert b == [1] + [D] * (n - 1) + [1]
        for w in mpo:
            assert w.shape[1] == 4 and w.shape[2] == 4


# ------------------------------------------------------------------- O3 apply
@pytest.mark.parametrize("n", [4, 5, 6])
def test_apply_matches_dense_stencils(n):
    N = 1 << n
    dx = 1.0 / N
    F = np.random.default_rng(n).standard_normal((N, N))
    A = O.from_dense(F)
    for mpo, sten, D in ((O.mpo_d1(n, dx), R.ddx, 3), (O.mpo_d2(n, dx), R.ddy, 3),
                         (O.mpo_laplacian(n, dx), R.lap5, 5)):
        B = O.apply_mpo(mpo, A)
        assert O.bonds(B)[1:-1] == [D * r for r in O.bonds(A)[1:-1]]
        assert rel(O.to_dense(B), sten(F, dx)) < 1e-12


def test_derivative_of_sine_is_analytic_stencil_and_rounds_to_bond_two():
    """D_1 sin(2 pi x) == cos(2 pi x) * sin(2 pi dx)/dx exactly for the central stencil."""
    n = 6
    N = 1 << n
    dx = 1.0 / N
    X, Y = I.grid(n)
    A = O.from_dense(np.sin(2 * np.pi * X), eps=1e-13)
    B = O.apply_mpo(O.mpo_d1(n, dx), A)
    want = np.cos(2 * np.pi * X) * np.sin(2 * np.pi * dx) / dx
    assert rel(O.to_dense(B), want) < 1e-12
    Br = O.round_mps(B, eps=1e-11)
    assert max(O.bonds(Br)) == 2
    # d/dy of a function of x only is zero
    Z = O.apply_mpo(O.mpo_d2(n, dx), A)
    assert np.linalg.norm(O.to_dense(Z)) < 1e-10 * np.linalg.norm(want)
    # Laplacian: -(2 - 2 cos(2 pi dx))/dx^2 * sin
    Lp = O.apply_mpo(O.mpo_laplacian(n, dx), A)
    assert rel(O.to_dense(Lp), -(2 - 2 * np.cos(2 * np.pi * dx)) / dx**2 * np.sin(2 * np.pi * X)) < 1e-11


# ---------------------------------------------------------------- stencils of any order
def _roll_stencil(F, coeffs, axis):
    K = (len(coeffs) - 1) // 2
    return sum(c * np.roll(F, -k, axis=axis) for k, c in zip(range(-K, K + 1), coeffs))


@pytest.mark.parametrize("direction", [1, 2])
@pytest.mark.parametrize("order", [2, 4, 8])
def test_mpo_stencil_equals_rolled_stencil(direction, order):
    n = 5
    dx = 1.0 / (1 << n)
    c = O.fd_coefficients(order, dx)
    W = O.mpo_stencil(n, direction, c)
    F = np.random.default_rng(order + direction).standard_normal((1 << n, 1 << n))
    got = O.to_dense(O.apply_mpo(W, O.from_dense(F)))
    want = _roll_stencil(F, c, axis=direction - 1)
    assert np.linalg.norm(got - want) <= 1e-12 * np.linalg.norm(want)
    assert [w.shape[0] for w in W[1:]] == [order + 1] * (n - 1)      # bond 2K + 1


def test_mpo_stencil_order_two_is_table_II_operator():
    """K = 1 with (-1, 0, 1) / (2 dx) is the operator of PAPER.md Table II (a different bond basis, same matrix)."""
    n = 4
    dx = 1.0 / (1 << n)
    for direction, ref in ((1, O.mpo_d1(n, dx)), (2, O.mpo_d2(n, dx))):
        A = O.mpo_to_dense(O.mpo_stencil(n, direction, O.fd_coefficients(2, dx)))
        B = O.mpo_to_dense(ref)
        assert np.max(np.abs(A - B)) <= 1e-12 * np.max(np.abs(B))


def test_mpo_stencil_convergence_orders():
    """d/dx sin(2 pi x) by the order-p stencil has error ~ dx^p: halving dx divides it by 2^p (within 15 %)."""
    for order in (2, 4, 6):
        errs = []
        for n in (4, 5):
            dx = 1.0 / (1 << n)
            X, _ = I.grid(n)
            F = np.sin(2 * np.pi * X)
            got = O.to_dense(O.apply_mpo(O.mpo_stencil(n, 1, O.fd_coefficients(order, dx)), O.from_dense(F)))
            errs.append(np.max(np.abs(got - 2 * np.pi * np.cos(2 * np.pi * X))))
        ratio = errs[0] / errs[1]
        assert 0.85 * 2**order < ratio < 1.15 * 2**order, (order, ratio)
