"""Pins for oracle O4-O9: Hadamard, direct sum, rounding, zip-up, rhs, RK4.

Brute force on 2^4..2^6 grids, the root-sum-square truncation identity, norm
preservation, an independent dense TT-SVD, and dense RK4 of the same stencils.
"""
import numpy as np
import pytest

from oracle import qtt_oracle as O
from tests import dense_ref as R
import qtt_inputs as I


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def rand_field(n, seed):
    N = 1 << n
    return np.random.default_rng(seed).standard_normal((N, N))


def smooth_field(n, seed):
    """Random low-wavenumber field: decaying Schmidt spectrum, distinct gaps."""
    N = 1 << n
    rng = np.random.default_rng(seed)
    X, Y = I.grid(n)
    F = np.zeros((N, N))
    for kx in range(-3, 4):
        for ky in range(-3, 4):
            a, p = rng.standard_normal(), rng.uniform(0, 2 * np.pi)
            F += a / (1 + kx * kx + ky * ky) * np.cos(2 * np.pi * (kx * X + ky * Y) + p)
    return F + np.tanh((Y - 0.5) / 0.1)


# ---------------------------------------------------------------- O4 hadamard
@pytest.mark.parametrize("n", [4, 5, 6])
def test_hadamard_is_elementwise_product(n):
    F, G = rand_field(n, 1), rand_field(n, 2)
    A, B = O.from_dense(F, chi_max=6), O.from_dense(G, chi_max=5)
    C = O.hadamard(A, B)
    # bond of the product = product of the bonds (<= chi^2)
    assert O.bonds(C) == [a * b for a, b in zip(O.bonds(A), O.bonds(B))]
    assert rel(O.to_dense(C), O.to_dense(A) * O.to_dense(B)) < 1e-12
    # not symmetric in general as tensors, but as fields it is
    assert rel(O.to_dense(O.hadamard(B, A)), O.to_dense(C)) < 1e-12


# ------------------------------------------------------------------ O5 lincomb
@pytest.mark.parametrize("n", [4, 5])
def test_lincomb_is_linear_combination(n):
    Fs = [rand_field(n, s) for s in range(4)]
    As = [O.from_dense(F, chi_max=4 + s) for s, F in enumerate(Fs)]
    al = [0.5, -2.0, 1e-3, 7.0]
    S = O.lincomb(list(zip(al, As)))
    want = sum(a * O.to_dense(A) for a, A in zip(al, As))
    assert rel(O.to_dense(S), want) < 1e-13
    assert O.bonds(S)[1:-1] == [sum(O.bonds(A)[l] for A in As) for l in range(1, n)]
    Y = O.axpy(-3.0, As[0], As[1])
    assert rel(O.to_dense(Y), -3.0 * O.to_dense(As[0]) + O.to_dense(As[1])) < 1e-13


# -------------------------------------------------------------------- O6 round
def test_round_without_truncation_reconstructs():
    n = 5
    A = O.from_dense(rand_field(n, 3), chi_max=7)
    B = O.lincomb([(1.0, A), (1.0, A)])  # rank-deficient by construction
    Rr = O.round_mps(B)
    assert rel(O.to_dense(Rr), 2 * O.to_dense(A)) < 1e-13


def test_qr_sweep_preserves_norm_and_orthogonality():
    n = 6
    A = O.apply_mpo(O.mpo_laplacian(n, 1 / 64), O.from_dense(smooth_field(n, 0), chi_max=9))
    want = np.linalg.norm(O.to_dense(A))
    C = O._sweep_lr(A)
    assert abs(np.linalg.norm(C[-1]) - want) <= 4e-15 * want
    for c in C[:-1]:
        M = c.reshape(-1, c.shape[2])
        assert np.allclose(M.T @ M, np.eye(M.shape[1]), atol=1e-13)
    Rr = O.round_mps(A, chi_max=5)
    for c in Rr[1:]:
        M = c.reshape(c.shape[0], -1)
        assert np.allclose(M @ M.T, np.eye(M.shape[0]), atol=1e-13)


@pytest.mark.parametrize("chi", [2, 4, 8])
def test_truncation_error_equals_rss_of_discarded_singular_values(chi):
    """||A - round(A)||_F == sqrt(sum_bonds sum_discarded sigma^2) with EQUALITY
    (nested orthogonal projectors)."""
    n = 5
    F = I.config1_field()
    A = O.apply_mpo(O.mpo_d1(n, 1 / 32), O.from_dense(F))
    info = {}
    Rr = O.round_mps(A, chi_max=chi, info=info)
    err = np.linalg.norm(O.to_dense(A) - O.to_dense(Rr))
    rss = np.sqrt(sum(d * d for d in info["discarded"]))
    assert abs(err - rss) <= 1e-12 * max(err, 1e-300) + 1e-13 * info["norm"]
    assert abs(info["norm"] - np.linalg.norm(O.to_dense(A))) <= 1e-13 * info["norm"]


@pytest.mark.parametrize("n,chi", [(4, 3), (5, 4), (5, 8), (6, 6)])
def test_round_of_exact_equals_dense_ttsvd(n, chi):
    """round(exact MPS) == R->L TT-SVD of the dense tensor, written here independently
    on the quantics vector of tests/dense_ref.py."""
    F = smooth_field(n, n)
    A = O.apply_mpo(O.mpo_d2(n, 1.0 / (1 << n)), O.from_dense(F))
    G = O.to_dense(A)
    Rr = O.round_mps(A, chi_max=chi)
    # independent dense TT-SVD, right to left
    v = R.quantics_vector(G)
    carry, r, cores = v.reshape(-1, 1), 1, []
    for k in range(n, 1, -1):
        U, s, Vt = np.linalg.svd(carry.reshape(4 ** (k - 1), 4 * r), full_matrices=False)
        rk = min(chi, len(s))
        cores.insert(0, Vt[:rk])
        carry, r = U[:, :rk] * s[:rk], rk
    T = carry.reshape(4, -1)
    for Vt in cores:
        T = (T @ Vt.reshape(Vt.shape[0], -1)).reshape(-1, Vt.shape[1] // 4)
    dense_tt = R.from_quantics_vector(T.reshape(-1), n)
    assert rel(O.to_dense(Rr), dense_tt) < 1e-11
    assert max(O.bonds(Rr)) <= chi


def test_round_eps_rule_total_error_and_zero_state():
    n = 5
    A = O.apply_mpo(O.mpo_laplacian(n, 1 / 32), O.from_dense(I.config1_field()))
    for eps in (1e-1, 1e-2, 1e-4):
        Rr = O.round_mps(A, eps=eps)
        assert rel(O.to_dense(Rr), O.to_dense(A)) <= eps
    Z = O.lincomb([(1.0, A), (-1.0, A)])
    Zr = O.round_mps(Z, chi_max=4)
    assert np.linalg.norm(O.to_dense(Zr)) <= 1e-12 * np.linalg.norm(O.to_dense(A))
    Zr = O.round_mps([np.zeros_like(c) for c in A], chi_max=4, eps=1e-3)
    assert all(np.all(np.isfinite(c)) for c in Zr) and np.linalg.norm(O.to_dense(Zr)) == 0.0
    assert max(O.bonds(Zr)) == 1


def test_diff_norm_and_dot_match_dense():
    n = 5
    A = O.from_dense(rand_field(n, 5), chi_max=6)
    B = O.from_dense(rand_field(n, 6), chi_max=4)
    a, b = O.to_dense(A), O.to_dense(B)
    assert abs(O.dot(A, B) - np.sum(a * b)) < 1e-12 * np.linalg.norm(a) * np.linalg.norm(b)
    assert abs(O.norm(A) - np.linalg.norm(a)) < 1e-13 * np.linalg.norm(a)
    assert abs(O.diff_norm(A, B) - np.linalg.norm(a - b)) < 1e-13 * np.linalg.norm(a)
    # tiny differences are resolved (the overlap formula cannot do this, reading 19)
    Bp = [c.copy() for c in A]
    Bp[2] = Bp[2] * (1 + 1e-13)
    assert abs(O.diff_norm(A, Bp) - 1e-13 * np.linalg.norm(a)) < 1e-15 * np.linalg.norm(a)


# ------------------------------------------------------------------- O7 zip-up
@pytest.mark.parametrize("n,ca,cb,chi", [(4, 3, 3, 4), (5, 4, 3, 6), (6, 4, 4, 8)])
def test_zipup_with_large_work_bond_equals_round_of_exact_product(n, ca, cb, chi):
    A = O.from_dense(smooth_field(n, 1), chi_max=ca)
    B = O.from_dense(smooth_field(n, 2), chi_max=cb)
    exact = O.hadamard(A, B)
    want = O.round_mps(exact, chi_max=chi)
    got = O.round_product(A, B, chi_max=chi, chi_work=10**6)
    assert O.bonds(got) == O.bonds(want)
    assert rel(O.to_dense(got), O.to_dense(want)) < 1e-11
    # and both equal the dense product up to the truncation they report
    info = {}
    O.round_product(A, B, chi_max=chi, chi_work=10**6, info=info)
    rss = np.sqrt(sum(d * d for d in info["discarded"]))
    err = np.linalg.norm(O.to_dense(got) - O.to_dense(A) * O.to_dense(B))
    assert abs(err - rss) <= 1e-11 * np.linalg.norm(O.to_dense(want))


def test_zipup_config1_chain_matches_dense():
    """BASELINE config 1 (reading 20): apply (exact) -> Hadamard (exact) -> ONE round to 8,
    against the dense 32x32 result; the same through the fused product path."""
    n, chi, dx = 5, 8, 1 / 32
    F = I.config1_field()
    u8 = O.from_dense(F, chi_max=chi)
    d = O.apply_mpo(O.mpo_d1(n, dx), u8)
    w_exact = O.hadamard(u8, d)
    U8 = O.to_dense(u8)
    W = U8 * R.ddx(U8, dx)
    assert rel(O.to_dense(w_exact), W) < 1e-12
    info = {}
    w8 = O.round_mps(w_exact, chi_max=chi, info=info)
    assert O.bonds(w8) == [1, 4, 8, 8, 4, 1]
    rss = np.sqrt(sum(x * x for x in info["discarded"]))
    assert abs(np.linalg.norm(O.to_dense(w8) - W) - rss) < 1e-12 * np.linalg.norm(W)
    # fused path with an untruncating work bond gives the same state
    w8z = O.round_product(u8, d, chi_max=chi, chi_work=4096)
    assert rel(O.to_dense(w8z), O.to_dense(w8)) < 1e-11


def test_zipup_finite_work_bond_error_bound_and_convergence():
    """Finite chi_work: the result is algorithm-defined; what can be pinned is that the
    error decreases to the optimal-rounding error as chi_work grows and never beats it."""
    n, chi = 6, 6
    A = O.from_dense(smooth_field(n, 3), chi_max=6)
    B = O.from_dense(smooth_field(n, 4), chi_max=6)
    W = O.to_dense(A) * O.to_dense(B)
    best = np.linalg.norm(O.to_dense(O.round_mps(O.hadamard(A, B), chi_max=chi)) - W)
    lo, _ = R.best_rank_error_bound(W, chi)
    errs = []
    for cw in (chi, 2 * chi, 4 * chi, 36):
        got = O.round_product(A, B, chi_max=chi, chi_work=cw)
        assert max(O.bonds(got)) <= chi
        errs.append(np.linalg.norm(O.to_dense(got) - W))
        assert errs[-1] >= lo * (1 - 1e-9)
    assert abs(errs[-1] - best) < 1e-9 * np.linalg.norm(W)
    assert errs[1] <= errs[0] * (1 + 1e-9)
    assert errs[1] < 3 * best + 1e-9 * np.linalg.norm(W)
    # default work bond is 2*chi
    d1 = O.round_product(A, B, chi_max=chi)
    d2 = O.round_product(A, B, chi_max=chi, chi_work=2 * chi)
    assert all(np.array_equal(x, y) for x, y in zip(d1, d2))


# ------------------------------------------------------------- O8/O9 rhs, RK4
def _ops(n):
    dx = 1.0 / (1 << n)
    return O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx), dx


@pytest.mark.parametrize("n", [4, 5])
def test_rhs_and_rk4_at_full_rank_equal_dense(n):
    """With chi_max >= full rank nothing is discarded, so the QTT step equals dense RK4
    of the same stencils on the N x N array."""
    Dx, Dy, Lap, dx = _ops(n)
    ux, uy = smooth_field(n, 7), smooth_field(n, 8)
    Re, dt = 50.0, 1e-3
    u = [O.from_dense(ux), O.from_dense(uy)]
    chi = 4 ** (n // 2)
    f = O.rhs(u, Dx, Dy, Lap, Re, chi, chi_work=10**6)
    fx, fy = R.rhs_dense(ux, uy, Re, dx)
    assert rel(O.to_dense(f[0]), fx) < 1e-11 and rel(O.to_dense(f[1]), fy) < 1e-11
    v = O.rk4_step(u, Dx, Dy, Lap, Re, dt, chi, chi_work=10**6)
    vx, vy = R.rk4_dense(ux, uy, Re, dt, dx)
    assert rel(O.to_dense(v[0]), vx) < 1e-12 and rel(O.to_dense(v[1]), vy) < 1e-12
    # the step really moved the field (a dropped term would show)
    assert rel(vx, ux) > 1e-5


def test_rk4_is_fourth_order_in_dt_against_dense():
    """Halving dt reduces the one-step difference to a fine-dt dense reference ~32x
    (local error O(dt^5))."""
    n = 4
    Dx, Dy, Lap, dx = _ops(n)
    ux, uy = smooth_field(n, 11), smooth_field(n, 12)
    Re = 20.0
    u = [O.from_dense(ux), O.from_dense(uy)]

    def ref(T, m=64):
        a, b = ux, uy
        for _ in range(m):
            a, b = R.rk4_dense(a, b, Re, T / m, dx)
        return a

    errs = []
    for dt in (4e-3, 2e-3):
        v = O.rk4_step(u, Dx, Dy, Lap, Re, dt, 16, chi_work=10**6)
        errs.append(np.linalg.norm(O.to_dense(v[0]) - ref(dt)))
    assert 20 < errs[0] / errs[1] < 45


def test_rk4_config2_shape_small():
    """Config-2-like shear layer at n=6: u_x depends on y only and u_y on x only, so a
    modest chi discards nothing significant and the QTT step equals the dense step."""
    n = 6
    Dx, Dy, Lap, dx = _ops(n)
    ux, uy = I.shear_layer(n)
    u = [O.from_dense(ux, chi_max=16), O.from_dense(uy, chi_max=16)]
    v = O.rk4_step(u, Dx, Dy, Lap, 1e4, 1e-4, 16)
    vx, vy = R.rk4_dense(O.to_dense(u[0]), O.to_dense(u[1]), 1e4, 1e-4, dx)
    assert rel(O.to_dense(v[0]), vx) < 1e-10 and rel(O.to_dense(v[1]), vy) < 1e-10
    assert max(O.bonds(v[0])) <= 16


def test_canonical_random_is_unit_norm_left_canonical():
    raw = I.random_cores(6, 8, seed=0)
    C = O.canonical_random(raw)
    assert abs(O.norm(C) - 1.0) < 1e-13
    assert O.bonds(C) == I.bond_profile(6, 8)


# ---------------------------------------------------------------- diagnostics (Eq. 12, 16-17)
def test_fidelity_closed_forms():
    n = 6
    X, Y = I.grid(n)
    s = O.from_dense(np.sin(2 * np.pi * X))
    c = O.from_dense(np.cos(2 * np.pi * X))
    assert abs(O.fidelity(s, s) - 1.0) < 1e-13
    assert O.fidelity(s, c) < 1e-26                      # orthogonal on the periodic grid
    m = O.from_dense(np.sin(2 * np.pi * X) + np.cos(2 * np.pi * X))
    assert abs(O.fidelity(s, m) - 0.5) < 1e-13           # cos^2 of 45 degrees
    # against the dense definition on a random pair
    rng = np.random.default_rng(3)
    F, G = rng.standard_normal((64, 64)), rng.standard_normal((64, 64))
    want = np.sum(F * G) ** 2 / (np.sum(F * F) * np.sum(G * G))
    assert abs(O.fidelity(O.from_dense(F), O.from_dense(G)) - want) < 1e-13


def test_chi_eps_against_dense_truncation():
    n = 6
    X, Y = I.grid(n)
    # sin(2 pi (x + y)) has exactly two Schmidt values at every interior bipartition
    chis, chi = O.chi_eps(O.from_dense(np.sin(2 * np.pi * (X + Y))), 1e-12)
    assert chi == 2 and chis[2:n - 1] == [2] * (n - 3)
    # definition check on a generic field: truncating bipartition l of the DENSE tensor to chi_l Schmidt values gives
    # a relative error <= eps, and chi_l - 1 values do not
    rng = np.random.default_rng(5)
    F = np.tanh((Y - 0.5) / 0.1) + 0.05 * rng.standard_normal((64, 64))
    eps = 0.02
    chis, chi = O.chi_eps(O.from_dense(F), eps)
    T = O.encode(F)
    for l in range(1, n):
        s = np.linalg.svd(T.reshape(4 ** l, -1), compute_uv=False)
        err = lambda k: np.sqrt(np.sum(s[k:] ** 2)) / np.linalg.norm(s)
        assert err(chis[l]) <= eps * (1 + 1e-12)
        assert chis[l] == 1 or err(chis[l] - 1) > eps * (1 - 1e-12)
    assert chi == max(chis)


# ---------------------------------------------------------------- skew-symmetric convection (PAPER.md Eq. B2)
@pytest.mark.parametrize("n", [4, 5])
def test_skew_rhs_and_rk4_equal_dense_at_full_rank(n):
    """with nothing discarded the QTT right-hand side / RK4 step in the paper's
    skew-symmetric form equals the dense one built from np.roll stencils (an independent restatement of Eq. B2)."""
    Dx, Dy, Lap, dx = _ops(n)
    ux, uy = smooth_field(n, 17), smooth_field(n, 18)
    Re, dt = 50.0, 1e-3
    u = [O.from_dense(ux), O.from_dense(uy)]
    chi = 4 ** (n // 2)
    f = O.rhs(u, Dx, Dy, Lap, Re, chi, chi_work=10**6, skew=True)
    fx, fy = R.rhs_dense(ux, uy, Re, dx, skew=True)
    assert rel(O.to_dense(f[0]), fx) < 1e-11 and rel(O.to_dense(f[1]), fy) < 1e-11
    # the two forms differ on a field that is not divergence free: a dropped 1/2 or a missing term would show
    gx, _ = R.rhs_dense(ux, uy, Re, dx)
    assert rel(fx, gx) > 1e-3
    v = O.rk4_step(u, Dx, Dy, Lap, Re, dt, chi, chi_work=10**6, skew=True)
    vx, vy = R.rk4_dense(ux, uy, Re, dt, dx, skew=True)
    assert rel(O.to_dense(v[0]), vx) < 1e-12 and rel(O.to_dense(v[1]), vy) < 1e-12


def test_skew_convection_conserves_discrete_energy():
    """The point of Eq. B2 ("better numerical stability"): with D^T = -D the
    skew-symmetric convection does no work, sum_i <u_i, conv_i(u)> = 0 exactly, for ANY field; the convective form
    does not have this property.  Checked on the oracle's QTT result at full rank."""
    n = 5
    Dx, Dy, Lap, dx = _ops(n)
    ux, uy = smooth_field(n, 27), smooth_field(n, 28)
    u = [O.from_dense(ux), O.from_dense(uy)]
    chi = 4 ** (n // 2)
    Re = 1e300  # no diffusion: f = -convection
    f = O.rhs(u, Dx, Dy, Lap, Re, chi, chi_work=10**6, skew=True)
    work = O.dot(u[0], f[0]) + O.dot(u[1], f[1])
    scale = O.norm(u[0]) * O.norm(f[0]) + O.norm(u[1]) * O.norm(f[1])
    assert abs(work) < 1e-12 * scale
    g = O.rhs(u, Dx, Dy, Lap, Re, chi, chi_work=10**6)
    assert abs(O.dot(u[0], g[0]) + O.dot(u[1], g[1])) > 1e-4 * scale


# ---------------------------------------------------------------- TKE spectrum (Eq. 13-15)
def test_tke_spectrum_closed_forms_parseval_and_brute_force():
    n = 5
    N = 1 << n
    X, Y = I.grid(n)
    A_, B_ = 0.7, 1.3
    u1 = O.from_dense(A_ * np.sin(2 * np.pi * (3 * X + 4 * Y)))      # |k| = 5: coefficients -+ A/(2i) at +-(3,4)
    u2 = O.from_dense(B_ * np.cos(2 * np.pi * 7 * Y) + 0.25)         # |k| = 7, plus a mean flow in shell 0
    E = O.tke_spectrum(u1, u2)
    assert len(E) == int(np.floor(np.sqrt(2.0) * N / 2 + 0.5)) + 1
    want = np.zeros_like(E)
    want[5], want[7], want[0] = A_**2 / 4, B_**2 / 4, 0.25**2 / 2
    assert np.max(np.abs(E - want)) < 1e-14
    # Eq. 14: subtracting the mean flow empties shell 0 and nothing else
    mean2 = O.from_dense(np.full((N, N), 0.25))
    E2 = O.tke_spectrum(u1, u2, None, mean2)
    want[0] = 0.0
    assert np.max(np.abs(E2 - want)) < 1e-14
    assert np.max(np.abs(O.tke_spectrum(u1, u2, u1, u2))) < 1e-28
    # Parseval on a generic field: sum_k E(k) = 1/2 mean(u1^2 + u2^2)
    F, G = smooth_field(n, 31), smooth_field(n, 32)
    E = O.tke_spectrum(O.from_dense(F), O.from_dense(G))
    assert abs(E.sum() - 0.5 * np.mean(F * F + G * G)) < 1e-13 * E.sum()
    # brute force on an 8 x 8 grid: the DFT written as plain loops (no FFT), integer shells by rounding
    n = 3
    N = 8
    F, G = rand_field(n, 41), rand_field(n, 42)
    got = O.tke_spectrum(O.from_dense(F), O.from_dense(G))
    bf = np.zeros(len(got))
    for k1 in range(-N // 2, N // 2):
        for k2 in range(-N // 2, N // 2):
            c1 = c2 = 0.0 + 0.0j
            for x in range(N):
                for y in range(N):
                    ph = np.exp(-2j * np.pi * (k1 * x + k2 * y) / N)
                    c1 += F[x, y] * ph
                    c2 += G[x, y] * ph
            e = 0.5 * (abs(c1 / N**2) ** 2 + abs(c2 / N**2) ** 2)
            bf[int(np.floor(np.hypot(k1, k2) + 0.5))] += e
    assert np.max(np.abs(got - bf)) < 1e-13 * bf.max()
