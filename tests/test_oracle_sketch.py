"""Pins for the oracle's sketched zip-up ("a cheaper product compression (randomised ...)",
PAPER.md:318; reading 25): the counter-based sign generator, the range-finder step, and the product rounding
built on it.  What fixes them other than themselves: an independent big-integer restatement of the generator, the
algebra of an orthogonal projector, exactness on matrices of rank <= the sketch size, the randomised-range-finder error
bound against an independent SVD, and the dense elementwise product."""
import numpy as np
import pytest

from oracle import qtt_oracle as O
import qtt_inputs as I

M64 = (1 << 64) - 1


def sign_bigint(seed, site, c, t):
    z = (seed * 0x9E3779B97F4A7C15 + site * 0xD1B54A32D192ED03 + (c << 20) + t) & M64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & M64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & M64
    z ^= z >> 31
    return -1.0 if (z >> 63) else 1.0


def test_sign_generator_matches_a_bigint_restatement_and_is_balanced():
    Om = O.sketch_signs(7, 3, 300, 40)
    assert Om.shape == (300, 40) and set(np.unique(Om)) == {-1.0, 1.0}
    rng = np.random.default_rng(0)
    for _ in range(200):
        c, t = int(rng.integers(300)), int(rng.integers(40))
        assert Om[c, t] == sign_bigint(7, 3, c, t)
    big = O.sketch_signs(123456789, 9, 4096, 128)
    for c, t in ((4095, 127), (0, 0), (2048, 1), (77, 99)):
        assert big[c, t] == sign_bigint(123456789, 9, c, t)
    # balanced, and different seeds / sites give different matrices
    assert abs(big.mean()) < 4.0 / np.sqrt(big.size)
    assert np.any(O.sketch_signs(8, 3, 300, 40) != Om) and np.any(O.sketch_signs(7, 4, 300, 40) != Om)
    # probe columns are nearly orthogonal (what a range finder needs)
    G = big.T @ big / big.shape[0]
    assert np.max(np.abs(G - np.eye(128))) < 6.0 / np.sqrt(big.shape[0])


def graded(rng, m, k, decades):
    r = min(m, k)
    U, _ = np.linalg.qr(rng.standard_normal((m, r)))
    V, _ = np.linalg.qr(rng.standard_normal((k, r)))
    return (U * np.logspace(0, -decades, r)) @ V.T


def test_sketch_factor_is_a_projection_exact_on_low_rank_and_within_the_range_finder_bound():
    rng = np.random.default_rng(1)
    T = graded(rng, 96, 400, 8)
    keep = 32
    Q, R = O.sketch_factor(T, keep, seed=5, site=2)
    assert Q.shape == (96, keep) and R.shape == (keep, 400)
    assert np.linalg.norm(Q.T @ Q - np.eye(keep)) < 1e-13
    assert np.linalg.norm(R - Q.T @ T) == 0.0
    # Q R' is the orthogonal projection of T on range(T Omega): T - Q R' is orthogonal to Q, and range(Q) contains T Omega
    assert np.linalg.norm(Q.T @ (T - Q @ R)) < 1e-13 * np.linalg.norm(T)
    Y = T @ O.sketch_signs(5, 2, 400, keep)
    assert np.linalg.norm(Y - Q @ (Q.T @ Y)) < 1e-12 * np.linalg.norm(Y)
    # exact when rank(T) <= keep
    L = rng.standard_normal((96, 20)) @ rng.standard_normal((20, 400))
    Ql, Rl = O.sketch_factor(L, keep, seed=5, site=2)
    assert np.linalg.norm(L - Ql @ Rl) < 1e-12 * np.linalg.norm(L)
    # randomised range finder (Halko-Martinsson-Tropp, Thm 10.5 in expectation): with keep = k + p probes the error is about
    # sqrt(1 + k / (p - 1)) times the optimal rank-k tail; for k = p = keep / 2 that is ~sqrt(2).  Checked with a factor 2
    # on several seeds against an independent SVD -- and it can never beat the optimal rank-keep error.
    s = np.linalg.svd(T, compute_uv=False)
    tail = lambda r: np.sqrt(np.sum(s[r:] ** 2))
    for seed in range(6):
        Qs, Rs = O.sketch_factor(T, keep, seed=seed, site=0)
        err = np.linalg.norm(T - Qs @ Rs)
        assert tail(keep) * (1 - 1e-12) <= err <= 2.0 * tail(keep // 2)


def fields(n, seed):
    X, Y = I.grid(n)
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(2):
        F = np.tanh((Y - 0.5) / 0.08) * (1 + 0.2 * np.cos(2 * np.pi * X))
        for kx in range(-3, 4):
            for ky in range(-3, 4):
                F = F + rng.standard_normal() / (1 + kx * kx + ky * ky) * np.cos(2 * np.pi * (kx * X + ky * Y) + rng.uniform(0, 6.28))
        out.append(F)
    return out


def test_sketched_product_rounding_against_the_dense_product_and_the_deterministic_zip_up():
    n, chi = 6, 8
    Fa, Fb = fields(n, 3)
    A, B = O.from_dense(Fa, 16), O.from_dense(Fb, 16)
    exact = Fa_Fb = O.to_dense(A) * O.to_dense(B)
    info_d, info_s = {}, {}
    det = O.round_product(A, B, chi, chi_work=2 * chi, info=info_d)
    ske = O.round_product(A, B, chi, chi_work=2 * chi, info=info_s, sketch_seed=11)
    # the sketch replaces exactly the truncating SVD steps, nothing else
    bd = [z["branch"] for z in info_d["zip"]]
    bs = [z["branch"] for z in info_s["zip"]]
    assert "svd" in bd and [b if b != "svd" else "sketch" for b in bd] == bs
    assert O.bonds(ske) == O.bonds(det)
    for z in info_s["zip"]:
        if z["branch"] == "sketch":
            assert z["Q"].shape[1] == 2 * chi
            assert np.linalg.norm(z["Q"].T @ z["Q"] - np.eye(2 * chi)) < 1e-12
            assert np.linalg.norm(z["R"] - z["Q"].T @ z["T"]) < 1e-12 * np.linalg.norm(z["T"])
    e_det = np.linalg.norm(O.to_dense(det) - exact) / np.linalg.norm(exact)
    e_ske = np.linalg.norm(O.to_dense(ske) - exact) / np.linalg.norm(exact)
    best = np.linalg.norm(O.to_dense(O.round_mps(O.hadamard(A, B), chi)) - exact) / np.linalg.norm(exact)
    assert best * (1 - 1e-9) <= e_det and e_ske <= 3.0 * max(e_det, best)
    # a working bond that never truncates: both modes are the exact rounding of the exact product
    full = O.round_product(A, B, chi, chi_work=10**6, sketch_seed=11)
    ref = O.round_mps(O.hadamard(A, B), chi)
    assert np.linalg.norm(O.to_dense(full) - O.to_dense(ref)) < 1e-11 * np.linalg.norm(exact)


def test_rk4_step_with_the_sketched_products_stays_within_the_truncation_error():
    n, chi, Re, dt = 6, 10, 200.0, 1e-3
    dx = 1.0 / (1 << n)
    Fa, Fb = fields(n, 5)
    u = [O.from_dense(Fa, chi), O.from_dense(0.5 * Fb, chi)]
    ops = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    det = O.rk4_step(u, *ops, Re, dt, chi)
    ske = O.rk4_step(u, *ops, Re, dt, chi, sketch_seed=3)
    big = O.rk4_step(u, *ops, Re, dt, 4 * chi)  # nearly untruncated step as the yardstick
    for i in range(2):
        ref = O.to_dense(big[i])
        e_det = np.linalg.norm(O.to_dense(det[i]) - ref) / np.linalg.norm(ref)
        e_ske = np.linalg.norm(O.to_dense(ske[i]) - ref) / np.linalg.norm(ref)
        assert e_ske <= 3.0 * e_det + 1e-12
