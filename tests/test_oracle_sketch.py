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
    Om = O.sketch_signs(5, 2, 400, keep)
    Q, R = O.sketch_factor(T, Om)
    assert Q.shape == (96, keep) and R.shape == (keep, 400)
    assert np.linalg.norm(Q.T @ Q - np.eye(keep)) < 1e-13
    assert np.linalg.norm(R - Q.T @ T) == 0.0
    # Q R' is the orthogonal projection of T on range(T S): T - Q R' is orthogonal to Q, and range(Q) contains T S
    assert np.linalg.norm(Q.T @ (T - Q @ R)) < 1e-13 * np.linalg.norm(T)
    Y = T @ Om
    assert np.linalg.norm(Y - Q @ (Q.T @ Y)) < 1e-12 * np.linalg.norm(Y)
    # exact when rank(T) <= keep
    L = rng.standard_normal((96, 20)) @ rng.standard_normal((20, 400))
    Ql, Rl = O.sketch_factor(L, Om)
    assert np.linalg.norm(L - Ql @ Rl) < 1e-12 * np.linalg.norm(L)
    # ... and then only rank(T) columns of Q are non-zero (orthonormal), the rest exact zeros: the bond keeps its size
    nz = np.linalg.norm(Ql, axis=0) > 0
    assert nz.sum() == 20 and np.all(nz[:20]) and np.linalg.norm(Ql[:, :20].T @ Ql[:, :20] - np.eye(20)) < 1e-13
    # coinciding probes (two equal columns of S) lose one direction, nothing else
    Om2 = Om.copy()
    Om2[:, 5] = Om2[:, 4]
    Q2, R2 = O.sketch_factor(T, Om2)
    assert (np.linalg.norm(Q2, axis=0) > 0).sum() == keep - 1
    assert np.linalg.norm(Q2.T @ (T - Q2 @ R2)) < 1e-13 * np.linalg.norm(T)
    # randomised range finder (Halko-Martinsson-Tropp, Thm 10.5 in expectation): with keep = k + p probes the error is about
    # sqrt(1 + k / (p - 1)) times the optimal rank-k tail; for k = p = keep / 2 that is ~sqrt(2).  Checked with a factor 2
    # on several seeds against an independent SVD -- and it can never beat the optimal rank-keep error.
    s = np.linalg.svd(T, compute_uv=False)
    tail = lambda r: np.sqrt(np.sum(s[r:] ** 2))
    for seed in range(6):
        Qs, Rs = O.sketch_factor(T, O.sketch_signs(seed, 0, 400, keep))
        err = np.linalg.norm(T - Qs @ Rs)
        assert tail(keep) * (1 - 1e-12) <= err <= 2.0 * tail(keep // 2)


def random_gauge(cores, rng):
    """The same MPS in another gauge: core_k <- G_{k-1}^T core_k G_k with random ORTHOGONAL G (two right-canonical forms of
    one state -- what two implementations of the roundings hand to the product -- differ by exactly that; the truncated SVDs
    of the zip-up, deterministic or not, are only defined up to such gauges)."""
    out = [c.copy() for c in cores]
    for k in range(len(cores) - 1):
        r = cores[k].shape[2]
        G = np.linalg.qr(rng.standard_normal((r, r)))[0]
        out[k] = np.einsum("awb,bc->awc", out[k], G)
        out[k + 1] = np.einsum("ba,bwc->awc", G, out[k + 1])
    return out


def test_probes_are_the_dense_contraction_and_the_result_does_not_depend_on_the_gauge():
    n, P, seed = 4, 6, 9
    rng = np.random.default_rng(2)
    A = O.from_dense(rng.standard_normal((16, 16)), 5)
    B = O.from_dense(rng.standard_normal((16, 16)), 5)
    S = O.sketch_probes(A, B, P, seed)
    assert S[n].shape == (1, 1, P) and np.all(S[n] == 1.0)
    # the cores of the probe train are the generator's signs, row w P + u, column t, over sqrt(P)
    for k in (0, 3):
        G = O.sketch_mixers(seed, k, P)
        assert G.shape == (4, P, P)
        for w, uu, t in ((0, 0, 0), (3, 5, 5), (2, 1, 4), (1, 4, 0)):
            assert G[w, uu, t] == sign_bigint(seed, k, w * P + uu, t) / np.sqrt(P)
    # brute force: the probes are the dense tensor Omega[w_l .. w_{n-1}; t] of that train (closed by ones at the right end),
    # contracted with the dense right part of the Hadamard product MPS
    H = O.hadamard(A, B)
    for l in (1, 2, 3):
        right = H[l]
        for k in range(l + 1, n):
            right = np.tensordot(right, H[k], axes=([right.ndim - 1], [0]))
        right = right.reshape(right.shape[0], -1)  # (bond, (w_l, ..., w_{n-1}))
        Om = None
        for k in range(n - 1, l - 1, -1):
            G = np.array([[[sign_bigint(seed, k, w * P + uu, t) for t in range(P)] for uu in range(P)] for w in range(4)]) / np.sqrt(P)
            if Om is None:
                Om = G.sum(axis=1)  # (w_{n-1}, t)
            else:
                Om = np.tensordot(G, Om, axes=([1], [Om.ndim - 1]))  # (w_k, t, w_{k+1}, ...) -> move t last
                Om = np.moveaxis(Om, 1, -1)
        v = right @ Om.reshape(-1, P)
        assert np.allclose(v, S[l].reshape(-1, P), rtol=1e-12, atol=1e-12 * np.abs(v).max())
    # a bond-1 train (one rank-one sign tensor per probe) would also be gauge invariant, but its range finder fails too often;
    # this one stays within the optimal rank-P/2 tail of the TRUE unfolding (T times the dense right part) on every seed tried
    n6, cw = 7, 8
    Fa, Fb = fields(n6, 3)
    A6, B6 = O.from_dense(Fa, 16), O.from_dense(Fb, 16)
    H6 = O.hadamard(A6, B6)
    for sd in range(1, 7):
        info = {}
        O.round_product(A6, B6, cw // 2, chi_work=cw, sketch_seed=sd, info=info)
        took = exact = 0
        for l, z in enumerate(info["zip"]):
            if z["branch"] != "sketch":
                continue
            took += 1
            E = np.ones((1, 1))
            for k in range(n6 - 1, l, -1):
                r0, d, r1 = H6[k].shape
                E = (H6[k].reshape(r0 * d, r1) @ E).reshape(r0, -1)
            M = z["T"] @ E
            s = np.linalg.svd(M, compute_uv=False)
            err = np.linalg.norm(M - z["Q"] @ (z["Q"].T @ M))
            assert err <= 2.0 * np.sqrt(np.sum(s[cw // 2:] ** 2)) + 1e-11 * s[0]
            if 4 ** (n6 - 1 - l) <= cw:  # few configurations left: the probes span the whole range, nothing is lost
                exact += 1
                assert err <= 1e-11 * s[0] and (np.linalg.norm(z["Q"], axis=0) > 0).sum() <= 4 ** (n6 - 1 - l)
        assert took >= 4 and exact >= 1
    # gauge invariance of the whole sketched rounding (what a random matrix on the bond indices would NOT have)
    n, chi = 6, 8
    Fa, Fb = fields(n, 3)
    A, B = O.from_dense(Fa, 16), O.from_dense(Fb, 16)
    ref = O.to_dense(O.round_product(A, B, chi, chi_work=2 * chi, sketch_seed=11))
    A2, B2 = random_gauge(A, rng), random_gauge(B, rng)
    assert np.linalg.norm(O.to_dense(A2) - O.to_dense(A)) < 1e-11 * np.linalg.norm(O.to_dense(A))
    got = O.to_dense(O.round_product(A2, B2, chi, chi_work=2 * chi, sketch_seed=11))
    assert np.linalg.norm(got - ref) < 1e-9 * np.linalg.norm(ref)
    # ... and it does depend on the seed
    other = O.to_dense(O.round_product(A, B, chi, chi_work=2 * chi, sketch_seed=12))
    assert np.linalg.norm(other - ref) > 1e-6 * np.linalg.norm(ref)


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
    assert "sketch" in bs and all(x == y or (x == "svd" and y == "sketch") for x, y in zip(bd, bs))
    for l, (x, y) in enumerate(zip(bd, bs)):  # the sketch is taken exactly where sketch_applies says
        m, k = info_d["zip"][l]["T"].shape
        assert (y == "sketch") == (x == "svd" and O.sketch_applies(n, l, m, k, 2 * chi))
    assert O.bonds(ske) == O.bonds(det)
    for z in info_s["zip"]:
        if z["branch"] == "sketch":
            assert z["Q"].shape[1] == 2 * chi
            nzc = np.linalg.norm(z["Q"], axis=0) > 0
            Qn = z["Q"][:, nzc]
            assert np.linalg.norm(Qn.T @ Qn - np.eye(Qn.shape[1])) < 1e-12
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
    n, chi, Re, dt = 7, 6, 200.0, 1e-3
    dx = 1.0 / (1 << n)
    Fa, Fb = fields(n, 5)
    u = [O.from_dense(Fa, chi), O.from_dense(0.5 * Fb, chi)]
    ops = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    info = {}
    O.round_product(u[0], u[1], chi, sketch_seed=3, info=info)
    assert "sketch" in [z["branch"] for z in info["zip"]]  # these sizes do take the sketch
    det = O.rk4_step(u, *ops, Re, dt, chi)
    ske = O.rk4_step(u, *ops, Re, dt, chi, sketch_seed=3)
    big = O.rk4_step(u, *ops, Re, dt, 4 * chi)  # nearly untruncated step as the yardstick
    for i in range(2):
        ref = O.to_dense(big[i])
        e_det = np.linalg.norm(O.to_dense(det[i]) - ref) / np.linalg.norm(ref)
        e_ske = np.linalg.norm(O.to_dense(ske[i]) - ref) / np.linalg.norm(ref)
        assert e_ske <= 3.0 * e_det + 1e-12
