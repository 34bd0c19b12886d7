"""Pins for the TRUNCATING branch of oracle O7 (zip-up, reading 8) and for the eps rank rule (reading 6).

The zip-up with a working bond chi_w that really truncates is algorithm-defined, but every one of its steps has a
plain mathematical meaning that is checked here against something other than the oracle itself:

  per site l (info["zip"][l] = T, Q, R'):
   (a) Q^T Q = I                                  -- Q is an isometry (PAPER.md:498-518 Eq. B15-B19, left-canonical form)
   (b) R' = Q^T T                                 -- the carry is the projection of T (so "S V^T" must carry the S)
   (c) ||T - Q R'||_F = sqrt(sum_{i > keep} sigma_i(T)^2), sigma from an independent svdvals(T)
                                                  -- Eckart-Young: exactly the keep = min(chi_w, rank dims) largest
                                                     ("compressed down to chi")
   (d) T_l = (Phi_{<l}^T (x) I_4) X_l             -- X_l = left part of the EXACT product built from the explicit
                                                     hadamard() cores (oracle O4, pinned by dense brute force),
                                                     Phi_{<l} = contracted Q_1 .. Q_{l-1}
   (e) a planted spectrum with a gap at chi_w: the kept subspace and the carry are the known ones; keep +- 1 fails.
  and the state handed to the R->L sweep is the dense product projected on span(Phi_{<n}).

  rank rule: hand-computed tails where r, r - 1 and the 1/sqrt(n-1) split are each decisive (Eq. 16).

Each assertion was checked to FAIL under the mutations keep +- 1, R' = V^T (S dropped), delta without sqrt(n-1),
r + 1 (see tests/golden/README.md, "mutation log").
"""
import math

import numpy as np
import pytest

from oracle import qtt_oracle as O
import qtt_inputs as I


def smooth_field(n, seed):
    N = 1 << n
    rng = np.random.default_rng(seed)
    X, Y = I.grid(n)
    F = np.zeros((N, N))
    for kx in range(-3, 4):
        for ky in range(-3, 4):
            a, p = rng.standard_normal(), rng.uniform(0, 2 * np.pi)
            F += a / (1 + kx * kx + ky * ky) * np.cos(2 * np.pi * (kx * X + ky * Y) + p)
    return F + np.tanh((Y - 0.5) / 0.1)


def exact_left_parts(C):
    """X_l for l = 1..n: the first l cores of an MPS contracted to a (4^l) x r_l matrix."""
    out = []
    X = C[0].reshape(4, -1)
    out.append(X)
    for c in C[1:]:
        r0, d, r1 = c.shape
        X = (X @ c.reshape(r0, d * r1)).reshape(-1, r1)
        out.append(X)
    return out


@pytest.mark.parametrize("n,ca,cb,chi,cw", [(5, 6, 6, 4, 4), (5, 6, 6, 4, 8), (6, 6, 5, 5, 5), (6, 6, 6, 6, 12),
                                            (6, 8, 8, 4, 7)])
def test_zipup_truncating_branch_per_site_invariants(n, ca, cb, chi, cw):
    A = O.from_dense(smooth_field(n, 3), chi_max=ca)
    B = O.from_dense(smooth_field(n, 4), chi_max=cb)
    info = {}
    got = O.round_product(A, B, chi_max=chi, chi_work=cw, info=info)
    zl = info["zip"]
    assert len(zl) == n - 1
    X = exact_left_parts(O.hadamard(A, B))          # (d): exact product, oracle O4 (pinned against dense brute force)
    Phi = np.ones((1, 1))                            # (4^{l-1}) x r_{l-1}
    truncating_sites = 0
    for l, z in enumerate(zl):
        T, Q, R = z["T"], z["Q"], z["R"]
        m, k = T.shape
        r_prev = Phi.shape[1]
        assert m == 4 * r_prev and k == X[l].shape[1]
        # (d) T_l == (Phi^T (x) I_4) X_l
        Xl = X[l].reshape(Phi.shape[0], 4, k)
        Tl = np.einsum("si,swk->iwk", Phi, Xl).reshape(m, k)
        scale = max(np.linalg.norm(Tl), 1e-300)
        assert np.linalg.norm(T - Tl) <= 1e-12 * scale, (l, "T is not the projected exact product")
        # (a) isometry
        keep = Q.shape[1]
        assert np.linalg.norm(Q.T @ Q - np.eye(keep)) <= 1e-12
        # (b) carry = projection
        assert np.linalg.norm(R - Q.T @ T) <= 1e-12 * scale, (l, "R' != Q^T T")
        # (c) Eckart-Young with an independent svdvals
        s = np.linalg.svd(T, compute_uv=False)
        want_keep = min(m, k, cw)
        assert keep == want_keep, (l, keep, want_keep)
        tail = math.sqrt(float(np.sum(s[keep:] ** 2)))
        err = np.linalg.norm(T - Q @ R)
        assert abs(err - tail) <= 1e-11 * scale, (l, err, tail)
        if z["branch"] == "svd" and keep < min(m, k):
            # the case is decisive only if the neighbours of the cut are well above rounding
            if s[keep] > 1e-6 * s[0] and s[keep - 1] > 1e-6 * s[0]:
                truncating_sites += 1
                # keep - 1 or keep + 1 singular triplets would give a different error
                assert abs(math.sqrt(float(np.sum(s[keep - 1:] ** 2))) - err) > 1e-7 * scale
                assert abs(math.sqrt(float(np.sum(s[keep + 1:] ** 2))) - err) > 1e-7 * scale
        # next left basis: Phi'[(s,w), j] = sum_i Phi[s,i] Q[(i,w), j]
        Phi = np.einsum("si,iwj->swj", Phi, Q.reshape(r_prev, 4, keep)).reshape(-1, keep)
    if cw < ca * cb:
        assert truncating_sites >= 1, "the case never reached the truncating SVD branch decisively"
    # the state handed to the R->L sweep is the dense product projected on span(Phi_{<n}) over the first n-1 sites
    W = O.encode(O.to_dense(A) * O.to_dense(B)).reshape(4 ** (n - 1), 4)
    Z = O.to_tensor(info["zip_cores"]).reshape(4 ** (n - 1), 4)
    assert np.linalg.norm(Phi.T @ Phi - np.eye(Phi.shape[1])) <= 1e-11
    assert np.linalg.norm(Z - Phi @ (Phi.T @ W)) <= 1e-11 * np.linalg.norm(W)
    # and the R->L sweep is the pinned step (ii) of O6: the final state == round_mps of that state
    want = O.round_mps(info["zip_cores"], chi_max=chi)
    assert np.linalg.norm(O.to_dense(got) - O.to_dense(want)) <= 1e-11 * np.linalg.norm(W)


def _planted(sig, seed=0):
    """3-site operands whose zip-up matrix T_2 is EXACTLY M = U diag(sig) V^T (16 x 8): A_1 = identity (1,4,4),
    A_2 = M as (4,4,8), A_3 random (8,4,1); B = the all-ones field (bond 1), so A (.) B = A."""
    rng = np.random.default_rng(seed)
    U, _ = np.linalg.qr(rng.standard_normal((16, 8)))
    V, _ = np.linalg.qr(rng.standard_normal((8, 8)))
    M = (U * sig) @ V.T
    A = [np.eye(4).reshape(1, 4, 4), M.reshape(4, 4, 8), rng.standard_normal((8, 4, 1))]
    B = [np.ones((1, 4, 1)) for _ in range(3)]
    return A, B, U, V, M


def test_zipup_planted_gap_keeps_exactly_chi_work_triplets():
    sig = np.array([8.0, 4.0, 2.0, 1.0, 1e-3, 5e-4, 2e-4, 1e-4])
    A, B, U, V, M = _planted(sig)
    cw = 4
    info = {}
    O.round_product(A, B, chi_max=8, chi_work=cw, info=info)
    z1, z2 = info["zip"]
    assert z1["branch"] == "identity" and np.array_equal(z1["R"], z1["T"])
    assert z2["branch"] == "svd"
    T, Q, R = z2["T"], z2["Q"], z2["R"]
    assert np.linalg.norm(T - M) <= 1e-14 * np.linalg.norm(M)
    assert Q.shape == (16, cw) and R.shape == (cw, 8)       # keep == chi_w: not chi_w - 1, not chi_w + 1
    # the kept subspace is span(U[:, :4]) (gap 1 : 1e-3, so it is well conditioned) ...
    P_want = U[:, :cw] @ U[:, :cw].T
    assert np.linalg.norm(Q @ Q.T - P_want) <= 1e-12
    # ... and the carry holds S V^T, not V^T:  R'^T R' = V4 S4^2 V4^T
    assert np.linalg.norm(R.T @ R - (V[:, :cw] * sig[:cw] ** 2) @ V[:, :cw].T) <= 1e-12 * sig[0] ** 2
    assert np.linalg.norm(Q @ R - (U[:, :cw] * sig[:cw]) @ V[:, :cw].T) <= 1e-13 * sig[0]
    # discarded weight = the planted tail
    assert abs(np.linalg.norm(T - Q @ R) - math.sqrt(np.sum(sig[cw:] ** 2))) <= 1e-13 * sig[0]
    # a larger working bond keeps more (the result is NOT independent of chi_w here)
    info6 = {}
    O.round_product(A, B, chi_max=8, chi_work=6, info=info6)
    assert info6["zip"][1]["Q"].shape == (16, 6)


def test_zipup_planted_full_result_equals_truncated_dense():
    """End to end on the planted case: the zip-up result with chi_w = chi_max = 4 is the dense tensor whose 16 x 32
    unfolding is U4 S4 V4^T A_3 (the working truncation is the only truncation: rank 4 passes the R->L sweep)."""
    sig = np.array([8.0, 4.0, 2.0, 1.0, 1e-3, 5e-4, 2e-4, 1e-4])
    A, B, U, V, M = _planted(sig, seed=1)
    got = O.round_product(A, B, chi_max=4, chi_work=4)
    M4 = (U[:, :4] * sig[:4]) @ V[:, :4].T
    want = (M4 @ A[2].reshape(8, 4)).reshape(4, 4, 4)
    assert O.bonds(got) == [1, 4, 4, 1]
    assert np.linalg.norm(O.to_tensor(got) - want) <= 1e-13 * np.linalg.norm(want)


# ------------------------------------------------------------------------------------------ rank rule (reading 6)
def test_rank_rule_hand_computed_tails():
    """s = (4, 3, 2, 1, 1/2): tail(r) = sqrt(sum_{i>r} s_i^2) = 5.5, 3.775.., 2.291.., 1.118.., 0.5, 0 for r = 0..5."""
    s = np.array([4.0, 3.0, 2.0, 1.0, 0.5])
    t3 = math.sqrt(1.0 + 0.25)
    big = 10**6
    assert O._rank_rule(s, big, 1.2) == 3            # tail(3) = 1.118 <= 1.2 < tail(2) = 2.29
    assert O._rank_rule(s, big, t3) == 3             # equality counts as "<=" (Eq. 16: error <= eps)
    assert O._rank_rule(s, big, t3 * (1 - 1e-12)) == 4   # just below: one more value is needed (r - 1 is not enough)
    assert O._rank_rule(s, big, 0.5) == 4
    assert O._rank_rule(s, big, 0.49) == 5
    assert O._rank_rule(s, big, 5.5) == 1            # everything may go, but never below rank 1
    assert O._rank_rule(s, big, 2.3) == 2
    assert O._rank_rule(s, 2, 0.49) == 2             # chi_max clamps after the tolerance
    assert O._rank_rule(s, big, None) == 5 and O._rank_rule(s, 3, None) == 3   # eps = 0: pure cap


def test_rank_rule_is_minimal_brute_force():
    rng = np.random.default_rng(0)
    for _ in range(200):
        m = int(rng.integers(1, 9))
        s = np.sort(np.abs(rng.standard_normal(m)) * 10.0 ** rng.uniform(-3, 0, m))[::-1]
        delta = float(10.0 ** rng.uniform(-3.5, 0.5))
        r = O._rank_rule(s, 10**6, delta)
        tails = [math.sqrt(float(np.sum(s[k:] ** 2))) for k in range(m + 1)]
        ok = [k for k in range(m + 1) if tails[k] <= delta]
        assert r == max(1, min(ok))


def _planted_bond_mps(sig):
    """3-site MPS (bonds 1,4,4,1) whose LAST bond has exactly the Schmidt values sig (4 of them):
    U[(w1,w2), w3] = sum_k sig_k a_k[(w1,w2)] b_k[w3], a_k orthonormal in R^16, b_k orthonormal in R^4."""
    rng = np.random.default_rng(7)
    a, _ = np.linalg.qr(rng.standard_normal((16, 4)))
    b, _ = np.linalg.qr(rng.standard_normal((4, 4)))
    M = (a * sig) @ b.T                                  # 16 x 4
    return [np.eye(4).reshape(1, 4, 4), M.reshape(4, 4, 4), np.eye(4).reshape(4, 4, 1)], M


def test_eps_is_split_over_bonds_by_sqrt_n_minus_1():
    """sigma = (1, .1, .01, .001) at the last bond of a 3-site MPS (n - 1 = 2 bonds).  tails: r=3: 1e-3, r=2: 1.005e-2.
    eps ||A|| = 0.012: with delta = eps ||A|| / sqrt(2) = 8.49e-3 the rule keeps 3; WITHOUT the split (delta = 0.012)
    it would keep 2.  (Eq. 16 defines eps as the TOTAL relative error; reading 6 splits it evenly.)"""
    sig = np.array([1.0, 0.1, 0.01, 0.001])
    cores, M = _planted_bond_mps(sig)
    nrm = math.sqrt(float(np.sum(sig**2)))
    eps = 0.012 / nrm
    info = {}
    Rr = O.round_mps(cores, eps=eps, info=info)
    assert np.allclose(info["singular_values"][2], sig, rtol=1e-12, atol=0)
    assert O.bonds(Rr)[2] == 3
    assert abs(info["discarded"][2] - 1e-3) < 1e-15
    # total error stays below eps although each bond used its full share
    err = np.linalg.norm(O.to_tensor(Rr) - O.to_tensor(cores)) / nrm
    assert err <= eps
    # the same spectrum through from_dense (TT-SVD uses the same rule)
    F = O.decode(O.to_tensor(cores))
    assert O.bonds(O.from_dense(F, eps=eps))[2] == 3
    # decisive in the other direction too: eps ||A|| = 0.0145 -> delta = 1.025e-2 >= tail(2) = 1.005e-2 -> keep 2
    Rr2 = O.round_mps(cores, eps=0.0145 / nrm)
    assert O.bonds(Rr2)[2] == 2


def test_eps_rule_keeps_no_more_than_needed_on_a_field():
    """Minimality on a real field: at every bond the kept rank r satisfies tail(r) <= delta < tail(r - 1), with the
    tails recomputed from the singular values the sweep reports (independent arithmetic: plain sums here)."""
    n = 5
    A = O.apply_mpo(O.mpo_laplacian(n, 1 / 32), O.from_dense(I.config1_field()))
    for eps in (1e-1, 1e-2, 1e-4):
        info = {}
        Rr = O.round_mps(A, eps=eps, info=info)
        delta = eps * info["norm"] / math.sqrt(n - 1)
        for k in range(1, n):
            s = info["singular_values"][k]
            r = O.bonds(Rr)[k]
            assert math.sqrt(float(np.sum(s[r:] ** 2))) <= delta
            if r > 1:
                assert math.sqrt(float(np.sum(s[r - 1:] ** 2))) > delta
