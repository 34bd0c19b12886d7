"""GPU kernel-level parity (include/qtt_diag.h) against NumPy/LAPACK on seeded inputs: the grouped
DMMA GEMM, the Q-less LQ, the row-Jacobi SVD and the rank selection.  Sizes span several tiles and
ragged tails.  Everything goes through the C ABI."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_2406_17823_b200 import _lib
    lib = _lib.load()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    stream = torch.cuda.Stream()
    return lib, torch, stream


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def ptr(t):
    return C.c_void_p(t.data_ptr())


GEMM_CASES = [
    # M, N, K, transA, transB, nbatch
    (1, 1, 1, 0, 0, 1), (4, 12, 4, 0, 0, 1), (33, 17, 5, 0, 0, 3), (64, 64, 64, 0, 0, 1),
    (130, 70, 33, 0, 1, 2), (257, 129, 65, 1, 0, 1), (100, 260, 48, 1, 1, 2), (512, 256, 64, 0, 0, 4),
    (768, 192, 192, 0, 0, 1), (1024, 512, 128, 0, 1, 1), (31, 1000, 7, 1, 0, 1), (2048, 16, 256, 0, 0, 1),
]


@pytest.mark.parametrize("M,N,K,ta,tb,nb", GEMM_CASES)
def test_gemm_matches_numpy(env, M, N, K, ta, tb, nb):
    lib, torch, stream = env
    rng = np.random.default_rng(M * 131 + N * 17 + K)
    A = rng.standard_normal((nb, K, M) if ta else (nb, M, K))
    B = rng.standard_normal((nb, N, K) if tb else (nb, K, N))
    C0 = rng.standard_normal((nb, M, N))
    alpha, beta = 0.75, -0.5
    opA = A.transpose(0, 2, 1) if ta else A
    opB = B.transpose(0, 2, 1) if tb else B
    want = alpha * np.matmul(opA, opB) + beta * C0
    dA, dB, dC = dev(torch, A), dev(torch, B), dev(torch, C0)
    torch.cuda.synchronize()
    st = lib.qtt_diag_gemm(C.c_void_p(stream.cuda_stream), ptr(dA), ptr(dB), ptr(dC), M, N, K, ta, tb,
                           A.shape[2], B.shape[2], N, alpha, beta, nb, A.shape[1] * A.shape[2],
                           B.shape[1] * B.shape[2], M * N)
    assert st == 0
    stream.synchronize()
    got = dC.cpu().numpy()
    scale = np.abs(opA).sum(axis=2).max() * np.abs(opB).max() + np.abs(C0).max()
    assert np.max(np.abs(got - want)) <= 1e-13 * scale


def test_gemm_odd_leading_dimensions(env):
    """Odd strides / unaligned bases take the 8-byte copy path."""
    lib, torch, stream = env
    rng = np.random.default_rng(5)
    M, N, K, lda, ldb, ldc = 45, 37, 29, 31, 41, 39
    A = rng.standard_normal((M, lda))
    B = rng.standard_normal((K, ldb))
    Cm = np.zeros((M, ldc))
    dA, dB, dC = dev(torch, A), dev(torch, B), dev(torch, Cm)
    torch.cuda.synchronize()
    st = lib.qtt_diag_gemm(C.c_void_p(stream.cuda_stream), C.c_void_p(dA.data_ptr() + 8), ptr(dB),
                           C.c_void_p(dC.data_ptr() + 8), M, N, K, 0, 0, lda, ldb, ldc, 1.0, 0.0, 1, 0, 0, 0)
    assert st == 0
    stream.synchronize()
    got = dC.cpu().numpy().reshape(-1)[1:1 + (M - 1) * ldc + N]
    A1 = A.reshape(-1)[1:]
    want = np.array([[A1[i * lda:i * lda + K] @ B[:, j] for j in range(N)] for i in range(M)])
    got2 = np.array([[got[i * ldc + j] for j in range(N)] for i in range(M)])
    assert np.max(np.abs(got2 - want)) < 1e-12


LQ_CASES = [(4, 4, 1), (12, 16, 2), (16, 48, 3), (48, 64, 1), (192, 768, 2), (100, 333, 2), (320, 1280, 1),
            (64, 4096, 2), (256, 9000, 1), (512, 4096, 4), (100, 5000, 2), (40, 300, 2), (330, 4100, 2),
            (500, 8192, 3)]  # > 96 MB per batch: the two-level (64-row super-panel) blocking


@pytest.mark.parametrize("k,m,batch", LQ_CASES)
def test_lq_triangular_factor(env, k, m, batch):
    """Y = L Q: R = L^T must satisfy R^T R = Y Y^T and be upper triangular; |R| equals LAPACK's
    |R| of qr(Y^T) row by row (the factor is unique up to row signs for full-rank Y)."""
    lib, torch, stream = env
    rng = np.random.default_rng(k * 7 + m)
    Y = rng.standard_normal((batch, k, m))
    dY = dev(torch, Y)
    dR = torch.zeros((batch, k, k), dtype=torch.float64, device="cuda")
    scratch = torch.zeros(batch * 3 * 64 * m, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    st = lib.qtt_diag_lq(C.c_void_p(stream.cuda_stream), ptr(dY), batch, k, m, m, ptr(dR), ptr(scratch))
    assert st == 0
    stream.synchronize()
    R = dR.cpu().numpy()
    for b in range(batch):
        assert np.allclose(np.tril(R[b], -1), 0.0)
        G = Y[b] @ Y[b].T
        assert np.linalg.norm(R[b].T @ R[b] - G) <= 1e-12 * np.linalg.norm(G)
        Rl = np.linalg.qr(Y[b].T, mode="r")
        assert np.linalg.norm(np.abs(R[b]) - np.abs(Rl)) <= 1e-10 * np.linalg.norm(Rl)


def test_lq_rank_deficient(env):
    lib, torch, stream = env
    rng = np.random.default_rng(3)
    k, m = 48, 200
    Y = rng.standard_normal((k, 7)) @ rng.standard_normal((7, m))
    Y[10] = 0.0
    dY = dev(torch, Y)
    dR = torch.zeros((k, k), dtype=torch.float64, device="cuda")
    scratch = torch.zeros(3 * 64 * m, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_lq(C.c_void_p(stream.cuda_stream), ptr(dY), 1, k, m, m, ptr(dR), ptr(scratch)) == 0
    stream.synchronize()
    R = dR.cpu().numpy()
    G = Y @ Y.T
    assert np.all(np.isfinite(R))
    assert np.linalg.norm(R.T @ R - G) <= 1e-12 * np.linalg.norm(G)


JAC_CASES = [(2, 8, 1), (4, 4, 2), (12, 4, 1), (16, 48, 3), (48, 16, 1), (64, 256, 2), (192, 256, 2), (37, 101, 2),
             (256, 256, 1), (384, 512, 1),
             (24, 700, 2), (6, 2500, 1)]  # rows too long for bj2 and no work buffer for sbj: the column-sliced last-resort kernel


@pytest.mark.parametrize("p,q,batch", JAC_CASES)
def test_rowjacobi_gives_singular_values_and_orthogonal_rows(env, p, q, batch):
    lib, torch, stream = env
    rng = np.random.default_rng(p * 3 + q)
    # decaying spectrum so that the test sees relative accuracy on small singular values
    X = rng.standard_normal((batch, p, q)) * np.logspace(0, -6, q)[None, None, :]
    dX = dev(torch, X)
    status = torch.zeros(2, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_rowjacobi(C.c_void_p(stream.cuda_stream), ptr(dX), batch, p, q, q, ptr(status)) == 0
    stream.synchronize()
    Z = dX.cpu().numpy()
    stt = status.cpu().numpy()
    assert stt[1] == 0 and 1 <= stt[0] <= 60
    for b in range(batch):
        s = np.sort(np.linalg.norm(Z[b], axis=1))[::-1]
        want = np.linalg.svd(X[b], compute_uv=False)
        mn = min(p, q)
        assert np.max(np.abs(s[:mn] - want)) <= 1e-12 * want[0]
        G = Z[b] @ Z[b].T
        d = np.sqrt(np.maximum(np.diag(G), 1e-300))
        off = (G - np.diag(np.diag(G))) / np.outer(d, d)
        big = d > 1e-9 * d.max()
        assert np.max(np.abs(off[np.ix_(big, big)])) < 1e-13 * np.sqrt(q) * 4
        # the row space is unchanged: Z = J X with J orthogonal
        assert abs(np.linalg.norm(Z[b]) - np.linalg.norm(X[b])) <= 1e-13 * np.linalg.norm(X[b])


def test_select_rank_rule_and_normalised_rows(env):
    lib, torch, stream = env
    rng = np.random.default_rng(11)
    p, q = 20, 50
    sig = np.array([10.0 * 0.5**i for i in range(p)])
    V = np.linalg.qr(rng.standard_normal((q, p)))[0].T
    perm = rng.permutation(p)
    X = (sig[:, None] * V)[perm]
    dX = dev(torch, X)
    for chi, delta in [(8, -1.0), (30, -1.0), (30, 0.3), (4, 0.3), (30, 1e-30), (30, 1e9)]:
        r_cap = p
        out = torch.full((r_cap, q), 7.0, dtype=torch.float64, device="cuda")
        sg = torch.zeros(p + 1, dtype=torch.float64, device="cuda")
        rk = torch.zeros(1, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        assert lib.qtt_diag_select(C.c_void_p(stream.cuda_stream), ptr(dX), p, q, q, ptr(out), r_cap, ptr(sg), ptr(rk),
                                   chi, delta) == 0
        stream.synchronize()
        s = sg.cpu().numpy()[:p]
        assert np.allclose(s, sig, rtol=1e-13)
        if delta < 0:
            want = min(chi, p, q)
        else:
            tails = [np.sqrt(np.sum(sig[r:] ** 2)) for r in range(p + 1)]
            want = next(r for r in range(p + 1) if tails[r] <= delta)
            want = max(1, min(want, chi, p))
        r = int(rk.cpu().numpy()[0])
        assert r == want
        o = out.cpu().numpy()
        assert np.allclose(o[:r], V[:r], atol=1e-13)
        assert np.all(o[r:] == 0.0)


def test_fp64_probes_report_plausible_rates(env):
    lib, torch, stream = env
    for kind in (0, 1):
        t = C.c_double()
        assert lib.qtt_diag_fp64_probe(C.c_void_p(stream.cuda_stream), kind, 148 * 4, 2000, C.byref(t)) == 0
        assert 1.0 < t.value < 200.0


SVD_CASES = [
    # p, q, batch, true rank (0 = full)
    (1, 4, 1, 0), (2, 4, 2, 0), (12, 4, 3, 0), (16, 64, 2, 0), (48, 16, 1, 0), (64, 256, 2, 20), (192, 256, 3, 70),
    (320, 256, 2, 100), (100, 37, 2, 0), (256, 256, 1, 0), (512, 512, 1, 150),
]


@pytest.mark.parametrize("p,q,batch,rk", SVD_CASES)
def test_pivoted_qr_preconditioner_then_jacobi(env, p, q, batch, rk):
    """qtt_diag_svd_rows: X <- Q^T X keeps X^T X (row space, singular values), reveals the numerical rank, zeroes the
    rows below it; Jacobi on the graded rows then reproduces LAPACK's singular values in few sweeps."""
    lib, torch, stream = env
    rng = np.random.default_rng(p * 7 + q + rk)
    mn = min(p, q)
    if rk:
        X = (rng.standard_normal((batch, p, rk)) * np.logspace(0, -9, rk)[None, None, :]) @ rng.standard_normal((batch, rk, q))
    else:
        X = rng.standard_normal((batch, p, q)) * np.logspace(0, -7, q)[None, None, :]
    want = [np.linalg.svd(X[b], compute_uv=False) for b in range(batch)]
    # preconditioner only
    dX = dev(torch, X)
    rank = torch.zeros(batch, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_svd_rows(C.c_void_p(stream.cuda_stream), ptr(dX), batch, p, q, q, ptr(rank), None) == 0
    stream.synchronize()
    R = dX.cpu().numpy()
    rr = rank.cpu().numpy()
    for b in range(batch):
        nx = np.linalg.norm(X[b])
        assert 1 <= rr[b] <= mn
        if rk:
            assert rk <= rr[b] <= rk + 2  # exact rank rk plus at most a couple of noise rows above 8 eps ||X||
        assert np.all(R[b][rr[b]:] == 0.0)
        assert np.linalg.norm(R[b].T @ R[b] - X[b].T @ X[b]) <= 1e-13 * nx * nx
        # graded rows: norms of the rows decrease up to the usual pivoted-QR slack
        rn = np.linalg.norm(R[b][: rr[b]], axis=1)
        assert np.all(rn[1:] <= rn[:-1] * np.sqrt(q) * 1.0001)
    # preconditioner + Jacobi
    dX = dev(torch, X)
    status = torch.zeros(2, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_svd_rows(C.c_void_p(stream.cuda_stream), ptr(dX), batch, p, q, q, ptr(rank), ptr(status)) == 0
    stream.synchronize()
    Z = dX.cpu().numpy()
    stt = status.cpu().numpy()
    assert stt[1] == 0 and stt[0] <= 16, stt
    for b in range(batch):
        s = np.sort(np.linalg.norm(Z[b], axis=1))[::-1]
        assert np.max(np.abs(s[:mn] - want[b])) <= 1e-12 * want[b][0]
        G = Z[b] @ Z[b].T
        d = np.sqrt(np.maximum(np.diag(G), 1e-300))
        big = d > 1e-9 * d.max()
        off = (G - np.diag(np.diag(G))) / np.outer(d, d)
        assert np.max(np.abs(off[np.ix_(big, big)])) < 1e-13 * np.sqrt(q) * 4


@pytest.mark.parametrize("p,q,batch", [(40, 600, 2), (300, 700, 2), (100, 1000, 1), (1024, 1024, 2), (70, 1500, 2),
                                       (260, 2048, 1), (2048, 2048, 1)])
def test_streamed_block_jacobi(env, p, q, batch):
    """qtt_diag_rowjacobi_streamed (rows too long for the cluster-resident kernel): singular values against LAPACK,
    mutually orthogonal rows, unchanged Frobenius norm."""
    lib, torch, stream = env
    rng = np.random.default_rng(p + q)
    mn = min(p, q)
    # graded rows, as the triangular factors of the zip-up are
    X = rng.standard_normal((batch, p, q)) * np.logspace(0, -8, p)[None, :, None]
    dX = dev(torch, X)
    status = torch.zeros(2, dtype=torch.int32, device="cuda")
    work = torch.zeros(8 * batch, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_rowjacobi_streamed(C.c_void_p(stream.cuda_stream), ptr(dX), batch, p, q, q, ptr(status),
                                           ptr(work)) == 0
    stream.synchronize()
    Z = dX.cpu().numpy()
    stt = status.cpu().numpy()
    assert stt[1] == 0 and 1 <= stt[0] <= 40, stt
    for b in range(batch):
        s = np.sort(np.linalg.norm(Z[b], axis=1))[::-1]
        want = np.linalg.svd(X[b], compute_uv=False)
        assert np.max(np.abs(s[:mn] - want)) <= 1e-12 * want[0]
        G = Z[b] @ Z[b].T
        d = np.sqrt(np.maximum(np.diag(G), 1e-300))
        big = d > 1e-9 * d.max()
        off = (G - np.diag(np.diag(G))) / np.outer(d, d)
        assert np.max(np.abs(off[np.ix_(big, big)])) < 1e-13 * np.sqrt(q) * 4
        assert abs(np.linalg.norm(Z[b]) - np.linalg.norm(X[b])) <= 1e-13 * np.linalg.norm(X[b])


def test_select_sorts_more_than_2048_rows(env):
    """The rank selection beyond the former 2048-row cap (dynamic shared-memory sort keys): 3000 rows of known norms."""
    lib, torch, stream = env
    rng = np.random.default_rng(5)
    p, q, chi = 3000, 8, 5
    sig = rng.permutation(np.linspace(1.0, 4.0, p))
    V = rng.standard_normal((p, q))
    V /= np.linalg.norm(V, axis=1)[:, None]
    X = sig[:, None] * V
    dX = dev(torch, X)
    out = torch.zeros((chi, q), dtype=torch.float64, device="cuda")
    sg = torch.zeros(p + 1, dtype=torch.float64, device="cuda")
    rk = torch.zeros(1, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_select(C.c_void_p(stream.cuda_stream), ptr(dX), p, q, q, ptr(out), chi, ptr(sg), ptr(rk), chi,
                               -1.0) == 0
    stream.synchronize()
    order = np.argsort(-sig, kind="stable")
    assert np.allclose(sg.cpu().numpy()[:p], sig[order], rtol=1e-13)
    assert int(rk.cpu().numpy()[0]) == chi
    assert np.allclose(out.cpu().numpy(), V[order[:chi]], atol=1e-13)
