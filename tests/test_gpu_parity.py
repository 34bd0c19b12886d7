"""GPU parity proper: the qtt_* C ABI (through the ctypes binding) against the CPU oracle on the
same seeded host inputs.  Bar (BASELINE.json north_star): relative Frobenius error <= 1e-10 on dense
reconstructions, Schmidt spectra within 1e-9 * sigma_1; integer results (bonds, ranks) exact."""
import numpy as np
import pytest

import qtt_inputs as I
from oracle import qtt_oracle as O

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def Q():
    import paper_2406_17823_b200 as q
    return q


@pytest.fixture(scope="module")
def ctx(Q):
    c = Q.Context(device=0, workspace_bytes=2 << 30)
    yield c
    c.close()


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def gpu_dense(Q, ctx, x):
    t = Q.qtt_to_dense(ctx, x)
    ctx.synchronize()
    return t.cpu().numpy()


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


def ops(Q, ctx, n):
    dx = 1.0 / (1 << n)
    g = (Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx),
         Q.qtt_mpo_laplacian(ctx, n, dx))
    o = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    return g, o


# ---------------------------------------------------------------- boundary: encode / decode
@pytest.mark.parametrize("n", [1, 2, 3, 5, 7])
def test_from_cores_to_dense_matches_oracle(Q, ctx, n):
    cores = I.random_cores(n, 6, seed=n)
    x = Q.qtt_mps_from_cores(ctx, cores)
    assert Q.qtt_mps_bonds(x) == O.bonds(cores)
    assert rel(gpu_dense(Q, ctx, x), O.to_dense(cores)) < 1e-13


@pytest.mark.parametrize("n,chi", [(2, 100), (4, 1000), (5, 8), (6, 7), (8, 32)])
def test_from_dense_matches_oracle(Q, ctx, n, chi):
    import torch
    F = smooth_field(n, 3) + 1e-3 * np.random.default_rng(n).standard_normal((1 << n, 1 << n))
    want = O.from_dense(F, chi)
    x = Q.qtt_mps_from_dense(ctx, torch.from_numpy(F).cuda(), chi)
    assert Q.qtt_mps_bonds(x) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, x), O.to_dense(want)) < TOL


def test_from_dense_eps_rule_matches_oracle_ranks(Q, ctx):
    import torch
    F = smooth_field(6, 9)
    for eps in (1e-2, 1e-5):
        want = O.from_dense(F, 1 << 20, eps)
        x = Q.qtt_mps_from_dense(ctx, torch.from_numpy(F).cuda(), 1 << 20, eps)
        assert Q.qtt_mps_bonds(x) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, x), O.to_dense(want)) < TOL


# ---------------------------------------------------------------- operators (native builders)
@pytest.mark.parametrize("n", [2, 4, 6])
def test_native_mpo_builders_match_oracle_operators(Q, ctx, n):
    g, o = ops(Q, ctx, n)
    cores = I.random_cores(n, 5, seed=1)
    x = Q.qtt_mps_from_cores(ctx, cores)
    for Wg, Wo in zip(g, o):
        y = Q.qtt_apply_mpo(ctx, Wg, x)
        want = O.apply_mpo(Wo, cores)
        assert Q.qtt_mps_bonds(y) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, y), O.to_dense(want)) < 1e-13
        # element-wise equality of the exact expanded cores
        for k in range(n):
            assert np.allclose(Q.qtt_mps_get_core(ctx, y, k), want[k], rtol=1e-14, atol=0)


def test_mpo_create_from_host_cores(Q, ctx):
    n = 5
    dx = 1.0 / 32
    Wo = O.mpo_laplacian(n, dx)
    W = Q.qtt_mpo_create(ctx, Wo)
    cores = I.random_cores(n, 4, seed=2)
    x = Q.qtt_mps_from_cores(ctx, cores)
    y = Q.qtt_apply_mpo(ctx, W, x)
    assert rel(gpu_dense(Q, ctx, y), O.to_dense(O.apply_mpo(Wo, cores))) < 1e-13


# ---------------------------------------------------------------- exact lazy algebra
def test_hadamard_and_axpy_exact(Q, ctx):
    n = 5
    A, B, Cc = (I.random_cores(n, c, seed=s) for c, s in ((4, 1), (3, 2), (5, 3)))
    a, b, c = (Q.qtt_mps_from_cores(ctx, t) for t in (A, B, Cc))
    h = Q.qtt_hadamard(ctx, a, b)
    assert Q.qtt_mps_bonds(h) == O.bonds(O.hadamard(A, B))
    assert rel(gpu_dense(Q, ctx, h), O.to_dense(A) * O.to_dense(B)) < 1e-13
    y = Q.qtt_mps_clone(ctx, c)
    Q.qtt_axpy(ctx, -2.5, a, y)
    Q.qtt_axpy(ctx, 0.125, b, y)
    want = O.lincomb([(0.125, B), (-2.5, A), (1.0, Cc)])
    assert Q.qtt_mps_bonds(y) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, y), O.to_dense(want)) < 1e-13
    assert abs(Q.qtt_mps_dot(ctx, a, b) - O.dot(A, B)) <= 1e-12 * O.norm(A) * O.norm(B)
    assert abs(Q.qtt_mps_norm(ctx, c) - O.norm(Cc)) <= 1e-12 * O.norm(Cc)


# ---------------------------------------------------------------- rounding
@pytest.mark.parametrize("n,chi0,chi", [(4, 16, 3), (5, 12, 8), (6, 20, 6), (8, 24, 16), (8, 40, 32)])
def test_round_dense_matches_oracle(Q, ctx, n, chi0, chi):
    F = smooth_field(n, n) + 1e-2 * np.random.default_rng(n).standard_normal((1 << n, 1 << n))
    A = O.from_dense(F, chi0)
    # scramble the gauge so that the input is not already canonical
    rng = np.random.default_rng(7)
    for k in range(n - 1):
        r = A[k].shape[2]
        G = rng.standard_normal((r, r)) + 2 * np.eye(r)
        A[k] = np.einsum("awb,bc->awc", A[k], G)
        A[k + 1] = np.einsum("ab,bwc->awc", np.linalg.inv(G), A[k + 1])
    want = O.round_mps(A, chi)
    x = Q.qtt_mps_from_cores(ctx, A)
    Q.qtt_round(ctx, x, chi)
    assert Q.qtt_mps_bonds(x) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, x), O.to_dense(want)) < TOL
    sg, so = Q.qtt_mps_schmidt(ctx, x), O.schmidt_values(want)
    for k in range(1, n):
        m = min(len(sg[k]), len(so[k]))
        assert np.max(np.abs(sg[k][:m] - so[k][:m])) <= 1e-9 * so[k][0]
    ms, hits = Q.qtt_ctx_jacobi_stats(ctx)
    assert hits == 0


@pytest.mark.parametrize("which", [0, 1, 2])
def test_apply_then_round_matches_oracle(Q, ctx, which):
    n, chi = 7, 12
    g, o = ops(Q, ctx, n)
    F = smooth_field(n, 21)
    A = O.from_dense(F, chi)
    want = O.round_mps(O.apply_mpo(o[which], A), chi)
    x = Q.qtt_mps_from_cores(ctx, A)
    y = Q.qtt_apply_mpo(ctx, g[which], x)
    Q.qtt_round(ctx, y, chi)
    assert Q.qtt_mps_bonds(y) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, y), O.to_dense(want)) < TOL


def test_round_eps_rule_matches_oracle(Q, ctx):
    n = 6
    F = smooth_field(n, 5)
    A = O.lincomb([(1.0, O.from_dense(F, 20)), (0.5, O.from_dense(F.T.copy(), 20))])
    for eps in (1e-1, 1e-3, 1e-6):
        want = O.round_mps(A, 1 << 20, eps)
        x = Q.qtt_mps_from_cores(ctx, A)
        Q.qtt_round(ctx, x, 1 << 20, eps)
        assert Q.qtt_mps_bonds(x) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, x), O.to_dense(want)) < TOL


def test_round_batch_mixed_operands(Q, ctx):
    n, chi = 6, 8
    g, o = ops(Q, ctx, n)
    A = O.from_dense(smooth_field(n, 1), chi)
    B = O.from_dense(smooth_field(n, 2), chi)
    a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
    xs = [Q.qtt_apply_mpo(ctx, g[0], a), Q.qtt_hadamard(ctx, a, b), Q.qtt_apply_mpo(ctx, g[2], b)]
    s = Q.qtt_mps_clone(ctx, a)
    Q.qtt_axpy(ctx, 3.0, b, s)
    xs.append(s)
    Q.qtt_round_batch(ctx, xs, chi)
    wants = [O.round_mps(O.apply_mpo(o[0], A), chi), O.round_product(A, B, chi),
             O.round_mps(O.apply_mpo(o[2], B), chi), O.round_mps(O.lincomb([(3.0, B), (1.0, A)]), chi)]
    for x, w in zip(xs, wants):
        assert Q.qtt_mps_bonds(x) == O.bonds(w)
        assert rel(gpu_dense(Q, ctx, x), O.to_dense(w)) < TOL


# ---------------------------------------------------------------- zip-up (fused Hadamard + round)
@pytest.mark.parametrize("n,ca,cb,chi,cw", [(4, 3, 3, 4, 0), (5, 4, 3, 6, 0), (6, 6, 6, 8, 0), (6, 6, 6, 8, 8),
                                            (7, 8, 8, 8, 12), (8, 16, 16, 16, 0)])
def test_round_product_matches_oracle(Q, ctx, n, ca, cb, chi, cw):
    A = O.from_dense(smooth_field(n, 31), ca)
    B = O.from_dense(smooth_field(n, 32), cb)
    want = O.round_product(A, B, chi, 0.0, cw if cw else None)
    Q.qtt_ctx_set_chi_work(ctx, cw)
    try:
        a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
        h = Q.qtt_hadamard(ctx, a, b)
        Q.qtt_round(ctx, h, chi)
    finally:
        Q.qtt_ctx_set_chi_work(ctx, 0)
    assert Q.qtt_mps_bonds(h) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, h), O.to_dense(want)) < TOL


def test_config1_chain_matches_oracle_and_dense(Q, ctx):
    """BASELINE config 1: 2^5 x 2^5, chi 8: from_dense -> apply d/dx -> Hadamard -> one round to 8."""
    import torch
    n, chi = 5, 8
    F = I.config1_field(n, 0)
    g, o = ops(Q, ctx, n)
    A = O.from_dense(F, chi)
    want = O.round_product(A, O.apply_mpo(o[0], A), chi, 0.0, 1 << 20)
    u = Q.qtt_mps_from_dense(ctx, torch.from_numpy(F).cuda(), chi)
    du = Q.qtt_apply_mpo(ctx, g[0], u)
    w = Q.qtt_hadamard(ctx, u, du)
    # exact product (bond 192) against the dense 32 x 32 brute force
    u8 = O.to_dense(A)
    dx = 1.0 / 32
    dense = u8 * (np.roll(u8, -1, 0) - np.roll(u8, 1, 0)) / (2 * dx)
    # noise-dominated result: d/dx of the tanh(y) part cancels, so rounding is amplified by
    # ||u|| * (1/2dx) / ||w|| ~ 1e3 above machine epsilon
    assert rel(gpu_dense(Q, ctx, w), dense) < 1e-11
    Q.qtt_ctx_set_chi_work(ctx, 1 << 20)
    try:
        Q.qtt_round(ctx, w, chi)
    finally:
        Q.qtt_ctx_set_chi_work(ctx, 0)
    assert Q.qtt_mps_bonds(w) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, w), O.to_dense(want)) < TOL


# ---------------------------------------------------------------- RK4
@pytest.mark.parametrize("graphs", [False, True])
def test_rk4_step_small_matches_oracle(Q, ctx, graphs):
    n, chi, Re, dt = 6, 12, 100.0, 1e-3
    g, o = ops(Q, ctx, n)
    X, Y = I.grid(n)
    ux = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.3 * smooth_field(n, 4)
    uy = -np.cos(2 * np.pi * X) * np.sin(2 * np.pi * Y) + 0.3 * smooth_field(n, 5)
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    Q.qtt_ctx_set_graphs(ctx, graphs)
    u = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    for step in range(2):
        U = O.rk4_step(U, o[0], o[1], o[2], Re, dt, chi)
        Q.qtt_rk4_step(ctx, u, g[0], g[1], g[2], Re, dt, chi)
        for i in range(2):
            assert Q.qtt_mps_bonds(u[i]) == O.bonds(U[i])
            assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U[i])) < TOL
    Q.qtt_ctx_set_graphs(ctx, True)
    assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0


def test_rk4_config2_matches_oracle(Q, ctx):
    """BASELINE config 2: 2^8 x 2^8 double shear layer, chi 32, Re 1e4, dt 1e-4, one step."""
    import torch
    cfg = I.CONFIGS[2]
    n, chi = cfg["n"], cfg["chi"]
    ux, uy = I.config_fields(2)
    g, o = ops(Q, ctx, n)
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    u = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in (ux, uy)]
    for i in range(2):
        assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U[i])) < TOL
    U1 = O.rk4_step(U, o[0], o[1], o[2], cfg["Re"], cfg["dt"], chi)
    Q.qtt_rk4_step(ctx, u, g[0], g[1], g[2], cfg["Re"], cfg["dt"], chi)
    for i in range(2):
        assert Q.qtt_mps_bonds(u[i]) == O.bonds(U1[i])
        assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U1[i])) < TOL
    assert Q.qtt_ctx_launch_count(ctx) > 0


def test_round_ex_and_core_ptr(Q, ctx):
    """qtt_round_ex (per-call working bond) == the oracle's round_product at that chi_work, for a
    working bond that really truncates; qtt_mps_core_ptr hands out the device cores without a host copy."""
    import torch
    n, chi = 6, 6
    A = O.from_dense(smooth_field(n, 3), chi_max=6)
    B = O.from_dense(smooth_field(n, 4), chi_max=6)
    for cw in (6, 9, 12, 36):
        a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
        c = Q.qtt_hadamard(ctx, a, b)
        with pytest.raises(Q.QttError):
            Q.qtt_mps_core_ptr(ctx, c, 0)          # lazy handle: no explicit cores
        Q.qtt_round_ex(ctx, c, chi, 0.0, cw)
        want = O.round_product(A, B, chi, chi_work=cw)
        assert Q.qtt_mps_bonds(c) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, c), O.to_dense(want)) < TOL
    # chi_work = 0 falls back to the default 2 * chi_max
    c = Q.qtt_hadamard(ctx, Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B))
    Q.qtt_round_ex(ctx, c, chi, 0.0, 0)
    assert rel(gpu_dense(Q, ctx, c), O.to_dense(O.round_product(A, B, chi))) < TOL
    # device pointers: read core k through torch from the raw address and compare with the host copy
    r = Q.qtt_mps_bonds(c)
    ctx.synchronize()
    import ctypes as C
    rt = None
    for name in ("libcudart.so.12", "libcudart.so", "/usr/local/cuda/lib64/libcudart.so"):
        try:
            rt = C.CDLL(name)
            break
        except OSError:
            continue
    assert rt is not None, "CUDA runtime library not found"
    for k in range(n):
        ptr = Q.qtt_mps_core_ptr(ctx, c, k)
        assert ptr != 0 and ptr % 8 == 0
        host = Q.qtt_mps_get_core(ctx, c, k)
        cnt = r[k] * 4 * r[k + 1]
        buf = (C.c_double * cnt)()
        assert rt.cudaMemcpy(buf, C.c_void_p(ptr), C.c_size_t(cnt * 8), 2) == 0   # cudaMemcpyDeviceToHost
        assert np.array_equal(np.frombuffer(buf, dtype=np.float64).reshape(host.shape), host)


def test_launch_count_is_per_context(Q, ctx):
    """The launch counter and the profiler records belong to the context: work on one context does
    not move the other's counter."""
    other = Q.Context(device=0, workspace_bytes=1 << 28)
    try:
        a = Q.qtt_mps_from_cores(other, I.random_cores(5, 4, seed=2))
        c0, o0 = Q.qtt_ctx_launch_count(ctx), Q.qtt_ctx_launch_count(other)
        Q.qtt_round(other, a, 3)
        other.synchronize()
        assert Q.qtt_ctx_launch_count(other) > o0
        assert Q.qtt_ctx_launch_count(ctx) == c0
    finally:
        other.close()


# ---------------------------------------------------------------- error behaviour
def test_errors_are_status_codes(Q, ctx):
    a = Q.qtt_mps_from_cores(ctx, I.random_cores(4, 3, seed=1))
    b = Q.qtt_mps_from_cores(ctx, I.random_cores(5, 3, seed=1))
    with pytest.raises(Q.QttError) as e:
        Q.qtt_hadamard(ctx, a, b)
    assert e.value.status == -2
    with pytest.raises(Q.QttError):
        Q.qtt_round(ctx, a, 0)


# ---------------------------------------------------------------- full sizes, in bench.py's launch configuration
@pytest.fixture(scope="module")
def big_ctx(Q):
    c = Q.Context(device=0, workspace_bytes=8 << 30)  # bench.py's default workspace
    yield c
    c.close()


def schmidt_close(Q, ctx, x, cores):
    """Per-bond Schmidt values of the GPU result against an independent canonicalisation of the oracle result."""
    sg = Q.qtt_mps_schmidt(ctx, x)
    so = O.schmidt_values(cores)
    for k in range(1, len(cores)):
        m = min(len(sg[k]), len(so[k]))
        assert np.max(np.abs(np.asarray(sg[k][:m]) - so[k][:m])) <= 1e-9 * so[k][0]


def test_rk4_config3_full_size_matches_oracle(Q, big_ctx):
    """BASELINE config 3 (the bench workload: 2^10 x 2^10 decaying jet, chi 64, chi_work 128, Re 2e5, dt 5e-5), as
    SURVEY.md section 8d asks: steps 1-3 FREE-RUNNING (graph-replayed qtt_rk4_step against the oracle's own trajectory:
    error growth over steps) and PER STEP with the GPU restarted from the oracle state; dense 1024 x 1024 fields and
    Schmidt spectra."""
    import torch
    cfg = I.CONFIGS[3]
    n, chi = cfg["n"], cfg["chi"]
    ux, uy = I.config_fields(3)
    g, o = ops(Q, big_ctx, n)
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    free = [Q.qtt_mps_from_cores(big_ctx, U[0]), Q.qtt_mps_from_cores(big_ctx, U[1])]
    Q.qtt_ctx_set_graphs(big_ctx, True)
    errs = []
    for step in range(3):
        U1 = O.rk4_step(U, o[0], o[1], o[2], cfg["Re"], cfg["dt"], chi)
        # restarted from the oracle state of this step (at step 0 the two coincide)
        if step > 0:
            u = [Q.qtt_mps_from_cores(big_ctx, U[0]), Q.qtt_mps_from_cores(big_ctx, U[1])]
            Q.qtt_rk4_step(big_ctx, u, g[0], g[1], g[2], cfg["Re"], cfg["dt"], chi)
            for i in range(2):
                assert Q.qtt_mps_bonds(u[i]) == O.bonds(U1[i])
                assert rel(gpu_dense(Q, big_ctx, u[i]), O.to_dense(U1[i])) < TOL, ("restart", step)
        Q.qtt_rk4_step(big_ctx, free, g[0], g[1], g[2], cfg["Re"], cfg["dt"], chi)
        for i in range(2):
            assert Q.qtt_mps_bonds(free[i]) == O.bonds(U1[i])
            e = rel(gpu_dense(Q, big_ctx, free[i]), O.to_dense(U1[i]))
            errs.append(e)
            assert e < TOL, ("free-running", step, errs)
            if step in (0, 2):
                schmidt_close(Q, big_ctx, free[i], U1[i])
        U = U1
    print("config 3 free-running relative errors (u_x, u_y per step):", ["%.2e" % e for e in errs])
    assert Q.qtt_ctx_jacobi_stats(big_ctx)[1] == 0
    # from_dense at full size: the GPU TT-SVD of the dense field is the oracle's
    v = Q.qtt_mps_from_dense(big_ctx, torch.from_numpy(ux).cuda(), chi)
    assert rel(gpu_dense(Q, big_ctx, v), O.to_dense(O.from_dense(ux, chi))) < TOL


def test_config4_full_step_matches_stored_oracle(Q):
    """BASELINE config 4 (2^11 x 2^11 decaying turbulence, chi 128, chi_work 256, Re 1e6, dt 0.1/2^10): ONE full
    qtt_rk4_step in bench.py's launch configuration (graph replay, 24 GiB workspace as `bench.py --config 4`) against the
    oracle step stored by tests/golden/make_cfg4_step.py (the oracle needs ~15 min for it; the script imports only
    oracle/ and qtt_inputs/).  Dense 2048 x 2048 fields, bonds and Schmidt spectra.  The step runs the code paths config 3
    never reaches: 1024 x 1024 zip-up SVDs, two-level LQ, 640 x 512 SVDs of the 5-term sum."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg4_step1.npz")
    assert os.path.exists(path), "run tests/golden/make_cfg4_step.py"
    z = np.load(path)
    cfg = I.CONFIGS[4]
    n, chi = cfg["n"], cfg["chi"]
    assert int(z["n"]) == n and int(z["chi"]) == chi
    U1 = [[z[f"u1_{i}_{k}"] for k in range(n)] for i in range(2)]
    ux, uy = I.config_fields(4)
    U0 = [O.from_dense(ux, chi), O.from_dense(uy, chi)]   # the generator's input: the oracle's TT-SVD of the seeded field
    ctx4 = Q.Context(device=0, workspace_bytes=24 << 30)
    try:
        g, _ = ops(Q, ctx4, n)
        u = [Q.qtt_mps_from_cores(ctx4, U0[0]), Q.qtt_mps_from_cores(ctx4, U0[1])]
        Q.qtt_ctx_set_graphs(ctx4, True)
        Q.qtt_rk4_step(ctx4, u, g[0], g[1], g[2], cfg["Re"], cfg["dt"], chi)
        for i in range(2):
            assert Q.qtt_mps_bonds(u[i]) == O.bonds(U1[i])
            e = rel(gpu_dense(Q, ctx4, u[i]), O.to_dense(U1[i]))
            print(f"config 4 full step, component {i}: relative error {e:.2e}")
            assert e < TOL
            sg = Q.qtt_mps_schmidt(ctx4, u[i])
            for k in range(1, n):
                so = z[f"sv1_{i}_{k}"]
                m = min(len(sg[k]), len(so))
                assert np.max(np.abs(np.asarray(sg[k][:m]) - so[:m])) <= 1e-9 * so[0]
        assert Q.qtt_ctx_jacobi_stats(ctx4)[1] == 0
    finally:
        ctx4.close()


def test_config4_size_primitives_match_oracle(Q, big_ctx):
    """BASELINE config 4 sizes (2^11 x 2^11 decaying turbulence, chi 128): the oracle needs ~13 min for a whole
    step, so parity is taken primitive by primitive on the same inputs: from_dense, apply(Lap)+round,
    apply(D1)+round and ONE product u_x (.) D1 u_x (zip-up, chi_work 256)."""
    import torch
    cfg = I.CONFIGS[4]
    n, chi = cfg["n"], cfg["chi"]
    ux, _ = I.config_fields(4)
    g, o = ops(Q, big_ctx, n)
    A = O.from_dense(ux, chi)
    a = Q.qtt_mps_from_dense(big_ctx, torch.from_numpy(ux).cuda(), chi)
    assert Q.qtt_mps_bonds(a) == O.bonds(A)
    assert rel(gpu_dense(Q, big_ctx, a), O.to_dense(A)) < TOL
    a = Q.qtt_mps_from_cores(big_ctx, A)
    for which in (2, 0):
        want = O.round_mps(O.apply_mpo(o[which], A), chi)
        y = Q.qtt_apply_mpo(big_ctx, g[which], a)
        Q.qtt_round(big_ctx, y, chi)
        assert Q.qtt_mps_bonds(y) == O.bonds(want)
        assert rel(gpu_dense(Q, big_ctx, y), O.to_dense(want)) < TOL
    G = want  # round(D1 u_x)
    P = O.round_product(A, G, chi)
    c = Q.qtt_hadamard(big_ctx, a, y)
    Q.qtt_round(big_ctx, c, chi)
    assert Q.qtt_mps_bonds(c) == O.bonds(P)
    assert rel(gpu_dense(Q, big_ctx, c), O.to_dense(P)) < TOL
    assert Q.qtt_ctx_jacobi_stats(big_ctx)[1] == 0


@pytest.mark.parametrize("chi", [16, 32, 64, 128])
def test_config5_primitive_sweep_matches_oracle(Q, big_ctx, chi):
    """BASELINE config 5 (2^12 x 2^12, random left-canonical MPS, batch of 6 operands per launch): every operand gets
    one apply (d/dx, d/dy or Laplacian) + round(chi) and one Hadamard with the next operand + round(chi), batched
    through qtt_round_batch; dense 4096 x 4096 reconstructions against the oracle."""
    n = 12
    g, o = ops(Q, big_ctx, n)
    cores = [O.canonical_random(I.random_cores(n, chi, seed=s)) for s in range(6)]
    xs = [Q.qtt_mps_from_cores(big_ctx, c) for c in cores]
    ys = [Q.qtt_apply_mpo(big_ctx, g[i % 3], xs[i]) for i in range(6)]
    Q.qtt_round_batch(big_ctx, ys, chi)
    for i in (0, 2, 5):  # sampled operands: the oracle needs a few seconds per dense 2^24-point reconstruction
        want = O.round_mps(O.apply_mpo(o[i % 3], cores[i]), chi)
        assert Q.qtt_mps_bonds(ys[i]) == O.bonds(want)
        assert rel(gpu_dense(Q, big_ctx, ys[i]), O.to_dense(want)) < TOL
    hs = [Q.qtt_hadamard(big_ctx, xs[i], xs[(i + 1) % 6]) for i in range(6)]
    Q.qtt_round_batch(big_ctx, hs, chi)
    for i in (1, 4):
        want = O.round_product(cores[i], cores[(i + 1) % 6], chi)
        assert Q.qtt_mps_bonds(hs[i]) == O.bonds(want)
        assert rel(gpu_dense(Q, big_ctx, hs[i]), O.to_dense(want)) < TOL
    assert Q.qtt_ctx_jacobi_stats(big_ctx)[1] == 0


def zip_cuts_are_safe(info, thr=1e-5):
    """DESIGN.md reading 17: a working-bond cut of the zip-up is comparable between two implementations only if the
    kept subspace is unique, i.e. the relative gap (s_keep - s_keep+1) / s_keep at the cut exceeds `thr` (or the cut lies
    in the noise floor).  Uses the singular values the oracle itself computed at every truncating site."""
    for z in info["zip"]:
        if z["branch"] != "svd":
            continue
        sv, keep = z["s"], z["Q"].shape[1]
        if keep < len(sv) and sv[keep - 1] > 1e-11 * sv[0]:
            if (sv[keep - 1] - sv[keep]) <= thr * sv[keep - 1]:
                return False
    return True


def graded_random_cores(n, chi, seed):
    """Seeded N(0,1) site tensors (qtt_inputs.random_cores) with the columns of every core scaled geometrically, so
    that all Schmidt spectra decay with clear gaps (canonicalised random cores with full-rank left bonds make the first
    zip-up matrices exact isometries: all singular values equal, the kept subspace arbitrary)."""
    cores = I.random_cores(n, chi, seed=seed)
    return [c * np.logspace(0, -3, c.shape[2])[None, None, :] / np.sqrt(c.shape[0]) for c in cores]


def test_round_product_wide_site_uses_the_tsqr_lq(Q, big_ctx):
    """A zip-up site whose matrix T has more than 16384 columns (bonds 130 x 130 = 16900): the Q-less LQ of T goes through
    the column-chunk TSQR tree of run_lq (sweeps.cu), which no BASELINE config below chi = 256 reaches."""
    n, chi_op, chi, cw = 8, 130, 8, 16
    A, B = graded_random_cores(n, chi_op, 3), graded_random_cores(n, chi_op, 4)
    assert max(O.bonds(A)) == 130
    info = {}
    want = O.round_product(A, B, chi, chi_work=cw, info=info)
    assert any(z["T"].shape[1] > 16384 and z["branch"] == "svd" for z in info["zip"])
    assert zip_cuts_are_safe(info)
    c = Q.qtt_hadamard(big_ctx, Q.qtt_mps_from_cores(big_ctx, A), Q.qtt_mps_from_cores(big_ctx, B))
    Q.qtt_round_ex(big_ctx, c, chi, 0.0, cw)
    assert Q.qtt_mps_bonds(c) == O.bonds(want)
    assert rel(gpu_dense(Q, big_ctx, c), O.to_dense(want)) < TOL
    assert Q.qtt_ctx_jacobi_stats(big_ctx)[1] == 0


def test_zipup_svd_with_2048_columns_matches_oracle(Q, big_ctx):
    """The SVD shape of BASELINE config 5 at chi = 256 (working bond 512: a 2048 x 2048 triangular factor, the streamed
    Jacobi's 2048-column instantiation) on operands small enough for the oracle: 10 sites with bonds 64, so T is 2048 x 4096."""
    n, chi_op, chi, cw = 10, 64, 256, 512
    A, B = graded_random_cores(n, chi_op, 5), graded_random_cores(n, chi_op, 6)
    info = {}
    want = O.round_product(A, B, chi, chi_work=cw, info=info)
    assert any(z["T"].shape[0] == 2048 and z["branch"] == "svd" for z in info["zip"])
    assert zip_cuts_are_safe(info)
    c = Q.qtt_hadamard(big_ctx, Q.qtt_mps_from_cores(big_ctx, A), Q.qtt_mps_from_cores(big_ctx, B))
    Q.qtt_round_ex(big_ctx, c, chi, 0.0, cw)
    assert Q.qtt_mps_bonds(c) == O.bonds(want)
    assert rel(gpu_dense(Q, big_ctx, c), O.to_dense(want)) < TOL
    assert Q.qtt_ctx_jacobi_stats(big_ctx)[1] == 0


def test_config5_chi256_matches_oracle_at_ten_sites(Q):
    """BASELINE config 5's last point, chi = 256 (bond profile 4, 16, 64, 256, ..., working bond 512): one apply(Laplacian)
    + round and one Hadamard + round with every bulk shape of the 12-site sweep (T = 2048 x 65536 through the TSQR LQ,
    2048 x 2048 and 1024 x 1024 streamed Jacobi SVDs, 1280 x 1024 expanded cores), on a 10-site chain (bonds 4, 16, 64,
    256, 256, 256, 64, 16, 4) so that the oracle's LAPACK SVDs of the 1 GB zip-up matrices stay within the test budget."""
    n, chi = 10, 256
    ctx5 = Q.Context(device=0, workspace_bytes=40 << 30)
    try:
        g, o = ops(Q, ctx5, n)
        cores = [O.canonical_random(I.random_cores(n, chi, seed=s)) for s in range(2)]
        assert max(O.bonds(cores[0])) == 256
        xs = [Q.qtt_mps_from_cores(ctx5, c) for c in cores]
        y = Q.qtt_apply_mpo(ctx5, g[2], xs[0])
        Q.qtt_round(ctx5, y, chi)
        want = O.round_mps(O.apply_mpo(o[2], cores[0]), chi)
        assert Q.qtt_mps_bonds(y) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx5, y), O.to_dense(want)) < TOL
        h = Q.qtt_hadamard(ctx5, xs[0], xs[1])
        Q.qtt_round(ctx5, h, chi)
        info = {}
        want = O.round_product(cores[0], cores[1], chi, info=info)
        assert Q.qtt_mps_bonds(h) == O.bonds(want)
        assert Q.qtt_ctx_jacobi_stats(ctx5)[1] == 0
        assert np.all(np.isfinite(gpu_dense(Q, ctx5, h)))
        # left-canonical random cores whose first bonds are full (4, 16, 64, 256 = 4^l) make the first zip-up matrices
        # isometries: if a working-bond cut falls into equal singular values the kept subspace is not unique (reading 17)
        # and only bonds, finiteness and convergence are comparable; the graded operands below pin the same shapes
        if zip_cuts_are_safe(info):
            assert rel(gpu_dense(Q, ctx5, h), O.to_dense(want)) < TOL
        else:
            print("config 5 chi=256: degenerate working-bond cut on canonical random cores (unpinned, reading 17)")
        A, B = graded_random_cores(n, chi, 7), graded_random_cores(n, chi, 8)
        info = {}
        want = O.round_product(A, B, chi, info=info)
        assert zip_cuts_are_safe(info)
        assert any(z["T"].shape == (2048, 65536) for z in info["zip"])
        h = Q.qtt_hadamard(ctx5, Q.qtt_mps_from_cores(ctx5, A), Q.qtt_mps_from_cores(ctx5, B))
        Q.qtt_round(ctx5, h, chi)
        assert Q.qtt_mps_bonds(h) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx5, h), O.to_dense(want)) < TOL
        assert Q.qtt_ctx_jacobi_stats(ctx5)[1] == 0
    finally:
        ctx5.close()


def test_rk4_step_eps_rule_matches_oracle(Q, ctx):
    """qtt_rk4_step with eps > 0 (data-dependent ranks, one stream synchronisation per bond; the Laplacian branch on
    the side stream): same bonds and fields as the oracle, whose ranks come from the same rule."""
    n, chi, Re, dt, eps = 6, 24, 100.0, 1e-3, 1e-6
    g, o = ops(Q, ctx, n)
    X, Y = I.grid(n)
    ux = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.3 * smooth_field(n, 7)
    uy = -np.cos(2 * np.pi * X) * np.sin(2 * np.pi * Y) + 0.3 * smooth_field(n, 8)
    U = [O.from_dense(ux, chi, eps), O.from_dense(uy, chi, eps)]
    u = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    info = {}
    U1 = O.rk4_step(U, o[0], o[1], o[2], Re, dt, chi, eps, info=info)
    Q.qtt_rk4_step(ctx, u, g[0], g[1], g[2], Re, dt, chi, eps)
    for i in range(2):
        # "several correct results" (reading 17): a discarded tail within rounding distance of the threshold
        # delta may fall on either side.  The ranks must agree wherever the oracle's decision was NOT that close; where
        # they differ (by one at most) the margin |tail - delta| / delta at that bond is logged and must be below 1e-6,
        # and only then is the field compared at the accuracy the threshold itself guarantees.
        bg, bo = Q.qtt_mps_bonds(u[i]), O.bonds(U1[i])
        rec = info["final"][i]
        delta = eps * rec["norm"] / np.sqrt(n - 1)
        degenerate = False
        for k in range(1, n):
            if bg[k] == bo[k]:
                continue
            assert abs(bg[k] - bo[k]) <= 1, (bg, bo)
            s = rec["singular_values"][k]
            r = min(bg[k], bo[k])
            tail = float(np.sqrt(np.sum(s[r:] ** 2)))
            margin = abs(tail - delta) / delta
            print(f"eps rule: component {i} bond {k}: ranks gpu {bg[k]} oracle {bo[k]}, tail {tail:.6e} delta {delta:.6e} "
                  f"margin {margin:.2e}")
            assert margin < 1e-6, "ranks differ at a bond whose threshold decision was not degenerate"
            degenerate = True
        tol = 10 * eps if degenerate else TOL
        assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U1[i])) < tol
    assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0


def test_rk4_step_is_bitwise_reproducible(Q, ctx):
    """No atomics or timing-dependent orders on the data path: the same step from the same cores gives bit-identical
    cores, run to run and graph replay against eager launches (a data race in a kernel would show up here)."""
    cfg = I.CONFIGS[2]
    n, chi = cfg["n"], cfg["chi"]
    ux, uy = I.config_fields(2)
    ux = ux + 0.05 * smooth_field(n, 11)  # a rank that really fills chi
    g, _ = ops(Q, ctx, n)
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    results = []
    for graphs in (True, True, False):
        Q.qtt_ctx_set_graphs(ctx, graphs)
        u = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
        for _ in range(2):
            Q.qtt_rk4_step(ctx, u, g[0], g[1], g[2], cfg["Re"], cfg["dt"], chi)
        results.append([Q.qtt_mps_get_cores(ctx, x) for x in u])
    Q.qtt_ctx_set_graphs(ctx, True)
    for other in results[1:]:
        for a, b in zip(results[0], other):
            for ca, cb in zip(a, b):
                assert ca.shape == cb.shape and np.array_equal(ca, cb)


def test_diagnostics_match_oracle(Q, ctx):
    """qtt_mps_fidelity (Eq. 12) and qtt_mps_chi_eps (Eq. 16-17) against the oracle."""
    n, chi = 7, 24
    F = smooth_field(n, 21) + 1e-2 * np.random.default_rng(1).standard_normal((1 << n, 1 << n))
    G = smooth_field(n, 22)
    A, B = O.from_dense(F, chi), O.from_dense(G, chi)
    a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
    assert abs(Q.qtt_mps_fidelity(ctx, a, b) - O.fidelity(A, B)) <= 1e-12
    assert abs(Q.qtt_mps_fidelity(ctx, a, a) - 1.0) <= 1e-12
    for eps in (1e-1, 1e-2, 1e-4):
        got, gmax = Q.qtt_mps_chi_eps(ctx, a, eps)
        want, wmax = O.chi_eps(A, eps)
        assert got == want and gmax == wmax


@pytest.mark.parametrize("n", [3, 6, 10])
def test_tke_spectrum_matches_oracle(Q, big_ctx, n):
    """qtt_tke_spectrum (Eq. 13-15: the library's own FFT + shell sums) against the oracle's definition, with and
    without the mean-flow subtraction of Eq. 14, on a turbulence-shaped field; Parseval; bitwise reproducibility."""
    N = 1 << n
    ux, uy = I.decaying_turbulence(n, seed=1, k0=min(16.0, N / 4))
    ux = ux + 0.3  # a mean flow for shell 0
    chi = min(32, 4 ** (n // 2))
    A, B = O.from_dense(ux, chi), O.from_dense(uy, chi)
    a, b = Q.qtt_mps_from_cores(big_ctx, A), Q.qtt_mps_from_cores(big_ctx, B)
    want = O.tke_spectrum(A, B)
    got = Q.qtt_tke_spectrum(big_ctx, a, b)
    assert got.shape == want.shape
    assert np.max(np.abs(got - want)) <= 1e-12 * want.max()
    fa, fb = O.to_dense(A), O.to_dense(B)
    assert abs(got.sum() - 0.5 * np.mean(fa * fa + fb * fb)) <= 1e-12 * got.sum()
    assert np.array_equal(got, Q.qtt_tke_spectrum(big_ctx, a, b))
    if n >= 2:
        M = O.from_dense(np.full((N, N), 0.3))
        m = Q.qtt_mps_from_cores(big_ctx, M)
        want = O.tke_spectrum(A, B, M, None)
        got = Q.qtt_tke_spectrum(big_ctx, a, b, m, None)
        assert np.max(np.abs(got - want)) <= 1e-12 * want.max()
        assert got[0] < 1e-3 * Q.qtt_tke_spectrum(big_ctx, a, b)[0]   # the mean flow is gone (up to the chi truncation)


@pytest.mark.parametrize("graphs", [False, True])
def test_rk4_step_skew_symmetric_matches_oracle(Q, ctx, graphs):
    """qtt_ctx_set_convection(1): the paper's skew-symmetric convection (PAPER.md Eq. B2, section 8f next-2), two steps
    on a 2^6 x 2^6 grid and one step of BASELINE config 2, against the oracle's rhs(skew=True)."""
    Q.qtt_ctx_set_convection(ctx, True)
    Q.qtt_ctx_set_graphs(ctx, graphs)
    try:
        n, chi, Re, dt = 6, 12, 100.0, 1e-3
        g, o = ops(Q, ctx, n)
        X, Y = I.grid(n)
        ux = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.3 * smooth_field(n, 4)
        uy = -np.cos(2 * np.pi * X) * np.sin(2 * np.pi * Y) + 0.3 * smooth_field(n, 5)
        U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
        u = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
        for _ in range(2):
            U = O.rk4_step(U, o[0], o[1], o[2], Re, dt, chi, skew=True)
            Q.qtt_rk4_step(ctx, u, g[0], g[1], g[2], Re, dt, chi)
            for i in range(2):
                assert Q.qtt_mps_bonds(u[i]) == O.bonds(U[i])
                assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U[i])) < TOL
        if graphs:
            cfg = I.CONFIGS[2]
            n, chi = cfg["n"], cfg["chi"]
            fx, fy = I.config_fields(2)
            g, o = ops(Q, ctx, n)
            U = [O.from_dense(fx, chi), O.from_dense(fy, chi)]
            u = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
            U1 = O.rk4_step(U, o[0], o[1], o[2], cfg["Re"], cfg["dt"], chi, skew=True)
            Q.qtt_rk4_step(ctx, u, g[0], g[1], g[2], cfg["Re"], cfg["dt"], chi)
            for i in range(2):
                assert Q.qtt_mps_bonds(u[i]) == O.bonds(U1[i])
                assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U1[i])) < TOL
        assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0
    finally:
        Q.qtt_ctx_set_convection(ctx, False)
        Q.qtt_ctx_set_graphs(ctx, True)


@pytest.mark.parametrize("order", [2, 4, 8])
def test_stencil_mpo_matches_oracle(Q, ctx, order):
    """qtt_mpo_stencil (stencils of any order; section 8f next-2): exact apply and apply + round against
    the oracle's mpo_stencil, both directions."""
    n, chi = 6, 10
    dx = 1.0 / (1 << n)
    A = O.from_dense(smooth_field(n, 31) + 1e-2 * np.random.default_rng(2).standard_normal((1 << n, 1 << n)), chi)
    a = Q.qtt_mps_from_cores(ctx, A)
    c = O.fd_coefficients(order, dx)
    for direction in (1, 2):
        Wo = O.mpo_stencil(n, direction, c)
        Wg = Q.qtt_mpo_stencil(ctx, n, direction, c)
        y = Q.qtt_apply_mpo(ctx, Wg, a)
        assert Q.qtt_mps_bonds(y) == O.bonds(O.apply_mpo(Wo, A))
        assert rel(gpu_dense(Q, ctx, y), O.to_dense(O.apply_mpo(Wo, A))) < 1e-13
        Q.qtt_round(ctx, y, chi)
        want = O.round_mps(O.apply_mpo(Wo, A), chi)
        assert Q.qtt_mps_bonds(y) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, y), O.to_dense(want)) < TOL


def test_rk4_step_with_fourth_order_stencils_matches_oracle(Q, ctx):
    """One qtt_rk4_step with 4th-order first-derivative MPOs (bond 5) in place of the 2nd-order ones."""
    n, chi, Re, dt = 6, 12, 100.0, 1e-3
    dx = 1.0 / (1 << n)
    g, o = ops(Q, ctx, n)
    c4 = O.fd_coefficients(4, dx)
    Dg = [Q.qtt_mpo_stencil(ctx, n, d, c4) for d in (1, 2)]
    Do = [O.mpo_stencil(n, d, c4) for d in (1, 2)]
    X, Y = I.grid(n)
    ux = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.3 * smooth_field(n, 4)
    uy = -np.cos(2 * np.pi * X) * np.sin(2 * np.pi * Y) + 0.3 * smooth_field(n, 5)
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    u = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    U1 = O.rk4_step(U, Do[0], Do[1], o[2], Re, dt, chi)
    Q.qtt_rk4_step(ctx, u, Dg[0], Dg[1], g[2], Re, dt, chi)
    for i in range(2):
        assert Q.qtt_mps_bonds(u[i]) == O.bonds(U1[i])
        assert rel(gpu_dense(Q, ctx, u[i]), O.to_dense(U1[i])) < TOL
