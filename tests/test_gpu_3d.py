"""GPU parity of the 3D encoding with physical dimension 8 (reading 26): the
qtt_* C ABI in a context switched with qtt_ctx_set_phys_dim(ctx, 8) against oracle/qtt_oracle_3d.py on the same seeded
inputs.  Bar as everywhere: <= 1e-10 relative on dense reconstructions, Schmidt spectra within 1e-9 sigma_1, bonds exact."""
import numpy as np
import pytest

import qtt_inputs as I
from oracle import qtt_oracle as O
from oracle import qtt_oracle_3d as O3

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def Q():
    import paper_2406_17823_b200 as q
    return q


@pytest.fixture(scope="module")
def ctx(Q):
    c = Q.Context(device=0, workspace_bytes=2 << 30)
    Q.qtt_ctx_set_phys_dim(c, 8)
    yield c
    c.close()


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def gpu_dense(Q, ctx, x):
    t = Q.qtt_to_dense(ctx, x)
    ctx.synchronize()
    return t.cpu().numpy()


def field3(n, seed):
    N = 1 << n
    rng = np.random.default_rng(seed)
    t = np.arange(N) / N
    X, Y, Z = np.meshgrid(t, t, t, indexing="ij")
    F = np.tanh((Y - 0.5) / 0.15) * np.cos(2 * np.pi * Z)
    for _ in range(6):
        k = rng.integers(-2, 3, size=3)
        F = F + rng.standard_normal() * np.cos(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + rng.uniform(0, 6.28))
    return F + 1e-3 * rng.standard_normal((N, N, N))


def test_phys_dim_switch_rules(Q, ctx):
    assert Q.qtt_ctx_phys_dim(ctx) == 8
    with pytest.raises(Q.QttError):
        Q.qtt_ctx_set_phys_dim(ctx, 5)
    x = Q.qtt_mps_from_cores(ctx, I.random_cores(3, 4, seed=1, d=8))
    with pytest.raises(Q.QttError):  # handles alive
        Q.qtt_ctx_set_phys_dim(ctx, 4)
    with pytest.raises(ValueError):  # 2D cores in a 3D context
        Q.qtt_mps_from_cores(ctx, I.random_cores(3, 4, seed=1, d=4))
    x.free()
    Q.qtt_ctx_set_phys_dim(ctx, 4)
    Q.qtt_ctx_set_phys_dim(ctx, 8)


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_from_cores_to_dense3(Q, ctx, n):
    cores = I.random_cores(n, 6, seed=n, d=8)
    x = Q.qtt_mps_from_cores(ctx, cores)
    assert Q.qtt_mps_bonds(x) == O.bonds(cores)
    got = gpu_dense(Q, ctx, x)
    assert got.shape == (1 << n,) * 3
    assert rel(got, O3.to_dense3(cores)) < 1e-13
    for k in range(n):
        assert np.array_equal(Q.qtt_mps_get_core(ctx, x, k), cores[k])


@pytest.mark.parametrize("n,chi", [(2, 100), (3, 1000), (4, 9), (5, 24), (6, 16)])
def test_from_dense3_matches_oracle(Q, ctx, n, chi):
    import torch
    F = field3(n, n)
    want = O3.from_dense3(F, chi)
    x = Q.qtt_mps_from_dense(ctx, torch.from_numpy(F).cuda(), chi)
    assert Q.qtt_mps_bonds(x) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, x), O3.to_dense3(want)) < TOL


def test_from_dense3_eps_rule(Q, ctx):
    import torch
    F = field3(4, 11)
    for eps in (1e-2, 1e-6):
        want = O3.from_dense3(F, 1 << 20, eps)
        x = Q.qtt_mps_from_dense(ctx, torch.from_numpy(F).cuda(), 1 << 20, eps)
        assert Q.qtt_mps_bonds(x) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, x), O3.to_dense3(want)) < TOL


def test_native_mpo_builders_match_oracle3(Q, ctx):
    n = 4
    dx = 1.0 / (1 << n)
    A = I.random_cores(n, 5, seed=2, d=8)
    x = Q.qtt_mps_from_cores(ctx, A)
    c = np.array([0.3, -1.1, 0.0, 2.0, 0.7])
    pairs = [(Q.qtt_mpo_central_difference(ctx, n, j, dx), O3.mpo_d3(n, j, dx)) for j in (1, 2, 3)]
    pairs += [(Q.qtt_mpo_stencil(ctx, n, j, c), O3.mpo_stencil3(n, j, c)) for j in (1, 2, 3)]
    pairs.append((Q.qtt_mpo_laplacian(ctx, n, dx), O3.mpo_laplacian3(n, dx)))
    for W, Wo in pairs:
        y = Q.qtt_apply_mpo(ctx, W, x)
        want = O.apply_mpo(Wo, A)
        assert Q.qtt_mps_bonds(y) == O.bonds(want)
        for k in range(n):  # the expanded cores element by element (exact: 0 / +-c weights)
            assert rel(Q.qtt_mps_get_core(ctx, y, k), want[k]) < 1e-15
    with pytest.raises(Q.QttError):
        Q.qtt_mpo_central_difference(ctx, n, 4, dx)
    # an MPO uploaded from the oracle's cores acts like the native one
    W2 = Q.qtt_mpo_create(ctx, O3.mpo_laplacian3(n, dx))
    assert rel(gpu_dense(Q, ctx, Q.qtt_apply_mpo(ctx, W2, x)), gpu_dense(Q, ctx, Q.qtt_apply_mpo(ctx, pairs[-1][0], x))) < 1e-15


@pytest.mark.parametrize("n,chi", [(3, 5), (4, 12), (5, 20)])
def test_apply_hadamard_axpy_round3(Q, ctx, n, chi):
    dx = 1.0 / (1 << n)
    A = O.canonical_random(I.random_cores(n, chi, seed=n, d=8))
    B = O.canonical_random(I.random_cores(n, max(chi // 2, 2), seed=n + 7, d=8))
    a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
    # exact lazy results
    h = Q.qtt_hadamard(ctx, a, b)
    if n <= 4:
        assert rel(gpu_dense(Q, ctx, h), O3.to_dense3(A) * O3.to_dense3(B)) < 1e-12
    s = Q.qtt_mps_clone(ctx, b)
    Q.qtt_axpy(ctx, -0.7, a, s)
    assert rel(gpu_dense(Q, ctx, s), O3.to_dense3(O.axpy(-0.7, A, B))) < 1e-13
    assert abs(Q.qtt_mps_dot(ctx, a, b) - O.dot(A, B)) < 1e-12
    # apply + round, sum + round, with the Schmidt spectra
    Wg, Wo = Q.qtt_mpo_laplacian(ctx, n, dx), O3.mpo_laplacian3(n, dx)
    y = Q.qtt_apply_mpo(ctx, Wg, a)
    Q.qtt_round(ctx, y, chi)
    want = O.round_mps(O.apply_mpo(Wo, A), chi)
    assert Q.qtt_mps_bonds(y) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, y), O3.to_dense3(want)) < TOL
    Q.qtt_round(ctx, s, chi)
    want = O.round_mps(O.axpy(-0.7, A, B), chi)
    assert Q.qtt_mps_bonds(s) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, s), O3.to_dense3(want)) < TOL
    sg, so = Q.qtt_mps_schmidt(ctx, s), O.schmidt_values(want)
    for k in range(1, n):
        m = min(len(sg[k]), len(so[k]))
        assert np.max(np.abs(sg[k][:m] - so[k][:m])) <= 1e-9 * so[k][0]
    # the zip-up: exact working bond and truncating working bonds
    for cw in (0, max(chi // 2, 3), chi + 1):
        p = Q.qtt_hadamard(ctx, a, b)
        Q.qtt_round_ex(ctx, p, chi, 0.0, cw)
        want = O.round_product(A, B, chi, chi_work=(cw if cw else None))
        assert Q.qtt_mps_bonds(p) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, p), O3.to_dense3(want)) < TOL
    # batched rounding of mixed operands
    p = Q.qtt_hadamard(ctx, a, b)
    y2 = Q.qtt_apply_mpo(ctx, Q.qtt_mpo_central_difference(ctx, n, 3, dx), b)
    Q.qtt_round_batch(ctx, [p, y2], chi)
    assert rel(gpu_dense(Q, ctx, p), O3.to_dense3(O.round_product(A, B, chi))) < TOL
    assert rel(gpu_dense(Q, ctx, y2), O3.to_dense3(O.round_mps(O.apply_mpo(O3.mpo_d3(n, 3, dx), B), chi))) < TOL


def test_round_eps_rule3(Q, ctx):
    n = 4
    A = O3.from_dense3(field3(n, 5), 40)
    a = Q.qtt_mps_from_cores(ctx, A)
    for eps in (1e-3, 1e-7):
        x = Q.qtt_mps_clone(ctx, a)
        Q.qtt_round(ctx, x, 1 << 20, eps)
        want = O.round_mps(A, 1 << 20, eps)
        assert Q.qtt_mps_bonds(x) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, x), O3.to_dense3(want)) < TOL


def test_rk4_step3_from_primitives_matches_oracle(Q, ctx):
    """A 3D Burgers RK4 step (Taylor-Green + noise, 16^3, chi = 12) composed from the C-ABI calls (batched per level: 12
    applies, 9 zip-ups, 3 sums per right-hand side) against oracle rk4_step3."""
    import torch
    n, chi, Re, dt = 4, 12, 100.0, 2e-3
    dx = 1.0 / (1 << n)
    u0 = list(I.taylor_green_3d(n, seed=0, noise=1e-3))
    Uo = [O3.from_dense3(f, chi) for f in u0]
    Djo = [O3.mpo_d3(n, j, dx) for j in (1, 2, 3)]
    Lapo = O3.mpo_laplacian3(n, dx)
    want = O3.rk4_step3(Uo, Djo, Lapo, Re, dt, chi)

    Dj = [Q.qtt_mpo_central_difference(ctx, n, j, dx) for j in (1, 2, 3)]
    Lap = Q.qtt_mpo_laplacian(ctx, n, dx)
    u = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in u0]

    def lincomb(terms):
        """sum alpha_j X_j; the last term must have weight 1 (it is the axpy's Y)."""
        assert terms[-1][0] == 1.0
        y = Q.qtt_mps_clone(ctx, terms[-1][1])
        for alpha, x in reversed(terms[:-1]):
            Q.qtt_axpy(ctx, alpha, x, y)
        return y

    def rhs(v):
        g = [[Q.qtt_apply_mpo(ctx, Dj[j], v[i]) for j in range(3)] for i in range(3)]
        lap = [Q.qtt_apply_mpo(ctx, Lap, v[i]) for i in range(3)]
        Q.qtt_round_batch(ctx, [x for row in g for x in row] + lap, chi)
        c = [[Q.qtt_hadamard(ctx, v[j], g[i][j]) for j in range(3)] for i in range(3)]
        Q.qtt_round_batch(ctx, [x for row in c for x in row], chi)
        f = []
        for i in range(3):
            # qtt_axpy weights the term it adds, the handle it adds to keeps weight 1: build Re * f_i = lap - Re (c_i1 + c_i2 + c_i3).
            # The rounding keeps chi singular triplets per bond, which do not depend on the scale or on the order of the
            # summands, so round(Re * f_i) = Re * round(f_i); the factor is undone in the stage weights below.
            y = Q.qtt_mps_clone(ctx, lap[i])
            for j in (2, 1, 0):
                Q.qtt_axpy(ctx, -Re, c[i][j], y)
            f.append(y)
        Q.qtt_round_batch(ctx, f, chi)
        return f

    def stage(k, h):
        out = [lincomb([(h / Re, k[i]), (1.0, u[i])]) for i in range(3)]
        Q.qtt_round_batch(ctx, out, chi)
        return out

    k1 = rhs(u)
    k2 = rhs(stage(k1, dt / 2))
    k3 = rhs(stage(k2, dt / 2))
    k4 = rhs(stage(k3, dt))
    out = [lincomb([(dt / 6 / Re, k1[i]), (dt / 3 / Re, k2[i]), (dt / 3 / Re, k3[i]), (dt / 6 / Re, k4[i]), (1.0, u[i])])
           for i in range(3)]
    Q.qtt_round_batch(ctx, out, chi)
    ctx.synchronize()
    assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0
    for i in range(3):
        assert Q.qtt_mps_bonds(out[i]) == O.bonds(want[i])
        ref = O3.to_dense3(want[i])
        # the step itself moves the field by far more than the bar
        assert rel(gpu_dense(Q, ctx, out[i]), ref) < TOL
        assert rel(ref, O3.to_dense3(Uo[i])) > 1e-6


@pytest.mark.parametrize("n,chi,eps", [(3, 64, 0.0), (4, 12, 0.0), (4, 10, 1e-6), (5, 16, 0.0)])
def test_rk4_step3_matches_oracle(Q, ctx, n, chi, eps):
    """qtt_rk4_step3 against oracle rk4_step3 (n = 3 with chi = 64: nothing truncates, so also == the dense RK4 the oracle is
    pinned to); two steps in a row at n = 4."""
    import torch
    Re, dt = 100.0, 2e-3
    dx = 1.0 / (1 << n)
    u0 = list(I.taylor_green_3d(n, seed=n, noise=1e-3))
    Uo = [O3.from_dense3(f, chi) for f in u0]
    Djo = [O3.mpo_d3(n, j, dx) for j in (1, 2, 3)]
    Lapo = O3.mpo_laplacian3(n, dx)
    Dj = [Q.qtt_mpo_central_difference(ctx, n, j, dx) for j in (1, 2, 3)]
    Lap = Q.qtt_mpo_laplacian(ctx, n, dx)
    u = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in u0]
    for step in range(2 if (n == 4 and eps == 0.0) else 1):
        Uo = O3.rk4_step3(Uo, Djo, Lapo, Re, dt, chi, eps)
        Q.qtt_rk4_step3(ctx, u, Dj, Lap, Re, dt, chi, eps)
        for i in range(3):
            if eps == 0.0:
                assert Q.qtt_mps_bonds(u[i]) == O.bonds(Uo[i])
            assert rel(gpu_dense(Q, ctx, u[i]), O3.to_dense3(Uo[i])) < (TOL if eps == 0.0 else 10 * eps)
    assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0
    if eps > 0.0:  # ranks by the eps rule: equal unless a singular value sits on the threshold (reading 17)
        for i in range(3):
            bg, bo = Q.qtt_mps_bonds(u[i]), O.bonds(Uo[i])
            assert all(abs(a - b) <= 1 for a, b in zip(bg, bo))


def test_rk4_step3_needs_a_3d_context(Q):
    c = Q.Context(device=0, workspace_bytes=256 << 20)
    try:
        n, dx = 3, 1.0 / 8
        a = [Q.qtt_mps_from_cores(c, I.random_cores(n, 4, seed=s)) for s in range(3)]
        D = [Q.qtt_mpo_central_difference(c, n, 1 + (j % 2), dx) for j in range(3)]
        with pytest.raises(Q.QttError):
            Q.qtt_rk4_step3(c, a, D, Q.qtt_mpo_laplacian(c, n, dx), 100.0, 1e-3, 4)
    finally:
        c.close()


def test_edge_cases3(Q, ctx):
    """One and two sites, a zero operand, bonds that already fit, chi = 1."""
    # one site: rounding is a copy, the dense cube is the core
    c1 = I.random_cores(1, 3, seed=4, d=8)
    x = Q.qtt_mps_from_cores(ctx, c1)
    Q.qtt_round(ctx, x, 2)
    assert rel(gpu_dense(Q, ctx, x), O3.to_dense3(c1)) < 1e-15
    assert abs(Q.qtt_mps_norm(ctx, x) - np.linalg.norm(c1[0])) < 1e-13
    # two sites, chi = 1 and chi beyond the full rank
    A = I.random_cores(2, 8, seed=5, d=8)
    for chi in (1, 3, 100):
        x = Q.qtt_mps_from_cores(ctx, A)
        Q.qtt_round(ctx, x, chi)
        want = O.round_mps(A, chi)
        assert Q.qtt_mps_bonds(x) == O.bonds(want)
        assert rel(gpu_dense(Q, ctx, x), O3.to_dense3(want)) < TOL
    # a zero operand stays zero through product, sum and rounding (no normalisation anywhere)
    n = 3
    Bc = I.random_cores(n, 4, seed=6, d=8)
    Z = [np.zeros_like(c) for c in Bc]
    b, z = Q.qtt_mps_from_cores(ctx, Bc), Q.qtt_mps_from_cores(ctx, Z)
    p = Q.qtt_hadamard(ctx, b, z)
    Q.qtt_round(ctx, p, 4)
    assert np.all(gpu_dense(Q, ctx, p) == 0.0)
    s = Q.qtt_mps_clone(ctx, b)
    Q.qtt_axpy(ctx, 2.0, z, s)
    Q.qtt_round(ctx, s, 4)
    assert rel(gpu_dense(Q, ctx, s), O3.to_dense3(O.round_mps(Bc, 4))) < TOL
    assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0


def test_bench_launch_configuration_zipups3(Q, ctx):
    """The launch configuration bench.py --three-d 6 --three-d-chi 32 times (64^3, chi = 32, chi_work = 64, a batch of nine
    zip-ups of 512 x 1024 site matrices and a batch of twelve applies): products and applies of one right-hand side against
    the oracle, operand by operand."""
    n, chi = 6, 32
    dx = 1.0 / (1 << n)
    u0 = list(I.taylor_green_3d(n, seed=0, noise=1e-3))
    Uo = [O3.from_dense3(f, chi) for f in u0]
    u = [Q.qtt_mps_from_cores(ctx, x) for x in Uo]  # both sides start from the same host cores
    Dj = [Q.qtt_mpo_central_difference(ctx, n, j, dx) for j in (1, 2, 3)]
    Lap = Q.qtt_mpo_laplacian(ctx, n, dx)
    Djo = [O3.mpo_d3(n, j, dx) for j in (1, 2, 3)]
    g = [[Q.qtt_apply_mpo(ctx, Dj[j], u[i]) for j in range(3)] for i in range(3)]
    lap = [Q.qtt_apply_mpo(ctx, Lap, u[i]) for i in range(3)]
    Q.qtt_round_batch(ctx, [x for row in g for x in row] + lap, chi)
    go = [[O.round_mps(O.apply_mpo(Djo[j], Uo[i]), chi) for j in range(3)] for i in range(3)]
    for i in range(3):
        for j in range(3):
            assert Q.qtt_mps_bonds(g[i][j]) == O.bonds(go[i][j])
            assert O.diff_norm([np.ascontiguousarray(c) for c in Q.qtt_mps_get_cores(ctx, g[i][j])], go[i][j]) < TOL * O.norm(go[i][j])
    lo = O.round_mps(O.apply_mpo(O3.mpo_laplacian3(n, dx), Uo[0]), chi)
    assert O.diff_norm([np.ascontiguousarray(c) for c in Q.qtt_mps_get_cores(ctx, lap[0])], lo) < TOL * O.norm(lo)
    c = [[Q.qtt_hadamard(ctx, u[j], g[i][j]) for j in range(3)] for i in range(3)]
    Q.qtt_round_batch(ctx, [x for row in c for x in row], chi)
    for i, j in ((0, 0), (0, 1), (1, 2), (2, 0)):  # sampled operands of the batch of nine (the oracle needs ~2 s each)
        want = O.round_product(Uo[j], go[i][j], chi)
        got = [np.ascontiguousarray(x) for x in Q.qtt_mps_get_cores(ctx, c[i][j])]
        assert Q.qtt_mps_bonds(c[i][j]) == O.bonds(want)
        assert O.diff_norm(got, want) < TOL * max(O.norm(want), 1e-300)
    assert Q.qtt_ctx_jacobi_stats(ctx)[1] == 0


def test_2d_only_calls_refuse_a_3d_context(Q, ctx):
    n = 3
    dx = 1.0 / (1 << n)
    a = Q.qtt_mps_from_cores(ctx, I.random_cores(n, 4, seed=1, d=8))
    b = Q.qtt_mps_from_cores(ctx, I.random_cores(n, 4, seed=2, d=8))
    D1, D2, L = (Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx),
                 Q.qtt_mpo_laplacian(ctx, n, dx))
    with pytest.raises(Q.QttError):
        Q.qtt_rk4_step(ctx, [a, b], D1, D2, L, 100.0, 1e-3, 4)
    with pytest.raises(Q.QttError):
        Q.qtt_tke_spectrum(ctx, a, b)
