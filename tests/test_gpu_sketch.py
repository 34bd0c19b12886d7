"""GPU parity of the sketched zip-up ("a cheaper product compression"; reading 25):
qtt_ctx_set_product_compression(ctx, 1, seed) against the oracle's round_product(..., sketch_seed=seed) / rk4_step(...,
sketch_seed=seed), pinned by tests/test_oracle_sketch.py.  Both sides draw the same +-1 sign vectors over the physical
indices from the same counter-based generator and contract them through the product's own cores, so the sketched range is a
function of the state, not of the gauge its bonds happen to be in: the bar is the hot path's, 1e-10 relative on dense
reconstructions -- also when the operands reach the product through the library's own roundings (another gauge than the
oracle's)."""
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


@pytest.fixture()
def ctx(Q):
    c = Q.Context(device=0, workspace_bytes=4 << 30)
    yield c
    c.close()


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def gpu_dense(Q, ctx, x):
    t = Q.qtt_to_dense(ctx, x)
    ctx.synchronize()
    return t.cpu().numpy()


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


@pytest.mark.parametrize("n,chi0,chi,cw,seed", [(6, 16, 8, 16, 11), (7, 24, 12, 24, 5), (8, 32, 16, 20, 123456789), (6, 16, 8, 9, 0)])
def test_sketched_round_product_matches_oracle(Q, ctx, n, chi0, chi, cw, seed):
    Fa, Fb = fields(n, n + seed % 7)
    A, B = O.from_dense(Fa, chi0), O.from_dense(Fb, chi0)
    info = {}
    want = O.round_product(A, B, chi, chi_work=cw, sketch_seed=seed, info=info)
    assert "sketch" in [z["branch"] for z in info["zip"]]  # the case really exercises the sketch
    Q.qtt_ctx_set_product_compression(ctx, True, seed)
    a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
    h = Q.qtt_hadamard(ctx, a, b)
    Q.qtt_round_ex(ctx, h, chi, 0.0, cw)
    assert Q.qtt_mps_bonds(h) == O.bonds(want)
    assert rel(gpu_dense(Q, ctx, h), O.to_dense(want)) <= TOL
    # and it is a different result from the deterministic zip-up (the mode switch does something), which still works after
    Q.qtt_ctx_set_product_compression(ctx, False, 0)
    h2 = Q.qtt_hadamard(ctx, a, b)
    Q.qtt_round_ex(ctx, h2, chi, 0.0, cw)
    det = O.round_product(A, B, chi, chi_work=cw)
    assert rel(gpu_dense(Q, ctx, h2), O.to_dense(det)) <= TOL
    assert rel(O.to_dense(want), O.to_dense(det)) > 1e-6


def test_sketch_is_exact_when_the_working_bond_does_not_truncate(Q, ctx):
    n, chi = 5, 8
    Fa, Fb = fields(n, 2)
    A, B = O.from_dense(Fa, 4), O.from_dense(Fb, 4)
    Q.qtt_ctx_set_product_compression(ctx, True, 3)
    a, b = Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B)
    h = Q.qtt_hadamard(ctx, a, b)
    Q.qtt_round_ex(ctx, h, chi, 0.0, 1 << 20)
    want = O.round_mps(O.hadamard(A, B), chi)
    assert rel(gpu_dense(Q, ctx, h), O.to_dense(want)) <= TOL


@pytest.mark.parametrize("graphs", [False, True])
def test_rk4_step_with_sketched_products_matches_oracle(Q, ctx, graphs):
    n, chi, Re, dt, seed = 7, 6, 200.0, 1e-3, 3
    dx = 1.0 / (1 << n)
    Fa, Fb = fields(n, 5)
    U = [O.from_dense(Fa, chi), O.from_dense(0.5 * Fb, chi)]
    ops_o = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    ops_g = (Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx),
             Q.qtt_mpo_laplacian(ctx, n, dx))
    Q.qtt_ctx_set_graphs(ctx, graphs)
    Q.qtt_ctx_set_product_compression(ctx, True, seed)
    g = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    want = U
    for _ in range(2):
        Q.qtt_rk4_step(ctx, g, *ops_g, Re, dt, chi)
        want = O.rk4_step(want, *ops_o, Re, dt, chi, sketch_seed=seed)
    for i in range(2):
        assert rel(gpu_dense(Q, ctx, g[i]), O.to_dense(want[i])) <= TOL
    # switching the mode back re-captures the graph: the deterministic step again
    Q.qtt_ctx_set_product_compression(ctx, False, 0)
    g2 = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    Q.qtt_rk4_step(ctx, g2, *ops_g, Re, dt, chi)
    det = O.rk4_step(U, *ops_o, Re, dt, chi)
    for i in range(2):
        assert rel(gpu_dense(Q, ctx, g2[i]), O.to_dense(det[i])) <= TOL


def test_sketch_does_not_depend_on_the_gauge_of_the_operands(Q, ctx):
    """The second operand comes out of the library's own apply + round (a right-canonical form in ANOTHER gauge than the
    oracle's): the sketched product must still match -- a random matrix on the bond indices did not (0.13 instead of 1e-15)."""
    n, chi, seed = 7, 6, 3
    dx = 1.0 / (1 << n)
    Fa, Fb = fields(n, 5)
    U = [O.from_dense(Fa, chi), O.from_dense(0.5 * Fb, chi)]
    D = (O.mpo_d1(n, dx), O.mpo_d2(n, dx))
    Dg = (Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx))
    g = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    Q.qtt_ctx_set_product_compression(ctx, True, seed)
    for i in range(2):
        for j in range(2):
            go = O.round_mps(O.apply_mpo(D[j], U[i]), chi)
            info = {}
            want = O.round_product(U[j], go, chi, sketch_seed=seed, info=info)
            assert "sketch" in [z["branch"] for z in info["zip"]]
            gg = Q.qtt_apply_mpo(ctx, Dg[j], g[i])
            Q.qtt_round(ctx, gg, chi)
            h = Q.qtt_hadamard(ctx, g[j], gg)
            Q.qtt_round(ctx, h, chi)
            assert rel(gpu_dense(Q, ctx, h), O.to_dense(want)) <= TOL


def test_config3_full_size_sketched_steps_match_oracle(Q):
    """The launch configuration `bench.py --product-compression sketch` times (BASELINE config 3 shapes: 2^10 x 2^10, chi 64,
    chi_work = P = 128, graph replay): two free-running steps against the oracle's sketched steps with the same seed, dense
    1024 x 1024 fields; every kind of site occurs (many configurations to the right, few, and the deterministic ones between)."""
    cfg = I.CONFIGS[3]
    n, chi, seed = cfg["n"], cfg["chi"], 1
    dx = 1.0 / (1 << n)
    ux, uy = I.config_fields(3)
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    ops_o = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    info = {}
    O.round_product(U[0], U[1], chi, sketch_seed=seed, info=info)
    kinds = {(z["branch"], 4 ** (n - 1 - l) >= 4 * chi) for l, z in enumerate(info["zip"])}
    assert ("sketch", True) in kinds and ("sketch", False) in kinds
    c = Q.Context(device=0, workspace_bytes=8 << 30)
    try:
        ops_g = (Q.qtt_mpo_central_difference(c, n, 1, dx), Q.qtt_mpo_central_difference(c, n, 2, dx), Q.qtt_mpo_laplacian(c, n, dx))
        Q.qtt_ctx_set_graphs(c, True)
        Q.qtt_ctx_set_product_compression(c, True, seed)
        g = [Q.qtt_mps_from_cores(c, U[0]), Q.qtt_mps_from_cores(c, U[1])]
        for step in range(2):
            U = O.rk4_step(U, *ops_o, cfg["Re"], cfg["dt"], chi, sketch_seed=seed)
            Q.qtt_rk4_step(c, g, *ops_g, cfg["Re"], cfg["dt"], chi)
            for i in range(2):
                assert Q.qtt_mps_bonds(g[i]) == O.bonds(U[i])
                assert rel(gpu_dense(Q, c, g[i]), O.to_dense(U[i])) <= TOL, (step, i)
        assert Q.qtt_ctx_jacobi_stats(c)[1] == 0
    finally:
        c.close()


@pytest.mark.parametrize("skew,eps", [(True, 0.0), (False, 1e-6)])
def test_sketch_composes_with_skew_convection_and_the_eps_rule(Q, ctx, skew, eps):
    """The mode switch is orthogonal to the other two: the paper's skew-symmetric convection (7 products per right-hand side
    through the sketched zip-up) and the eps rank rule (data-dependent ranks, eager launches)."""
    n, chi, Re, dt, seed = 7, 6, 200.0, 1e-3, 17
    dx = 1.0 / (1 << n)
    Fa, Fb = fields(n, 8)
    U = [O.from_dense(Fa, chi), O.from_dense(0.5 * Fb, chi)]
    ops_o = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    ops_g = (Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx),
             Q.qtt_mpo_laplacian(ctx, n, dx))
    Q.qtt_ctx_set_convection(ctx, skew)
    Q.qtt_ctx_set_product_compression(ctx, True, seed)
    g = [Q.qtt_mps_from_cores(ctx, U[0]), Q.qtt_mps_from_cores(ctx, U[1])]
    Q.qtt_rk4_step(ctx, g, *ops_g, Re, dt, chi, eps)
    want = O.rk4_step(U, *ops_o, Re, dt, chi, eps=eps, skew=skew, sketch_seed=seed)
    for i in range(2):
        same = Q.qtt_mps_bonds(g[i]) == O.bonds(want[i])
        assert same or eps > 0.0  # eps > 0: a tail within rounding distance of the threshold may fall on either side (reading 17)
        assert rel(gpu_dense(Q, ctx, g[i]), O.to_dense(want[i])) <= (TOL if same else 10 * eps)


def test_sketch_edge_cases_short_chains_and_a_zero_operand(Q, ctx):
    """Chains too short for any site to satisfy the rule fall back to the deterministic zip-up; a zero operand gives a zero
    product (the sketch of a zero matrix has rank 0: every basis column is zero)."""
    Q.qtt_ctx_set_product_compression(ctx, True, 5)
    for n in (1, 2, 3):
        Fa, Fb = fields(n, n)
        A, B = O.from_dense(Fa, 4), O.from_dense(Fb, 4)
        info = {}
        want = O.round_product(A, B, 2, chi_work=2, sketch_seed=5, info=info)
        h = Q.qtt_hadamard(ctx, Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, B))
        Q.qtt_round_ex(ctx, h, 2, 0.0, 2)
        assert rel(gpu_dense(Q, ctx, h), O.to_dense(want)) <= TOL
    n, chi = 7, 6
    Fa, _ = fields(n, 4)
    A = O.from_dense(Fa, chi)
    Z = [np.zeros_like(c) for c in A]
    info = {}
    want = O.round_product(A, Z, chi, sketch_seed=5, info=info)
    assert "sketch" in [z["branch"] for z in info["zip"]] and np.all(O.to_dense(want) == 0.0)
    h = Q.qtt_hadamard(ctx, Q.qtt_mps_from_cores(ctx, A), Q.qtt_mps_from_cores(ctx, Z))
    Q.qtt_round(ctx, h, chi)
    got = gpu_dense(Q, ctx, h)
    assert np.all(np.isfinite(got)) and np.all(got == 0.0)
