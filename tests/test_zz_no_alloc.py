"""qtt_lq_noalloc (include/qtt_diag.h): the Q-less LQ with its scratch in a device array built into the library, for callers
that cannot allocate device memory.  Checked against the existing path (qtt_diag_lq with a caller-allocated buffer) on two
calls in a row that share the array, on the size limit, and on the device's free memory not moving across a call.
Named test_zz_* so that pytest collects it last: the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2406_17823_b200 as Q
    from paper_2406_17823_b200 import _lib
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return Q, _lib.load(), torch, torch.cuda.Stream()


def ptr(t):
    return C.c_void_p(t.data_ptr())


def existing_path(lib, torch, stream, Y):
    """qtt_diag_lq on a copy of Y with a torch-allocated scratch buffer."""
    batch, k, m = Y.shape
    dY = Y.clone()
    dR = torch.zeros((batch, k, k), dtype=torch.float64, device="cuda")
    scratch = torch.zeros(batch * 3 * 64 * m, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    assert lib.qtt_diag_lq(C.c_void_p(stream.cuda_stream), ptr(dY), batch, k, m, m, ptr(dR), ptr(scratch)) == 0
    stream.synchronize()
    return dR


def test_lq_noalloc_matches_the_existing_path_on_two_calls_in_a_row(env):
    Q, lib, torch, stream = env
    rng = np.random.default_rng(2406)
    # both shapes are too large for the cluster-resident kernel, so both really use the built-in scratch (batch * m <= 4096);
    # the second call finds the first one's contents in it
    shapes = [(1, 256, 4096), (2, 200, 2040)]
    Ys = [torch.from_numpy(rng.standard_normal(s)).cuda() for s in shapes]
    want = [existing_path(lib, torch, stream, Y) for Y in Ys]
    got = [torch.full((s[0], s[1], s[1]), float("nan"), dtype=torch.float64, device="cuda") for s in shapes]
    work = [Y.clone() for Y in Ys]
    torch.cuda.synchronize()
    Q.qtt_lq_noalloc(work[0].clone(), torch.empty_like(got[0]), stream)  # first use on this device: module load, attributes
    stream.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for Y, R in zip(work, got):  # two calls in a row on one stream, no synchronisation between them
        Q.qtt_lq_noalloc(Y, R, stream)
    stream.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0  # the calls took no device memory
    for Y, R, W in zip(Ys, got, want):
        R, W, Yh = R.cpu().numpy(), W.cpu().numpy(), Y.cpu().numpy()
        assert np.all(np.isfinite(R))
        for b in range(R.shape[0]):
            # the same kernels in the same order: equal to the existing path within the kernel tests' tolerance (1e-10)
            assert np.linalg.norm(R[b] - W[b]) <= 1e-10 * np.linalg.norm(W[b])
            assert np.allclose(np.tril(R[b], -1), 0.0)
            G = Yh[b] @ Yh[b].T
            assert np.linalg.norm(R[b].T @ R[b] - G) <= 1e-12 * np.linalg.norm(G)


def test_lq_noalloc_small_matrices_take_the_resident_kernel(env):
    Q, lib, torch, stream = env
    rng = np.random.default_rng(7)
    Y = torch.from_numpy(rng.standard_normal((3, 48, 768))).cuda()
    want = existing_path(lib, torch, stream, Y)
    R = torch.empty((3, 48, 48), dtype=torch.float64, device="cuda")
    Q.qtt_lq_noalloc(Y.clone(), R, stream)
    stream.synchronize()
    assert torch.linalg.norm(R - want) <= 1e-10 * torch.linalg.norm(want)


def test_lq_noalloc_rejects_sizes_beyond_the_built_in_scratch(env):
    Q, lib, torch, stream = env
    Y = torch.zeros((2, 64, 4096), dtype=torch.float64, device="cuda")  # batch * m = 8192 > 4096
    R = torch.full((2, 64, 64), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(ValueError, match="exceeds the built-in scratch"):
        Q.qtt_lq_noalloc(Y, R, stream)
    st = C.c_void_p(stream.cuda_stream)
    assert lib.qtt_lq_noalloc(st, ptr(Y), 2, 64, 4096, 4096, ptr(R)) == -2  # QTT_NOALLOC_TOO_LARGE
    assert lib.qtt_lq_noalloc(st, ptr(Y), 1, 64, 8192, 8192, ptr(R)) == -2
    assert lib.qtt_lq_noalloc(st, ptr(Y), 1, 64, 32, 32, ptr(R)) == -1  # QTT_NOALLOC_BAD_ARG: k > m
    assert lib.qtt_lq_noalloc(st, None, 1, 64, 4096, 4096, ptr(R)) == -1
    stream.synchronize()
    assert float(R.min()) == 7.0 and float(R.max()) == 7.0  # nothing was launched
