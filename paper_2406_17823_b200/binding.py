"""Thin Python binding of the C ABI in include/qtt.h: argument marshalling only.

PyTorch is used for device memory (the alloc/release callbacks hand out torch-owned blocks) and for
the CUDA stream; every numerical step runs in the kernels of libqtt_b200.so.  Function names follow
the C ABI (``qtt_mps_from_dense`` ...).  Errors raise :class:`QttError` with the library's message.
"""
from __future__ import annotations

import ctypes as C
from typing import Sequence

import numpy as np
import torch

from . import _lib


class QttError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_lib.STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class Context:
    """qtt_ctx: one CUDA device, one stream, one workspace.  Owns the torch blocks the library asks for."""

    def __init__(self, device: int = 0, workspace_bytes: int = 1 << 30, stream: "torch.cuda.Stream | None" = None):
        self.lib = _lib.load()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libqtt_b200 has no CPU fallback")
        self.device = torch.device("cuda", device)
        # stream capture (CUDA graphs) is not allowed on the legacy default stream
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        self._blocks: dict[int, torch.Tensor] = {}

        def _alloc(nbytes, _user):
            # the block is used only on self.stream and may be released with work still queued there (qtt.h): allocate
            # it UNDER that stream, so torch's caching allocator hands it back only to later work on the same stream
            try:
                with torch.cuda.stream(self.stream):
                    t = torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device=self.device)
            except Exception:
                return None
            self._blocks[t.data_ptr()] = t
            return t.data_ptr()

        def _release(ptr, _user):
            self._blocks.pop(ptr, None)

        self._alloc_cb = _lib.ALLOC_FN(_alloc)
        self._release_cb = _lib.RELEASE_FN(_release)
        h = C.c_void_p()
        st = self.lib.qtt_ctx_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream), self._alloc_cb,
                                     self._release_cb, None, workspace_bytes)
        if st != _lib.QTT_OK:
            raise QttError(st, "qtt_ctx_create failed")
        self.h = h

    def check(self, st: int):
        if st != _lib.QTT_OK:
            raise QttError(st, self.lib.qtt_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.lib.qtt_ctx_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize(self):
        self.stream.synchronize()


class Mps:
    def __init__(self, ctx: Context, h):
        self.ctx, self.h = ctx, h

    def free(self):
        if self.h and self.ctx.h:
            self.ctx.lib.qtt_mps_free(self.h)
        self.h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Mpo:
    def __init__(self, ctx: Context, h):
        self.ctx, self.h = ctx, h

    def free(self):
        if self.h and self.ctx.h:
            self.ctx.lib.qtt_mpo_free(self.h)
        self.h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def _cores_args(cores: Sequence[np.ndarray], ndim: int):
    arrs = [np.ascontiguousarray(c, dtype=np.float64) for c in cores]
    for a in arrs:
        if a.ndim != ndim:
            raise ValueError(f"cores must have {ndim} dimensions")
    n = len(arrs)
    bonds = (C.c_int * (n + 1))(*([a.shape[0] for a in arrs] + [arrs[-1].shape[-1]]))
    ptrs = (C.POINTER(C.c_double) * n)(*[a.ctypes.data_as(C.POINTER(C.c_double)) for a in arrs])
    return arrs, n, bonds, ptrs


# ------------------------------------------------------------------ the calls of include/qtt.h
def qtt_mps_from_dense(ctx: Context, dense: torch.Tensor, chi_max: int, eps: float = 0.0) -> Mps:
    """dense: N x N fp64 CUDA tensor F[x][y] (N x N x N, F[x][y][z], in a context of physical dimension 8)."""
    ndim = 3 if qtt_ctx_phys_dim(ctx) == 8 else 2
    if dense.dtype != torch.float64 or not dense.is_cuda or dense.dim() != ndim or len(set(dense.shape)) != 1:
        raise ValueError(f"dense must be a fp64 CUDA tensor with {ndim} equal dimensions")
    dense = dense.contiguous()
    n = int(dense.shape[0]).bit_length() - 1
    if (1 << n) != dense.shape[0]:
        raise ValueError("N must be a power of two")
    ctx.stream.wait_stream(torch.cuda.current_stream(ctx.device))
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mps_from_dense(ctx.h, C.c_void_p(dense.data_ptr()), n, int(chi_max), float(eps), C.byref(h)))
    dense.record_stream(ctx.stream)
    return Mps(ctx, h)


def _check_phys(ctx: Context, arrs, axes) -> None:
    d = qtt_ctx_phys_dim(ctx)
    for a in arrs:
        if any(a.shape[ax] != d for ax in axes):
            raise ValueError(f"site tensors of this context have physical dimension {d}")


def qtt_mps_from_cores(ctx: Context, cores: Sequence[np.ndarray]) -> Mps:
    arrs, n, bonds, ptrs = _cores_args(cores, 3)
    _check_phys(ctx, arrs, (1,))
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mps_from_cores(ctx.h, n, bonds, ptrs, C.byref(h)))
    return Mps(ctx, h)


def qtt_to_dense(ctx: Context, x: Mps) -> torch.Tensor:
    n = ctx.lib.qtt_mps_num_sites(x.h)
    N = 1 << n
    out = torch.empty((N,) * (3 if qtt_ctx_phys_dim(ctx) == 8 else 2), dtype=torch.float64, device=ctx.device)
    ctx.stream.wait_stream(torch.cuda.current_stream(ctx.device))
    ctx.check(ctx.lib.qtt_to_dense(ctx.h, x.h, C.c_void_p(out.data_ptr())))
    out.record_stream(ctx.stream)
    torch.cuda.current_stream(ctx.device).wait_stream(ctx.stream)
    return out


def qtt_mpo_create(ctx: Context, cores: Sequence[np.ndarray]) -> Mpo:
    arrs, n, bonds, ptrs = _cores_args(cores, 4)
    _check_phys(ctx, arrs, (1, 2))
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mpo_create(ctx.h, n, bonds, ptrs, C.byref(h)))
    return Mpo(ctx, h)


def qtt_mpo_central_difference(ctx: Context, n_sites: int, direction: int, dx: float) -> Mpo:
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mpo_central_difference(ctx.h, n_sites, direction, float(dx), C.byref(h)))
    return Mpo(ctx, h)


def qtt_mpo_stencil(ctx: Context, n_sites: int, direction: int, coeffs: Sequence[float]) -> Mpo:
    """(O F)[x] = sum_k coeffs[k + K] F[x + k], 2K + 1 = len(coeffs), along direction 1 (x) or 2 (y)."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    if c.ndim != 1 or len(c) % 2 != 1 or len(c) < 3:
        raise ValueError("coeffs must hold 2K + 1 >= 3 values")
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mpo_stencil(ctx.h, int(n_sites), int(direction), (len(c) - 1) // 2,
                                      c.ctypes.data_as(C.POINTER(C.c_double)), C.byref(h)))
    return Mpo(ctx, h)


def qtt_mpo_laplacian(ctx: Context, n_sites: int, dx: float) -> Mpo:
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mpo_laplacian(ctx.h, n_sites, float(dx), C.byref(h)))
    return Mpo(ctx, h)


def qtt_apply_mpo(ctx: Context, w: Mpo, x: Mps) -> Mps:
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_apply_mpo(ctx.h, w.h, x.h, C.byref(h)))
    return Mps(ctx, h)


def qtt_hadamard(ctx: Context, a: Mps, b: Mps) -> Mps:
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_hadamard(ctx.h, a.h, b.h, C.byref(h)))
    return Mps(ctx, h)


def qtt_axpy(ctx: Context, alpha: float, x: Mps, y: Mps) -> None:
    ctx.check(ctx.lib.qtt_axpy(ctx.h, float(alpha), x.h, y.h))


def qtt_round(ctx: Context, x: Mps, chi_max: int, eps: float = 0.0) -> None:
    ctx.check(ctx.lib.qtt_round(ctx.h, x.h, int(chi_max), float(eps)))


def qtt_round_ex(ctx: Context, x: Mps, chi_max: int, eps: float = 0.0, chi_work: int = 0) -> None:
    ctx.check(ctx.lib.qtt_round_ex(ctx.h, x.h, int(chi_max), float(eps), int(chi_work)))


def qtt_mps_core_ptr(ctx: Context, x: Mps, k: int) -> int:
    """Device address of core k of a handle with explicit cores (no copy)."""
    p = C.c_void_p()
    ctx.check(ctx.lib.qtt_mps_core_ptr(ctx.h, x.h, int(k), C.byref(p)))
    return int(p.value)


def qtt_round_batch(ctx: Context, xs: Sequence[Mps], chi_max: int, eps: float = 0.0) -> None:
    arr = (C.c_void_p * len(xs))(*[x.h for x in xs])
    ctx.check(ctx.lib.qtt_round_batch(ctx.h, len(xs), arr, int(chi_max), float(eps)))


def qtt_rk4_step(ctx: Context, u: Sequence[Mps], Dx: Mpo, Dy: Mpo, Lap: Mpo, Re: float, dt: float, chi_max: int,
                 eps: float = 0.0) -> None:
    arr = (C.c_void_p * 2)(u[0].h, u[1].h)
    ctx.check(ctx.lib.qtt_rk4_step(ctx.h, arr, Dx.h, Dy.h, Lap.h, float(Re), float(dt), int(chi_max), float(eps)))


def qtt_rk4_step3(ctx: Context, u: Sequence[Mps], D: Sequence[Mpo], Lap: Mpo, Re: float, dt: float, chi_max: int,
                  eps: float = 0.0) -> None:
    """One RK4 step of the three-component Burgers equations in a context of physical dimension 8 (in place)."""
    if len(u) != 3 or len(D) != 3:
        raise ValueError("three components and three derivative MPOs")
    ua = (C.c_void_p * 3)(u[0].h, u[1].h, u[2].h)
    da = (C.c_void_p * 3)(D[0].h, D[1].h, D[2].h)
    ctx.check(ctx.lib.qtt_rk4_step3(ctx.h, ua, da, Lap.h, float(Re), float(dt), int(chi_max), float(eps)))


def qtt_variational_cost(ctx: Context, v: Sequence[Mps], a: Sequence[Mps], B: Sequence[Mps], D1: Mpo, D2: Mpo, h: float,
                         mu: float) -> float:
    """Theta of PAPER.md Eq. B6."""
    out = C.c_double()
    pair = lambda x: (C.c_void_p * 2)(x[0].h, x[1].h)
    ctx.check(ctx.lib.qtt_variational_cost(ctx.h, pair(v), pair(a), pair(B), D1.h, D2.h, float(h), float(mu), C.byref(out)))
    return out.value


def qtt_variational_stage(ctx: Context, v: Sequence[Mps], a: Sequence[Mps], B: Sequence[Mps], D1: Mpo, D2: Mpo, h: float,
                          mu: float, max_sweeps: int = 20, sweep_tol: float = 1e-5, cg_maxit: int = 100,
                          cg_tol: float = 1e-5) -> dict:
    """One stage of the paper's variational solver (Sec. II.C, App. B); v is updated in place.  Returns the
    counters the library reports: sweeps, CG iterations in total, most CG iterations of one local solve."""
    sw, mx, tot = C.c_int(), C.c_int(), C.c_longlong()
    pair = lambda x: (C.c_void_p * 2)(x[0].h, x[1].h)
    ctx.check(ctx.lib.qtt_variational_stage(ctx.h, pair(v), pair(a), pair(B), D1.h, D2.h, float(h), float(mu), int(max_sweeps),
                                            float(sweep_tol), int(cg_maxit), float(cg_tol), C.byref(sw), C.byref(tot),
                                            C.byref(mx)))
    return {"sweeps": sw.value, "cg_iterations": tot.value, "cg_max": mx.value}


# ------------------------------------------------------------------ inspection
def qtt_mps_bonds(x: Mps) -> list[int]:
    n = x.ctx.lib.qtt_mps_num_sites(x.h)
    b = (C.c_int * (n + 1))()
    x.ctx.check(x.ctx.lib.qtt_mps_bonds(x.h, b))
    return list(b)


def _host_array(shape, pinned: bool) -> np.ndarray:
    """A float64 host array; pinned=True backs it with page-locked memory (torch owns it, the array is a view)."""
    if not pinned:
        return np.empty(shape, dtype=np.float64)
    return torch.empty(shape, dtype=torch.float64, pin_memory=True).numpy()


def qtt_mps_get_core(ctx: Context, x: Mps, k: int, pinned: bool = False) -> np.ndarray:
    r = qtt_mps_bonds(x)
    out = _host_array((r[k], qtt_ctx_phys_dim(ctx), r[k + 1]), pinned)
    ctx.check(ctx.lib.qtt_mps_get_core(ctx.h, x.h, k, out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


def qtt_mps_get_cores(ctx: Context, x: Mps, pinned: bool = False) -> list[np.ndarray]:
    return [qtt_mps_get_core(ctx, x, k, pinned) for k in range(ctx.lib.qtt_mps_num_sites(x.h))]


def qtt_mps_dot(ctx: Context, a: Mps, b: Mps) -> float:
    v = C.c_double()
    ctx.check(ctx.lib.qtt_mps_dot(ctx.h, a.h, b.h, C.byref(v)))
    return v.value


def qtt_mps_norm(ctx: Context, x: Mps) -> float:
    v = C.c_double()
    ctx.check(ctx.lib.qtt_mps_norm(ctx.h, x.h, C.byref(v)))
    return v.value


def qtt_mps_schmidt(ctx: Context, x: Mps) -> list:
    """Schmidt values per bond (index 1..n-1; entries 0 and n are None)."""
    r = qtt_mps_bonds(x)
    n = len(r) - 1
    cap = max(max(r), 1) * qtt_ctx_phys_dim(ctx)
    buf = np.zeros((n + 1, cap), dtype=np.float64)
    counts = (C.c_int * (n + 1))()
    ctx.check(ctx.lib.qtt_mps_schmidt(ctx.h, x.h, buf.ctypes.data_as(C.POINTER(C.c_double)), cap, counts))
    return [None] + [buf[k, : counts[k]].copy() for k in range(1, n)] + [None]


def qtt_mps_fidelity(ctx: Context, a: Mps, b: Mps) -> float:
    v = C.c_double()
    ctx.check(ctx.lib.qtt_mps_fidelity(ctx.h, a.h, b.h, C.byref(v)))
    return v.value


def qtt_mps_chi_eps(ctx: Context, x: Mps, eps: float) -> tuple[list[int], int]:
    """(chi_l for l = 0..n, max_l chi_l) of PAPER.md Eq. 16-17."""
    n = len(qtt_mps_bonds(x)) - 1
    out = (C.c_int * (n + 1))()
    mx = C.c_int()
    ctx.check(ctx.lib.qtt_mps_chi_eps(ctx.h, x.h, float(eps), out, C.byref(mx)))
    return list(out), mx.value


def qtt_tke_spectrum(ctx: Context, u1: Mps, u2: Mps, mean1: "Mps | None" = None, mean2: "Mps | None" = None) -> np.ndarray:
    """E(kappa) of PAPER.md Eq. 13-15 for shells kappa = 0 .. floor(N / sqrt(2) + 1/2)."""
    n = ctx.lib.qtt_mps_num_sites(u1.h)
    nbins = int(np.floor(np.sqrt(2.0) * (1 << n) / 2 + 0.5)) + 1
    out = np.zeros(nbins, dtype=np.float64)
    ctx.check(ctx.lib.qtt_tke_spectrum(ctx.h, u1.h, u2.h, mean1.h if mean1 is not None else None,
                                       mean2.h if mean2 is not None else None, nbins,
                                       out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


def qtt_mps_clone(ctx: Context, x: Mps) -> Mps:
    h = C.c_void_p()
    ctx.check(ctx.lib.qtt_mps_clone(ctx.h, x.h, C.byref(h)))
    return Mps(ctx, h)


def qtt_ctx_set_chi_work(ctx: Context, chi_work: int) -> None:
    ctx.check(ctx.lib.qtt_ctx_set_chi_work(ctx.h, int(chi_work)))


def qtt_ctx_set_phys_dim(ctx: Context, d: int) -> None:
    """4: 2D quantics encoding (default); 8: 3D (include/qtt.h).  Only while no MPS / MPO handle of the context is alive."""
    ctx.check(ctx.lib.qtt_ctx_set_phys_dim(ctx.h, int(d)))


def qtt_ctx_phys_dim(ctx: Context) -> int:
    return int(ctx.lib.qtt_ctx_phys_dim(ctx.h))


def qtt_ctx_set_convection(ctx: Context, skew_symmetric: bool) -> None:
    ctx.check(ctx.lib.qtt_ctx_set_convection(ctx.h, 1 if skew_symmetric else 0))


def qtt_ctx_set_product_compression(ctx: Context, sketch: bool, seed: int = 0) -> None:
    """False: truncated SVD in the zip-up (default); True: randomised range finder with sign probes (reading 25)."""
    ctx.check(ctx.lib.qtt_ctx_set_product_compression(ctx.h, 1 if sketch else 0, int(seed)))


def qtt_ctx_set_graphs(ctx: Context, enabled: bool) -> None:
    ctx.check(ctx.lib.qtt_ctx_set_graphs(ctx.h, 1 if enabled else 0))


def qtt_ctx_set_materialize_limit(ctx: Context, nbytes: int) -> None:
    ctx.check(ctx.lib.qtt_ctx_set_materialize_limit(ctx.h, int(nbytes)))


def qtt_ctx_jacobi_stats(ctx: Context) -> tuple[int, int]:
    a, b = C.c_int(), C.c_int()
    ctx.check(ctx.lib.qtt_ctx_jacobi_stats(ctx.h, C.byref(a), C.byref(b)))
    return a.value, b.value


def qtt_ctx_launch_count(ctx: Context) -> int:
    return int(ctx.lib.qtt_ctx_launch_count(ctx.h))


PROF_FAMILIES = ("gemm", "lq_panel", "lq_update", "rowjacobi", "select", "move", "qrcp")


def qtt_ctx_profile(ctx: Context, enabled: bool) -> None:
    ctx.check(ctx.lib.qtt_ctx_profile(ctx.h, 1 if enabled else 0))


def qtt_ctx_profile_report(ctx: Context) -> dict:
    """{family: {"ms": kernel milliseconds, "work": flops or bytes, "launches": count}} since the last report."""
    n = len(PROF_FAMILIES)
    ms, work, cnt = (C.c_double * n)(), (C.c_double * n)(), (C.c_longlong * n)()
    ctx.check(ctx.lib.qtt_ctx_profile_report(ctx.h, ms, work, cnt))
    return {f: {"ms": ms[i], "work": work[i], "launches": int(cnt[i])} for i, f in enumerate(PROF_FAMILIES)}


LQ_NOALLOC_MAX_DOUBLES = 3 * 64 * 4096  # include/qtt_diag.h QTT_LQ_NOALLOC_MAX_DOUBLES


def qtt_lq_noalloc(Y: torch.Tensor, R: torch.Tensor, stream: "torch.cuda.Stream | None" = None) -> None:
    """include/qtt_diag.h qtt_lq_noalloc: Q-less LQ of the batch Y (batch x k x m, fp64, CUDA, contiguous; destroyed) into R
    (batch x k x k) without any device allocation by the library: its scratch is a 6 MiB device array built into the library
    (matrices too large for the cluster-resident kernel: batch * m <= 4096).  Calls that overlap on the GPU race on it."""
    if Y.dim() != 3 or R.dim() != 3 or not (Y.is_cuda and R.is_cuda and Y.is_contiguous() and R.is_contiguous()) \
            or Y.dtype != torch.float64 or R.dtype != torch.float64:
        raise ValueError("qtt_lq_noalloc wants contiguous fp64 CUDA tensors Y (batch, k, m) and R (batch, k, k)")
    batch, k, m = Y.shape
    if tuple(R.shape) != (batch, k, k):
        raise ValueError(f"R must be {(batch, k, k)}, got {tuple(R.shape)}")
    st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
    rc = _lib.load().qtt_lq_noalloc(C.c_void_p(st), C.c_void_p(Y.data_ptr()), batch, k, m, m, C.c_void_p(R.data_ptr()))
    if rc == -2:
        raise ValueError(f"qtt_lq_noalloc: batch {batch} x m {m} exceeds the built-in scratch ({LQ_NOALLOC_MAX_DOUBLES} doubles: "
                         f"batch * m <= 4096); use qtt_diag_lq with a caller-allocated buffer")
    if rc == -1:
        raise ValueError(f"qtt_lq_noalloc: invalid sizes (1 <= batch {batch} <= 16, 1 <= k {k} <= m {m} <= 16384)")
    if rc != 0:
        raise RuntimeError(f"qtt_lq_noalloc: CUDA error {rc}")
