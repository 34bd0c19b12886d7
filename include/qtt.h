/* qtt.h -- C ABI of the B200-native QTT/MPS time-step algebra (arxiv 2406.17823, Hoelscher et al.).
 *
 * The library implements the per-time-step matrix-product-state (MPS) algebra of the paper's
 * quantics-tensor-train Navier-Stokes solver on ONE GPU, in fp64, with hand-written sm_100a kernels.
 * Citations are to /root/reference/PAPER.md (line, section / equation); DESIGN.md lists the readings
 * taken where the paper is silent.
 *
 * Data model (Sec. II.B, Eq. 3-4).  A field F[x][y] on an N x N periodic grid,
 * N = 2^n, x_j = y_j = j/N, is an n-site MPS.  Site k = 1..n carries the physical index
 * w_k = 2*x_bit_k + y_bit_k (d = 4) with bit 1 the MOST significant.  A site tensor ("core") is a dense
 * row-major array  core_k[r_{k-1}][4][r_k]  of doubles in device memory, r_0 = r_n = 1.  An MPO is a list
 * of n arrays  W_k[D_{k-1}][4 (output w)][4 (input w')][D_k], D_0 = D_n = 1 (Eq. 7 with the
 * boundary vectors L, R folded into the end cores).
 *
 * Conventions.
 *  - Handles (qtt_ctx, qtt_mps, qtt_mpo) are opaque, created by the library and released by the caller
 *    with the matching *_free / *_destroy.  A handle belongs to the context that created it.
 *  - Device memory comes ONLY from the caller's alloc/release callbacks (the Python binding hands out
 *    torch-owned memory): one workspace of `workspace_bytes` at qtt_ctx_create and one block per MPS.
 *  - All work is enqueued on the caller's CUDA stream given at qtt_ctx_create.  With eps == 0 every call
 *    that takes only device data is asynchronous (static shapes: rank = min(chi_max, rows, cols));
 *    with eps > 0 the rank of each bond is read back, i.e. ONE stream synchronisation per bond.
 *  - `release` may be called while kernels that read the block are still queued on the context's stream (the library
 *    never synchronises to free): the callback must be STREAM-ORDERED with respect to that stream, i.e. the block may
 *    be reused only by work enqueued on the same stream afterwards (a stream-ordered pool such as torch's caching
 *    allocator used under that stream, or cudaFreeAsync on it).  `alloc` is called on the calling thread, never
 *    inside a graph capture.
 *  - Jacobi SVDs that hit their sweep limit are recorded on the device.  Calls that synchronise (qtt_mps_get_core,
 *    qtt_mps_dot, qtt_mps_norm, qtt_mps_schmidt, every call with eps > 0, qtt_ctx_jacobi_stats) return QTT_NUMERIC
 *    once per new record, so non-convergence of an earlier asynchronous call cannot go unnoticed.
 *  - Every function returns a qtt_status; on error outputs are untouched and qtt_last_error() gives text.
 *    There is NO CPU fallback: without a usable CUDA device qtt_ctx_create fails with QTT_CUDA.
 *  - "dev" pointers are device pointers, "host" pointers are host pointers.
 *  - Lazy results.  qtt_apply_mpo, qtt_hadamard and qtt_axpy return / produce handles that DENOTE the
 *    exact result (bond D*chi, chi_a*chi_b, chi_x+chi_y) and keep references to their operands; nothing
 *    is computed until qtt_round (fused sweeps; the chi^2 bond of a product is never formed),
 *    qtt_to_dense / qtt_mps_get_core (materialise, bounded by the materialisation limit ->
 *    QTT_CAPACITY) or qtt_mps_dot.
 *  - Gauge is not part of the contract.  qtt_round / qtt_mps_from_dense return right-canonical cores
 *    (norm on site 1); compare only gauge-invariant quantities (dense field, norms, Schmidt values).
 */
#ifndef QTT_B200_H
#define QTT_B200_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qtt_ctx qtt_ctx;
typedef struct qtt_mps qtt_mps;
typedef struct qtt_mpo qtt_mpo;
typedef int qtt_status;
#define QTT_OK 0
#define QTT_INVALID_ARG (-1)
#define QTT_SHAPE_MISMATCH (-2)
#define QTT_CAPACITY (-3) /* workspace / materialisation limit exceeded */
#define QTT_CUDA (-4)     /* CUDA error, text in qtt_last_error */
#define QTT_NUMERIC (-5)  /* Jacobi sweep limit hit */

typedef void* (*qtt_alloc_fn)(size_t bytes, void* user); /* returns a device pointer, 256-byte aligned, or NULL */
typedef void (*qtt_release_fn)(void* dev_ptr, void* user);

/* Create a context on CUDA device `device`, enqueueing on `cuda_stream` (a cudaStream_t; NULL = legacy
 * default stream).  `workspace_bytes` of scratch are taken once through `alloc`. */
qtt_status qtt_ctx_create(qtt_ctx** out, int device, void* cuda_stream, qtt_alloc_fn alloc, qtt_release_fn release,
                          void* user, size_t workspace_bytes);
void qtt_ctx_destroy(qtt_ctx* ctx);
const char* qtt_last_error(const qtt_ctx* ctx);
/* Working bond chi_work of the fused Hadamard+round ("zip-up", reading 8); 0 = 2*chi_max. */
qtt_status qtt_ctx_set_chi_work(qtt_ctx* ctx, int chi_work);
/* SURVEY.md section 8f next-4, "3D (d = 8) encoding" ("the methods outlined here can be generalized to 3D",
 * PAPER.md:320-322; reading 26).  Physical dimension of every site of this context's MPS / MPO handles: 4
 * (default) = the 2D quantics encoding of PAPER.md Eq. 3, w_k = 2 x_k + y_k; 8 = a 2^n x 2^n x 2^n grid with
 * w_k = 4 x_k + 2 y_k + z_k (the bits of one length scale share a site, bit 1 most significant).  With d = 8:
 * qtt_mps_from_dense / qtt_to_dense take dense_dev[(x*N + y)*N + z] (n_bits <= 9), cores are r x 8 x r', MPO cores
 * D x 8 x 8 x D', the MPO builders accept direction 1, 2, 3 (x, y, z) and qtt_mpo_laplacian is the 7-point stencil of
 * bond 7; qtt_apply_mpo, qtt_hadamard, qtt_axpy, qtt_round / qtt_round_batch / qtt_round_ex (zip-up included), qtt_mps_dot /
 * norm / schmidt / fidelity / chi_eps / clone / get_core run the same kernels on d r-row unfoldings.  qtt_rk4_step,
 * qtt_variational_*, qtt_tke_spectrum and the sketched product compression are built for two velocity components on a 2D
 * grid and return QTT_INVALID_ARG when d = 8 (the 3D time step is qtt_rk4_step3).
 * Errors: QTT_INVALID_ARG for d outside {4, 8}, or for a switch while MPS / MPO handles of the context are alive. */
qtt_status qtt_ctx_set_phys_dim(qtt_ctx* ctx, int d);
int qtt_ctx_phys_dim(const qtt_ctx* ctx); /* 4 or 8; 0 for a NULL context */
/* Largest lazy result (bytes of all cores) that qtt_to_dense / qtt_mps_get_core may materialise. */
qtt_status qtt_ctx_set_materialize_limit(qtt_ctx* ctx, size_t bytes);
/* 1: qtt_rk4_step with eps == 0 is captured once into a CUDA graph per shape signature and replayed
 * (default); 0: launches are issued eagerly every step. */
qtt_status qtt_ctx_set_graphs(qtt_ctx* ctx, int enabled);
/* Convection form of qtt_rk4_step.  0 (default): convective, u_j (.) D_j u_i (BASELINE config 2; reading 4).
 * 1: the paper's skew-symmetric form, PAPER.md:432-435 Eq. B2, 1/2 (u_j (.) D_j u_i + D_j (u_j (.) u_i)): per
 * right-hand side three more products (u_1 u_1, u_1 u_2, u_2 u_2), four more applies and 5-term sums. */
qtt_status qtt_ctx_set_convection(qtt_ctx* ctx, int skew_symmetric);
/* SURVEY.md section 8f next-4, "a cheaper product compression" (the repeated SVDs are what the paper wants
 * replaced; reading 25).  mode 0 (default): every truncating step of the zip-up (qtt_round of a product handle,
 * the products inside qtt_rk4_step) keeps the chi_work largest left singular vectors of T_l (4 r_l x a_{l+1} b_{l+1}).
 * mode 1: at the sites where chi_work < min(4 r_l, a_{l+1} b_{l+1}) and c = 4^(n-1-l) satisfies c >= 2 chi_work or
 * c <= chi_work, it keeps an orthonormal basis Q of range(T_l S_{l+1}) instead.  The probes are a random tensor train over
 * the PHYSICAL indices with bond P = chi_work and sign cores G_k[w][u][t] = +-1/sqrt(P), (seed, site k, row w P + u,
 * column t) -> sign by the counter-based generator the oracle implements too (oracle sketch_signs, sketch_mixers);
 * S_{l+1} (a_{l+1} b_{l+1} x P) is that train contracted through the product's own cores from the last site down to l+1
 * (oracle sketch_probes): a function of the state, not of the gauge of its bonds.  Q spans the numerical range only
 * (singular values of the sketch above 8 eps ||.||_F; the other columns are zero).  Cost per site: three DMMA GEMMs for
 * S_l, one for the sketch, and the SVD step of a chi_work x 4 r_l matrix -- instead of the LQ of T_l and the SVD of its
 * 4 r_l x 4 r_l factor.  The result is the projection of T_l on a random chi_work-dimensional subspace of the range of
 * the true unfolding, not the truncated SVD of T_l: error <= ~sqrt(2) x the optimal rank-chi_work/2 tail in expectation
 * (Halko-Martinsson-Tropp), nothing lost where c <= chi_work or rank(T_l) <= chi_work.  seed is any 64-bit value.  Takes
 * effect at the next call; graphs are re-captured.  Errors: QTT_INVALID_ARG for a NULL ctx or mode outside {0, 1}. */
qtt_status qtt_ctx_set_product_compression(qtt_ctx* ctx, int mode, unsigned long long seed);
/* Synchronises the stream and reports the Jacobi convergence record since the last call:
 * the largest number of sweeps any SVD used, and how many SVDs hit the sweep limit (then QTT_NUMERIC). */
qtt_status qtt_ctx_jacobi_stats(qtt_ctx* ctx, int* max_sweeps, int* limit_hits);
/* Per-kernel-family device timing for bench.py's roofline.  While enabled, every kernel launch is bracketed
 * by a CUDA event pair on the stream and qtt_rk4_step runs eagerly (no graph replay).  qtt_ctx_profile_report
 * synchronises, then writes, for the QTT_PROF_FAMILIES families
 *   0 gemm (DMMA site contractions)  1 lq_panel  2 lq_update  3 rowjacobi  4 select  5 data movement
 *   6 qrcp (pivoted-QR preconditioner of the Jacobi SVD),
 * the summed kernel milliseconds, the summed algorithmic work (flops for 0-3 and 6, bytes for 4-5; the per-launch
 * formulas are stated in DESIGN.md) and the number of launches since the last report (host arrays). */
#define QTT_PROF_FAMILIES 7
qtt_status qtt_ctx_profile(qtt_ctx* ctx, int enabled);
qtt_status qtt_ctx_profile_report(qtt_ctx* ctx, double* ms_host, double* work_host, long long* launches_host);
/* Number of kernels launched (or graph nodes replayed) by this context so far (per context). */
long long qtt_ctx_launch_count(const qtt_ctx* ctx);

/* PAPER.md:67-72 Eq. 4 (reading 9): right-to-left TT-SVD of the dense field dense_dev[x*N + y], N = 2^n_bits,
 * keeping per bond r = rank rule(chi_max, eps) (see qtt_round).  (Physical dimension 8: dense_dev[(x*N + y)*N + z].) */
qtt_status qtt_mps_from_dense(qtt_ctx* ctx, const double* dense_dev, int n_bits, int chi_max, double eps,
                              qtt_mps** out);
/* Upload explicit cores (host arrays, core k is bonds[k] x d x bonds[k+1] row-major, d = qtt_ctx_phys_dim, bonds has
 * n+1 entries). */
qtt_status qtt_mps_from_cores(qtt_ctx* ctx, int n_sites, const int* bonds, const double* const* cores_host,
                              qtt_mps** out);
/* PAPER.md:69 Eq. 4: contract the MPS and undo the bit interleave; dense_dev_out holds N*N doubles (N*N*N for d = 8). */
qtt_status qtt_to_dense(qtt_ctx* ctx, const qtt_mps* x, double* dense_dev_out);

/* MPO from host cores W_k[D_{k-1}][d out][d in][D_k], d = qtt_ctx_phys_dim (Eq. 7, App. A Table II); bonds
 * has n+1 entries with both ends 1. */
qtt_status qtt_mpo_create(qtt_ctx* ctx, int n_sites, const int* bonds, const double* const* cores_host,
                          qtt_mpo** out);
/* PAPER.md:391-424 App. A (Eq. A1-A3, Table II): the periodic central-difference MPO
 * (F[i+1] - F[i-1]) / (2 dx) along direction 1 (x) or 2 (y) (or 3 (z) when d = 8), bond 3, boundary vectors L = (1,1,1) on the
 * most-significant site and R = (0, 1, -1)/(2 dx) on the least-significant site folded into the end cores.
 * Index convention: w = output, w' = contracted with the MPS (reading 1).  n_sites >= 2. */
qtt_status qtt_mpo_central_difference(qtt_ctx* ctx, int n_sites, int direction, double dx, qtt_mpo** out);
/* Compact periodic 5-point Laplacian MPO, bond 5 (reading 3): channels identity, x+1, x-1, y+1, y-1;
 * L = (1,1,1,1,1), R = (-4,1,1,1,1)/dx^2.  With d = 8: the 7-point Laplacian, bond 7, channels identity, x+-1, y+-1, z+-1,
 * R = (-6,1,1,1,1,1,1)/dx^2.  n_sites >= 2. */
qtt_status qtt_mpo_laplacian(qtt_ctx* ctx, int n_sites, double dx, qtt_mpo** out);
/* PAPER.md:98 ("MPOs for finite-difference stencils of any order"), construction of App. A generalised: the periodic
 * stencil (O F)[x] = sum_{k=-K..K} coeffs_host[k + K] * F[x + k] along direction 1 (x) or 2 (y) (or 3 (z) when d = 8), K = half_width in
 * 1..16, as an MPO of bond 2K + 1 (bond index = carry of the addition x + k + K).  n_sites >= 2. */
qtt_status qtt_mpo_stencil(qtt_ctx* ctx, int n_sites, int direction, int half_width, const double* coeffs_host,
                           qtt_mpo** out);
void qtt_mpo_free(qtt_mpo* w);

/* y = W x, exact, bond D*chi, composite bond index = alpha*chi + a (lazy). */
qtt_status qtt_apply_mpo(qtt_ctx* ctx, const qtt_mpo* w, const qtt_mps* x, qtt_mps** y);
/* PAPER.md:100-105 Eq. 8: c = a (.) b element-wise, exact, bond chi_a*chi_b (lazy, never formed by qtt_round). */
qtt_status qtt_hadamard(qtt_ctx* ctx, const qtt_mps* a, const qtt_mps* b, qtt_mps** c);
/* PAPER.md:126-130 Eq. 11: y <- alpha*x + y, exact, direct sum of the bonds (lazy; sums nest flat). */
qtt_status qtt_axpy(qtt_ctx* ctx, double alpha, const qtt_mps* x, qtt_mps* y);
/* PAPER.md:130 ("compression ... repeated SVDs"), ref. [15]; eps semantics PAPER.md:238 Eq. 16.
 * Left-to-right orthogonalisation, then right-to-left truncated SVD, in place on the handle.
 * Rank rule per bond: eps == 0: r' = min(chi_max, rows, cols) of the unfolding (static shapes);
 * eps > 0: smallest r with sqrt(sum_{i>r} sigma_i^2) <= eps*||x||_F/sqrt(n-1), clamped to [1, chi_max].
 * A product handle is rounded by the zip-up (reading 8) with working bond chi_work. */
qtt_status qtt_round(qtt_ctx* ctx, qtt_mps* x, int chi_max, double eps);
/* The same with the working bond of the zip-up given per call; chi_work == 0: the context's
 * setting (qtt_ctx_set_chi_work), else 2*chi_max.  Ignored for handles that are not products. */
qtt_status qtt_round_ex(qtt_ctx* ctx, qtt_mps* x, int chi_max, double eps, int chi_work);
/* The same for `batch` independent operands in single launches per site. */
qtt_status qtt_round_batch(qtt_ctx* ctx, int batch, qtt_mps* const* xs, int chi_max, double eps);
/* PAPER.md:124-128 Eq. 11 on u = (u_1, u_2), in place: classical RK4 of
 * f_i = -(u_1 (.) D_1 u_i + u_2 (.) D_2 u_i) + (1/Re) Lap u_i   (Eq. 2 without pressure),
 * one rounding after every apply, product and sum (readings 4, 5, 7, 10). */
qtt_status qtt_rk4_step(qtt_ctx* ctx, qtt_mps* const u[2], const qtt_mpo* Dx, const qtt_mpo* Dy, const qtt_mpo* Lap,
                        double Re, double dt, int chi_max, double eps);
/* The same step for three velocity components on a 3D grid (reading 26; needs
 * qtt_ctx_set_phys_dim(ctx, 8)): u = (u_1, u_2, u_3) in place, D = (D_x, D_y, D_z),
 * f_i = -sum_{j=1..3} u_j (.) D_j u_i + (1/Re) Lap u_i, roundings as above: per right-hand side one batch of 12 apply + round,
 * one of 9 zip-ups, one of 3 four-term sums; stage and final combinations as in qtt_rk4_step.  Launches are issued eagerly
 * (no CUDA graph); eps > 0 synchronises once per bond.  Errors: QTT_INVALID_ARG for NULL arguments, a context of physical
 * dimension 4, or the sketched product compression; QTT_SHAPE_MISMATCH for operands of different length or n < 2. */
qtt_status qtt_rk4_step3(qtt_ctx* ctx, qtt_mps* const u[3], const qtt_mpo* const D[3], const qtt_mpo* Lap, double Re, double dt,
                         int chi_max, double eps);

/* Inspection. */
int qtt_mps_num_sites(const qtt_mps* x);
qtt_status qtt_mps_bonds(const qtt_mps* x, int* bonds_out /* n+1 */);
/* Device pointer to core k (0-based, bonds[k] x 4 x bonds[k+1] doubles, row-major) of a handle with EXPLICIT cores
 * (from qtt_mps_from_dense / qtt_mps_from_cores / qtt_round / qtt_rk4_step / qtt_mps_clone); a lazy handle gives
 * QTT_INVALID_ARG.  The memory is owned by the handle and valid until it is freed, rounded or stepped; reads must be
 * ordered after the context's stream.  No copy, no synchronisation. */
qtt_status qtt_mps_core_ptr(qtt_ctx* ctx, const qtt_mps* x, int k, const double** core_dev_out);
/* Copy core k (0-based) to host_out (bonds[k]*4*bonds[k+1] doubles); materialises lazy handles. Synchronous. */
qtt_status qtt_mps_get_core(qtt_ctx* ctx, const qtt_mps* x, int k, double* host_out);
/* <a|b> by transfer matrices; result written to *out_host after a stream synchronisation. */
qtt_status qtt_mps_dot(qtt_ctx* ctx, const qtt_mps* a, const qtt_mps* b, double* out_host);
/* ||x||_F from an orthogonalisation sweep (no cancellation); synchronous. */
qtt_status qtt_mps_norm(qtt_ctx* ctx, const qtt_mps* x, double* out_host);
/* Schmidt values of every bond 1..n-1 (Eq. 16-17): sigma_host[bond*cap + i], counts[bond];
 * entries beyond counts[bond] are untouched.  Synchronous. */
qtt_status qtt_mps_schmidt(qtt_ctx* ctx, const qtt_mps* x, double* sigma_host, int cap, int* counts /* n+1 */);
/* PAPER.md:160 Eq. 12: fidelity F = <a|b>^2 / (||a||^2 ||b||^2) by MPS overlaps (qtt_mps_dot, qtt_mps_norm).
 * Synchronous; 0 if either operand is zero. */
qtt_status qtt_mps_fidelity(qtt_ctx* ctx, const qtt_mps* a, const qtt_mps* b, double* out_host);
/* PAPER.md:238-244 Eq. 16-17: chi_l(eps), the number of Schmidt values bipartition l = 1..n-1 needs for a relative
 * truncation error sqrt(sum_{i > chi_l} sigma_i^2) / ||x|| <= eps, written to chi_host[l] (n+1 ints, ends = 1), and
 * chi = max_l chi_l to *chi_max_host (may be NULL).  Synchronous. */
qtt_status qtt_mps_chi_eps(qtt_ctx* ctx, const qtt_mps* x, double eps, int* chi_host, int* chi_max_host);
/* ---- The variational stage of the paper's own solver (Sec. II.C, App. B).
 * Theta(v) = mu ||D1 v_1 + D2 v_2||^2 + sum_i ||(v_i - a_i) / h + B_i||^2   (PAPER.md:452 Eq. B6; mu: the
 * incompressibility penalty; a: the state the stage starts from, h: the stage's time increment, B: the
 * nonlinear part Eq. B21 given as an MPS pair, e.g. minus the right-hand side formed by the hot-path primitives),
 * evaluated with exact MPS sums; the three norms come from an orthogonalisation sweep, not from overlaps (with v close to
 * a the residual is a difference of terms 1/h times larger than itself, which <s|s> by transfer matrices cannot resolve).
 * Handles of any kind; *theta_host is written after a synchronisation. */
qtt_status qtt_variational_cost(qtt_ctx* ctx, const qtt_mps* const v[2], const qtt_mps* const a[2], const qtt_mps* const B[2],
                                const qtt_mpo* D1, const qtt_mpo* D2, double h, double mu, double* theta_host);
/* Minimises Theta over the MPS pair v (in-out; its bonds are kept, or shrink where a bond exceeds what its neighbours
 * allow) by one-site sweeps, site 1 -> n -> 1 per sweep: at the canonical centre the stationarity condition
 * Eq. B22 is the symmetric positive definite system Eq. B23-B24, C_i - mu h^2 sum_j <basis_i|D_i D_j|basis_j> C_j =
 * <basis_i|a_i - h B_i>, solved by conjugate gradients from the current centre tensors until ||r|| <= cg_tol ||rhs|| or
 * cg_maxit iterations (the paper: 1e-5, 100); the iteration stops when sum_i <v_i|v_i> changes by less than sweep_tol
 * (relative) between sweeps, or after max_sweeps.  D1, D2 must be antisymmetric first-derivative MPOs.
 * Environments and the local operator are DMMA GEMMs; the CG loop is driven from the host (synchronous call, two scalar
 * read-backs per iteration; not captured into a graph).  Host outputs (each may be NULL): sweeps done, CG iterations in
 * total, most CG iterations of one local solve.  On error v is untouched. */
qtt_status qtt_variational_stage(qtt_ctx* ctx, qtt_mps* const v[2], const qtt_mps* const a[2], const qtt_mps* const B[2],
                                 const qtt_mpo* D1, const qtt_mpo* D2, double h, double mu, int max_sweeps, double sweep_tol,
                                 int cg_maxit, double cg_tol, int* sweeps_host, long long* cg_iterations_host,
                                 int* cg_max_host);
/* PAPER.md:173-184 Eq. 13-15: turbulent-kinetic-energy spectrum.  With u_i' = u_i - mean_i (mean_i == NULL: zero mean; Eq. 14)
 * and the Fourier coefficients u_i'^(k) = (1/N^2) sum_x u_i'(x) exp(-2 pi i k.x), k in [-N/2, N/2)^2 (Eq. 13):
 *   E_host[b] = 1/2 sum over the shell round(|k|) = b of (|u_1'^(k)|^2 + |u_2'^(k)|^2),  b = 0 .. nbins-1  (Eq. 15),
 * so that sum_b E[b] = 1/2 mean(u_1'^2 + u_2'^2) (Parseval).  nbins >= floor(N / sqrt(2) + 1/2) + 1.  A diagnostic on
 * dense fields (qtt_to_dense + an FFT kernel); needs ~10 N^2 doubles of workspace.  Synchronous. */
qtt_status qtt_tke_spectrum(qtt_ctx* ctx, const qtt_mps* u1, const qtt_mps* u2, const qtt_mps* mean1, const qtt_mps* mean2,
                            int nbins, double* E_host);
qtt_status qtt_mps_clone(qtt_ctx* ctx, const qtt_mps* x, qtt_mps** out);
void qtt_mps_free(qtt_mps* x);

#ifdef __cplusplus
}
#endif
#endif
