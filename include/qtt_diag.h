/* qtt_diag.h -- kernel-level diagnostic entry points of libqtt_b200 (tests, profiling, peak probes).
 * Plain device pointers, no handles.  All return 0 on success or a cudaError_t value.  `stream` is a
 * cudaStream_t.  These run the SAME kernels the qtt_* calls of qtt.h are built from. */
#ifndef QTT_B200_DIAG_H
#define QTT_B200_DIAG_H
#ifdef __cplusplus
extern "C" {
#endif

/* C = alpha * op(A) * op(B) + beta * C, row-major, strided batch; op = transpose if trans* != 0.
 * A is M x K (lda) or, transposed, stored K x M (lda); B likewise; C is M x N (ldc).
 * SURVEY.md section 8 row a2 (site contractions on the fp64 tensor pipe). */
int qtt_diag_gemm(void* stream, const double* A_dev, const double* B_dev, double* C_dev, int M, int N, int K,
                  int transA, int transB, long long lda, long long ldb, long long ldc, double alpha, double beta,
                  int nbatch, long long strideA, long long strideB, long long strideC);

/* Q-less LQ of `batch` matrices Y_i (k x m, k <= m <= 16384, leading dimension ld, consecutive with stride
 * k*ld, DESTROYED unless small); R_i = L_i^T (k x k upper triangular, row-major, consecutive) with Y = L Q.
 * Matrices whose slices fit a cluster's shared memory go through the cluster-resident Householder kernel (and
 * are left alone), larger ones through the blocked panel + DMMA trailing-update path.
 * scratch_dev: batch * 3 * 64 * m doubles.  SURVEY.md section 8 row a4. */
int qtt_diag_lq(void* stream, double* Y_dev, int batch, int k, int m, int ld, double* R_dev, double* scratch_dev);

/* qtt_diag_lq for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same kernels and launch sequence, with the scratch of the blocked path in a device array
 * that is part of the library image (QTT_LQ_NOALLOC_MAX_DOUBLES doubles = 6 MiB, held by every GPU that loads the library
 * until the process exits).  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 * Arguments as qtt_diag_lq (device pointers, caller-owned: Y_dev destroyed unless small, R_dev <- batch k x k factors),
 * 1 <= batch <= 16, k <= m <= ld.  Limit: matrices too large for the cluster-resident kernel need batch * 3 * 64 * m doubles
 * of scratch, so batch * m <= 4096; beyond that the call launches nothing, prints the reason to stderr and returns
 * QTT_NOALLOC_TOO_LARGE (use qtt_diag_lq with your own buffer).  QTT_NOALLOC_BAD_ARG for NULL pointers or sizes out of
 * range; otherwise 0 or a cudaError_t value.  All calls share the one array (per device) and it keeps the previous call's
 * contents: the part a call uses is cleared on `stream` first, and calls that OVERLAP on the GPU (different streams without
 * a dependency between them) race on it -- keep them on one stream or order them with events.  SURVEY.md section 8 row a4. */
#define QTT_LQ_NOALLOC_MAX_DOUBLES 786432 /* 3 * 64 * 4096 */
#define QTT_NOALLOC_BAD_ARG (-1)
#define QTT_NOALLOC_TOO_LARGE (-2)
int qtt_lq_noalloc(void* stream, double* Y_dev, int batch, int k, int m, int ld, double* R_dev);

/* One-sided Jacobi on the rows of `batch` matrices X_i (p x q, ld, stride p*ld), in place: rows of the result
 * are mutually orthogonal (X = J^T Sigma V^T).  status_dev: 2 ints (zero them first): [0] <- max sweeps,
 * [1] += matrices that hit the sweep limit.  SURVEY.md section 8 row a5. */
int qtt_diag_rowjacobi(void* stream, double* X_dev, int batch, int p, int q, int ld, int* status_dev);

/* The same iteration for matrices too large for a cluster's shared memory (q <= 1024 columns, any p): L2-streamed
 * block Jacobi, one launch per tournament round over 16-row blocks, a static number of launches that return at once
 * after convergence.  work_dev: 8 doubles of scratch per matrix.  SURVEY.md section 8 row a6 (chi = 128). */
int qtt_diag_rowjacobi_streamed(void* stream, double* X_dev, int batch, int p, int q, int ld, int* status_dev,
                                double* work_dev);

/* The production SVD front end on `batch` matrices X_i (p x q, ld, stride p*ld), in place: rank-revealing
 * Householder QR with column pivoting X <- Q^T X (columns stay in place, rows from the numerical rank on are
 * exact zeros, rank_dev[i] <- rank), then -- unless status_dev is NULL -- one-sided Jacobi on the first
 * rank rows.  Right singular vectors and singular values of X are those of the result's rows.  Needs the
 * column slices to fit a cluster's shared memory (else cudaErrorInvalidConfiguration).  SURVEY.md section 8 row a5. */
int qtt_diag_svd_rows(void* stream, double* X_dev, int batch, int p, int q, int ld, int* rank_dev, int* status_dev);

/* Sort rows by norm, apply the rank rule (delta < 0: r = min(chi_max, p, q); else smallest r whose discarded
 * tail is <= delta, clamped to [1, chi_max]), write sigma (p), rank (1 int) and the normalised top rows
 * (r_cap x q) to out_dev. */
int qtt_diag_select(void* stream, const double* X_dev, int p, int q, int ld, double* out_dev, int r_cap,
                    double* sigma_dev, int* rank_dev, int chi_max, double delta);

/* fp64 issue-rate probes: kind 0 = register-only DMMA.8x8x4 loop, kind 1 = register-only DFMA loop, on
 * `ctas` CTAs of 256 threads, `iters` iterations of 64 independent instructions per warp / thread chain set.
 * *tflops_out <- achieved TFLOP/s (host pointer).  Synchronous. */
int qtt_diag_fp64_probe(void* stream, int kind, int ctas, int iters, double* tflops_out);

/* While qtt_ctx_profile (qtt.h) is enabled: synchronises the device and writes one CSV line per kernel launch
 * recorded since the last qtt_ctx_profile_report -- family, shape tag d0..d3, kernel milliseconds, algorithmic
 * work -- to the host path; the records are kept (the next report still sums them).  Shape tags:
 * gemm (M, N, K of the first problem, problems); lq_panel / lq_update (k, m, problems, first panel row);
 * rowjacobi (p, q, problems, CTAs per matrix); select (p, q, problems, 0); move (0). */
int qtt_diag_profile_dump(const char* path_host);

#ifdef __cplusplus
}
#endif
#endif
