// Shared declarations of the sm_100a kernels behind the qtt_* C ABI (include/qtt.h).
// Problem descriptors are passed BY VALUE as __grid_constant__ kernel parameters so that a whole
// RK4 step can be stream-captured into one CUDA graph (no descriptor upload, no host sync).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef long long i64;

#define QTT_CHECK_CUDA(expr)                                                     \
  do {                                                                           \
    cudaError_t _e = (expr);                                                     \
    if (_e != cudaSuccess) return _e;                                            \
  } while (0)

// ----------------------------------------------------------------------------------------------
// Grouped fp64 GEMM on the DMMA pipe:  C = alpha * A * B + beta * C  for a list of problems.
// Every operand is addressed through element strides, so reshapes / permutes / transposes of the
// site tensors are folded into the tile loads (no transpose kernel).  One of each operand's two
// strides must be 1 (the contiguous direction is what cp.async moves in 16-byte pieces).
//   A(m,k)  at A + (m / a_div) * a_hi + (m % a_div) * a_lo + k * a_k + z * a_bs     (a_div = 0: m * a_lo)
//   B(k,n)  at B + k * b_k + n * b_n + z * b_bs
//   C(m,n)  at C + (m / c_div) * c_hi + (m % c_div) * c_lo + n * c_n + z * c_bs     (c_div = 0: m * c_lo)
// z = 0..nbatch-1 is an inner strided batch.
struct GemmProb {
  const double* A;
  const double* B;
  double* C;
  int M, N, K, nbatch;
  i64 a_lo, a_hi, a_k, a_bs;
  i64 b_k, b_n, b_bs;
  i64 c_lo, c_hi, c_n, c_bs;
  int a_div, c_div;
  double alpha, beta;
  int tile0, tiles_m, tiles_n, flags;  // filled by the launcher
};
#define QTT_GEMM_MAX_GROUP 20
struct GemmGroup {
  int nprob;
  int total_tiles;
  GemmProb p[QTT_GEMM_MAX_GROUP];
};
// Launch as many kernels as needed for `n` problems (any n).  Returns cudaSuccess or the error.
// `family`: profiler family the launches are booked under (QK_GEMM unless the GEMM is a step of another family).
cudaError_t qtt_launch_gemm(const GemmProb* probs, int n, cudaStream_t stream, int family = 0);

// ----------------------------------------------------------------------------------------------
// Batched Q-less LQ (blocked Householder by rows).  Y is k x m (k <= m), rows contiguous with
// leading dimension ld, destroyed.  On exit the lower triangle of Y[:, 0:k] holds L with
// Y_in = L * Q for an orthonormal-row Q that is never formed.
struct LqProb {
  double* Y;
  int k, m, ld;
  double* V;   // scratch  64 x m : clean reflector rows of the current super-panel (4 sub-panels of 16 rows)
  double* TV;  // scratch  64 x m : T_agg * V_agg of the current super-panel
  double* W;   // scratch  64 x m : products X V^T of the trailing updates and their K-chunk partials
};
#define QTT_LQ_MAX_BATCH 16
#define QTT_LQ_NB 16
struct LqGroup {
  int nprob;
  int p0;  // first row of the current panel
  LqProb p[QTT_LQ_MAX_BATCH];
};
cudaError_t qtt_launch_lq(const LqProb* probs, int n, cudaStream_t stream);
size_t qtt_lq_scratch_doubles(int m);  // per problem, for each of V, TV and W

// Copy the triangular factor out of a factored Y:  mode 0: R = L^T (k x k upper, row-major, ld = ldr),
// mode 1: L itself (k x k lower) into dst with leading dimension ldr.
struct TriProb { const double* Y; int k, ld; double* dst; int ldr; };
struct TriGroup { int nprob; int mode; TriProb p[QTT_LQ_MAX_BATCH]; };
cudaError_t qtt_launch_extract_tri(const TriProb* probs, int n, int mode, cudaStream_t stream);

// ----------------------------------------------------------------------------------------------
// Batched one-sided Jacobi: rotates the ROWS of X (p x q, rows contiguous, leading dimension ld)
// in place until they are mutually orthogonal:  X <- J X,  J orthogonal, so X = Sigma V^T up to a
// row permutation.  Column-sliced over a thread-block cluster; slices live in (distributed) shared
// memory when they fit, else the kernel works on global memory (L2).
struct JacProb {
  double* X;
  int p, q, ld;
  const int* p_dev;  // if non-null: number of rows to rotate (<= p), read on the device (numerical rank from qrcp)
  double* work;      // 8 doubles of device scratch (any content) for the L2-streamed path, or null
  int sweep_cap;     // 0: the kernel's default sweep limit; else the limit for this problem (L2-streamed path: the launch
                     // count is static, so the limit is kept as tight as the kind of input allows)
  int* status;  // device ints, may be shared by all problems: [0] <- max(sweeps used), [1] += 1 if the sweep limit was hit
};
#define QTT_JAC_MAX_BATCH 16
struct JacGroup {
  int nprob;
  int cluster;    // CTAs per matrix
  int use_smem;   // slice resident in shared memory
  int wslice;     // columns per CTA (multiple of 4)
  int max_sweeps;
  JacProb p[QTT_JAC_MAX_BATCH];
};
cudaError_t qtt_launch_rowjacobi(const JacProb* probs, int n, cudaStream_t stream);
// Register-blocked cluster block Jacobi (bj2.cu): p <= 512 rows, q <= 512 columns.  Fills the launch fields of grp.
bool qtt_bj2_config(int pmax, int qmax, int& EPL, int& BR, int& C);
cudaError_t qtt_launch_bj2(JacGroup& grp, int pmax, int qmax, double flops, cudaStream_t stream);
// L2-streamed block Jacobi (sbj.cu) for q <= 1024 columns, any number of rows; needs JacProb::work.
cudaError_t qtt_launch_sbj(const JacProb* probs, int n, cudaStream_t stream);
bool qtt_sbj_fits(int p, int q);

// Cluster-resident Householder QR of X (p x q, rows contiguous, ld), one cluster per matrix, column slices in
// shared memory (qrcp.cu).
//  pivot = 1 (rank-revealing preconditioner of the row-Jacobi SVD): X <- Q^T X in place, columns stay in place,
//    rows from the numerical rank on are written as zeros and the rank goes to rank_out (device int, may be null).
//  pivot = 0 (Q-less factor of the L->R sweep): R (q x q upper triangular, ld = q) of X = Q R goes to R_out,
//    X is left alone; needs p >= q.  With transposed = 1, X is given as Y = X^T (q x p, ld), i.e. R^T = the
//    L factor of Y = L Q.
struct QrcpProb {
  double* X;
  int p, q, ld;
  int* rank_out;
  int transposed;
  double* R_out;
};
#define QTT_QRCP_MAX_BATCH 16
struct QrcpGroup {
  int nprob;
  int cluster;  // CTAs per matrix
  int w;        // columns per CTA (largest problem)
  int pp;       // column pitch in shared memory
  int chm;      // rows per staged pivot-column chunk (largest problem)
  int pivot;
  QrcpProb p[QTT_QRCP_MAX_BATCH];
};
cudaError_t qtt_launch_qrcp(const QrcpProb* probs, int n, int pivot, cudaStream_t stream);
bool qtt_qrcp_fits(int p, int q);  // the column slices of a p x q matrix fit in a cluster's shared memory

// After rowjacobi: sort the rows by norm, pick the rank, write normalised rows.
//   sigma[0..p) <- row norms, descending;  rank[0] <- r' ;  out (r_cap x q, ld = q) <- top rows / sigma.
// Rank rule (oracle O6): eps_delta < 0  ->  r' = min(chi_max, p, q);
// else smallest r with sqrt(sum_{i>=r} sigma_i^2) <= delta, delta = *delta_ptr, then clamp to [1, chi_max].
// If norm_out != nullptr, *norm_out <- sqrt(sum sigma^2) * norm_scale_for_delta (used to derive delta).
struct SelProb {
  const double* X; int p, q, ld;
  double* out; int out_ld; int r_cap;
  double* sigma; int* rank;
  const double* delta_ptr;  // device scalar or nullptr (eps = 0)
  double* delta_out;        // if non-null: *delta_out = delta_scale * ||X||_F  (first SVD of a sweep)
  double delta_scale;
  int chi_max;
};
#define QTT_SEL_MAX_BATCH 16
struct SelGroup { int nprob; SelProb p[QTT_SEL_MAX_BATCH]; };
cudaError_t qtt_launch_select(const SelProb* probs, int n, cudaStream_t stream);
int qtt_select_max_rows();  // largest p the sort handles (shared-memory keys)

// ----------------------------------------------------------------------------------------------
// Data movement (bandwidth-bound).
// MPO x MPS site expand (paper Sec. II.B): out[(al,a), w, (be,b)] = sum_w' W[al,w,w',be] * A[a,w',b].
struct ExpandProb { const double* W; const double* A; double* out; int Dl, Dr, a, b; int d; };  // d: physical dimension (4 or 8)
#define QTT_MOVE_MAX_BATCH 16
struct ExpandGroup { int nprob; ExpandProb p[QTT_MOVE_MAX_BATCH]; };
cudaError_t qtt_launch_expand(const ExpandProb* probs, int n, cudaStream_t stream);

// Direct sum of up to 5 site tensors (first / middle / last site), scalars on the first site.
struct ConcatProb {
  const double* src[5]; double alpha[5]; int rl[5], rr[5]; int nterm;
  double* out; int mode;  // 0 first (row concat of columns), 1 middle (block diagonal), 2 last (stack rows)
  int d;                  // physical dimension (4 or 8)
};
struct ConcatGroup { int nprob; ConcatProb p[QTT_MOVE_MAX_BATCH]; };
cudaError_t qtt_launch_concat(const ConcatProb* probs, int n, cudaStream_t stream);

// Hadamard site tensor (paper Eq. 8): out[(a,b), w, (a2,b2)] = A[a,w,a2] * B[b,w,b2].
struct KronProb { const double* A; const double* B; double* out; int a, a2, b, b2; int d; };
struct KronGroup { int nprob; KronProb p[QTT_MOVE_MAX_BATCH]; };
cudaError_t qtt_launch_kron(const KronProb* probs, int n, cudaStream_t stream);

// Quantics bit interleave (paper Eq. 3): dense F[x][y] (N x N) <-> tensor U[w_1..w_n], w_k = 2 x_k + y_k (ndim = 2), or
// dense F[x][y][z] (N^3) <-> U with w_k = 4 x_k + 2 y_k + z_k (ndim = 3; reading 26).
cudaError_t qtt_launch_interleave(const double* F, double* U, int nbits, int ndim, int inverse, cudaStream_t stream);
// Generic 2-D transpose / strided copy: dst[j * ldd + i] = src[i * lds + j], i < rows, j < cols.
cudaError_t qtt_launch_transpose(const double* src, int rows, int cols, int lds, double* dst, int ldd,
                                 cudaStream_t stream);
// dst[i*ldd + j] = src[i*lds + j]
cudaError_t qtt_launch_copy2d(const double* src, int rows, int cols, int lds, double* dst, int ldd,
                              cudaStream_t stream);
cudaError_t qtt_launch_fill(double* dst, i64 n, double value, cudaStream_t stream);
// X[a][w][b][t] *= x_t[w], the sign vector of probe t at site `site` of the sketched zip-up (movement.cu; a < na, b < nbp, t < P)
cudaError_t qtt_launch_sketch_mixers(unsigned long long seed, int site, double* G, int P, cudaStream_t stream);
// Diagnostics (spectrum.cu): unnormalised 2-D DFT of a real N x N field (complex output, interleaved re/im, transposed
// wave-number order; tmp_c: 2 N^2 doubles) and the shell sums of the TKE spectrum (Eq. 13-15).
cudaError_t qtt_launch_fft2_real(const double* F, double* out_c, double* tmp_c, int nbits, cudaStream_t stream);
cudaError_t qtt_launch_tke_shells(const double* U1_c, const double* U2_c, int nbits, int nbins, double* partial,
                                  double* E_dev, cudaStream_t stream);

// Per-context launch counter and per-kernel-family timing (qtt_ctx_launch_count, qtt_ctx_profile_*).  The launchers
// only know a stream, so the record they write to is a thread-local pointer that every qtt_* call binds to its
// context on entry; the handle-less diagnostic entry points (qtt_diag.h) fall back to one process-wide record.
enum QttKernelFamily { QK_GEMM = 0, QK_LQ_PANEL, QK_LQ_UPDATE, QK_JACOBI, QK_SELECT, QK_MOVE, QK_QRCP, QK_COUNT };
struct QttProfRec { int fam; cudaEvent_t e0, e1; double work; int d[4]; };
struct QttStats {
  long long launches = 0;  // kernels enqueued by the launchers above
  bool prof_on = false;    // bracket every launch by a CUDA event pair (must be off while a stream is being captured)
  void* recs = nullptr;    // std::vector<QttProfRec>*, owned by probe.cu
};
QttStats* qtt_stats_current();
void qtt_stats_bind(QttStats* s);  // nullptr: back to the process-wide default record
void qtt_stats_destroy(QttStats* s);
struct QttProf {
  QttStats* stats;
  cudaStream_t st;
  bool live;
  // work: algorithmic flops (GEMM, LQ, Jacobi) or bytes (select, move) of this launch
  // d0..d3: shape tag of the launch (per family, see qtt_diag_profile_dump in include/qtt_diag.h)
  QttProf(int family, cudaStream_t stream, double work, int d0 = 0, int d1 = 0, int d2 = 0, int d3 = 0);
  ~QttProf();
};
// Synchronises the device, sums the event pairs recorded in `s` so far and clears them.
cudaError_t qtt_prof_collect(QttStats* s, double ms[QK_COUNT], double work[QK_COUNT], long long launches[QK_COUNT]);

// Kernel attributes (opt-in shared memory, non-portable cluster size) are per DEVICE: true the first time `key`
// (the kernel's address) is seen on the current device.  Thread-safe.
bool qtt_first_use_on_device(const void* key);
