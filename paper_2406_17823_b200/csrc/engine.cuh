// Host-side engine behind the qtt_* C ABI: handles, the two-ended workspace stack, and the batched
// sweeps that sequence the kernels of common.cuh.  Everything here only ENQUEUES work on the context's
// stream; with eps == 0 no call synchronises, so a whole RK4 step can be stream-captured.
#pragma once
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "../../include/qtt.h"
#include "common.cuh"

struct QttError {
  int status;
  std::string msg;
};
#define QTT_THROW(st, m) throw QttError{(st), std::string(m)}
#define QTT_CU(expr)                                                                                   \
  do {                                                                                                 \
    cudaError_t _e = (expr);                                                                           \
    if (_e != cudaSuccess)                                                                             \
      throw QttError{QTT_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e)};                    \
  } while (0)

// Workspace: "keep" stack grows from the bottom (results that outlive one rounding), "tmp" stack grows
// from the top (scratch of one rounding level).
struct Arena {
  char* base = nullptr;
  size_t size = 0, lo = 0, hi = 0;
  double* keep(size_t doubles);
  double* tmp(size_t doubles);
};

// An MPS with explicit dense cores in device memory: core[k] is r[k] x d x r[k+1], row-major, d = ctx->d (4 or 8).
struct View {
  int n = 0;
  std::vector<int> r;
  std::vector<const double*> core;
};

struct MpoData {
  int refs = 1;
  qtt_ctx* ctx = nullptr;
  int n = 0;
  std::vector<int> D;
  double* storage = nullptr;
  std::vector<const double*> core;
};

enum BodyKind { BODY_DENSE = 0, BODY_APPLIED = 1, BODY_PRODUCT = 2, BODY_SUM = 3 };
struct Body {
  int refs = 1;
  qtt_ctx* ctx = nullptr;
  int kind = BODY_DENSE;
  int n = 0;
  std::vector<int> r;
  // DENSE
  double* storage = nullptr;
  size_t storage_doubles = 0;
  bool tight = false;  // cores packed back to back in storage with exactly the bonds r
  std::vector<double*> core;
  // lazy kinds
  MpoData* mpo = nullptr;
  Body* x = nullptr;
  Body *a = nullptr, *b = nullptr;
  std::vector<std::pair<double, Body*>> terms;
};

struct qtt_mps {
  qtt_ctx* ctx;
  Body* body;
};
struct qtt_mpo {
  MpoData* data;
};

struct Rk4Plan;

struct qtt_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  qtt_alloc_fn alloc = nullptr;
  qtt_release_fn release = nullptr;
  void* user = nullptr;
  Arena arena;
  // a second stream with its own scratch region (the top quarter of the workspace): qtt_rk4_step runs the two
  // Laplacian roundings of a right-hand side there, concurrently with the four products that do not need them
  cudaStream_t side = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  Arena side_arena;
  std::string err;
  int d = 4;  // physical dimension: 4 = 2D grid (Eq. 3), 8 = 3D grid (reading 26); fixed while handles live
  int live = 0;  // MPS / MPO handles alive (qtt_ctx_set_phys_dim refuses to switch under them)
  int chi_work = 0;
  size_t mat_limit = (size_t)2 << 30;
  int graphs = 1;
  int skew = 0;  // 1: skew-symmetric convection (PAPER.md Eq. B2) in qtt_rk4_step
  int sketch = 0;  // 1: the truncating steps of the zip-up use a randomised range finder (reading 25)
  unsigned long long sketch_seed = 0;
  int profiling = 0;
  QttStats stats;           // this context's launch counter and profiler records (bound on entry of every qtt_* call)
  double* ones = nullptr;   // device: 1.0
  int* jac_status = nullptr;  // device: [max sweeps, limit hits]
  int numeric_seen = 0;       // limit hits already reported through QTT_NUMERIC
  long long graph_launches = 0;
  std::vector<Rk4Plan*> plans;
};

// Output of a rounding: cores are written into caller-provided slots sized for the capacity bonds.
struct OutMps {
  int n = 0;
  std::vector<int> rcap;  // capacity bonds (= exact bonds when eps == 0)
  std::vector<int> r;     // actual bonds, filled by the sweep
  std::vector<double*> core;
};

// static (eps == 0) bonds of round(dense MPS with bonds r, chi)
// (d = physical dimension; the default serves the callers that are built for the 2D encoding only)
std::vector<int> qtt_round_caps(const std::vector<int>& r, int chi, int d = 4);
// working bonds of the zip-up and static bonds of its result
void qtt_zip_caps(const std::vector<int>& ra, const std::vector<int>& rb, int chi, int chi_work,
                  std::vector<int>& rwork, std::vector<int>& rout, int d = 4);

struct SigmaCapture {
  // per item, per bond k (1..n-1): device pointer to the singular values (count[k] of them)
  std::vector<std::vector<double*>> sigma;
  std::vector<std::vector<int>> count;
};

// Oracle O6 on a batch of dense MPS (same n).  out[i].core slots must be allocated by the caller.
void qtt_round_dense_batch(qtt_ctx* ctx, const std::vector<View>& in, int chi, double eps, std::vector<OutMps>& out,
                           SigmaCapture* cap = nullptr);
// Oracle O7 on a batch of pairs (A, B).
void qtt_round_product_batch(qtt_ctx* ctx, const std::vector<View>& A, const std::vector<View>& B, int chi, double eps,
                             int chi_work, std::vector<OutMps>& out);

// exact lazy results materialised as dense cores in the tmp stack
View qtt_expand_apply(qtt_ctx* ctx, const MpoData* W, const View& x);
void qtt_expand_apply_batch(qtt_ctx* ctx, const std::vector<const MpoData*>& W, const std::vector<View>& x,
                            std::vector<View>& out);
void qtt_concat_batch(qtt_ctx* ctx, const std::vector<std::vector<std::pair<double, View>>>& terms,
                      std::vector<View>& out);
View qtt_kron(qtt_ctx* ctx, const View& a, const View& b);

void qtt_rk4_eager(qtt_ctx* ctx, const View u[2], const MpoData* Dx, const MpoData* Dy, const MpoData* Lap, double Re,
                   double dt, int chi, double eps, int chi_work, int skew, OutMps out[2]);

void qtt_rk4_eager3(qtt_ctx* ctx, const View u[3], const MpoData* const Dj[3], const MpoData* Lap, double Re, double dt,
                    int chi, double eps, int chi_work, OutMps out[3]);

void qtt_to_dense_view(qtt_ctx* ctx, const View& v, double* dense_dev_out);
void qtt_from_dense(qtt_ctx* ctx, const double* dense_dev, int nbits, int chi, double eps, OutMps& out);
double* qtt_dot_view(qtt_ctx* ctx, const View& a, const View& b);  // device scalar in tmp




// ------------------------------------------------------------------------------------------ GEMM views (row-major)
inline GemmProb gemm_base(const double* A, const double* B, double* C, int M, int N, int K) {
  GemmProb p;
  std::memset(&p, 0, sizeof(p));
  p.A = A; p.B = B; p.C = C;
  p.M = M; p.N = N; p.K = K;
  p.nbatch = 1;
  p.alpha = 1.0; p.beta = 0.0;
  return p;
}
// plain row-major C(MxN, ldc) = A(MxK, lda) * B(KxN, ldb)
inline GemmProb gemm_nn(const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc, int M, int N, int K) {
  GemmProb p = gemm_base(A, B, C, M, N, K);
  p.a_lo = lda; p.a_k = 1;
  p.b_k = ldb; p.b_n = 1;
  p.c_lo = ldc; p.c_n = 1;
  return p;
}
// C = A * B^T with B stored N x K (ldb)
inline GemmProb gemm_nt(const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc, int M, int N, int K) {
  GemmProb p = gemm_nn(A, lda, B, 0, C, ldc, M, N, K);
  p.b_k = 1; p.b_n = ldb;
  return p;
}
// C = A^T * B with A stored K x M (lda)
inline GemmProb gemm_tn(const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc, int M, int N, int K) {
  GemmProb p = gemm_nn(A, 0, B, ldb, C, ldc, M, N, K);
  p.a_lo = 1; p.a_k = lda;
  return p;
}


void qtt_row_space_basis(qtt_ctx* ctx, double* X, int p, int q, double* out);

// The variational stage (variational.cu; Sec. II.C, App. B): out[i].core slots sized for the bonds of v0[i].
void qtt_variational_stage_impl(qtt_ctx* ctx, const View v0[2], const View a[2], const View Bm[2], const MpoData* D1,
                                const MpoData* D2, double h, double mu, int max_sweeps, double sweep_tol, int cg_maxit,
                                double cg_tol, OutMps out[2], int* sweeps_out, long long* cg_total, int* cg_max);
double qtt_variational_cost_impl(qtt_ctx* ctx, const View v[2], const View a[2], const View Bm[2], const MpoData* D1,
                                 const MpoData* D2, double h, double mu);

