// The variational (DMRG-like) stage of the paper's solver (Sec. II.C,
// App. B): minimise
//     Theta(v) = mu || D_1 v_1 + D_2 v_2 ||^2 + sum_i || (v_i - a_i) / h + B_i ||^2        (PAPER.md:452 Eq. B6)
// over the velocity MPS pair v with fixed bonds by one-site sweeps.  At the canonical centre d the stationarity
// condition (Eq. B22) is the coupled linear system (Eq. B23-B24)
//     C_i - mu h^2 sum_j <basis_i| D_i D_j |basis_j> C_j = <basis_i| a_i - h B_i>,        i = 1, 2,
// symmetric positive definite because D^T = -D, solved by conjugate gradients from the current centre
// tensors (at most 100 iterations, relative residual 1e-5).  Everything heavy is a contraction:
//   * environments LH_ij (bond_i x m x bond_j, m the bond of the product MPO D_i D_j) and LG_i (bond_i x bond_g):
//     grouped DMMA GEMMs (gemm.cu) around one small gather kernel that contracts the MPO core (K = 4 m <= 36, 0/+-1
//     weights: not a tensor-core problem, as row a1 of the hot path);
//   * the local operator of a CG iteration: the same three steps per (i, j);
//   * the centre is moved with the SVD step of the rounding sweeps (an orthonormal basis of the row space; the paper and
//     the oracle use a QR factorisation -- the gauge differs, the represented state and the Krylov iterates do not).
// The CG loop is driven from the host (two scalar read-backs per iteration): this stage is iterative and its length is
// data dependent, so it is not graph-captured.
#include <algorithm>
#include <cmath>
#include <vector>

#include "engine.cuh"

namespace {

// out[o1, o2, r1, r2] = sum_{s1 < S1, s2 < S2} W[o1, o2, s1, s2] * in[s1, s2, r1, r2], every array through element strides
struct MpocProb {
  const double* W;
  const double* in;
  double* out;
  int O1, O2, S1, S2, R1, R2;
  i64 wo1, wo2, ws1, ws2;
  i64 is1, is2, ir1, ir2;
  i64 oo1, oo2, or1, or2;
};
__global__ void qtt_mpoc_kernel(const __grid_constant__ MpocProb P) {
  const i64 total = (i64)P.O1 * P.O2 * P.R1 * P.R2;
  for (i64 idx = (i64)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (i64)gridDim.x * blockDim.x) {
    // the fastest output stride first, so that neighbouring threads write neighbouring words
    i64 t = idx;
    int r2, r1, o2, o1;
    if (P.or2 == 1) {
      r2 = (int)(t % P.R2); t /= P.R2;
      o2 = (int)(t % P.O2); t /= P.O2;
      r1 = (int)(t % P.R1); t /= P.R1;
      o1 = (int)t;
    } else {
      o2 = (int)(t % P.O2); t /= P.O2;
      r2 = (int)(t % P.R2); t /= P.R2;
      o1 = (int)(t % P.O1); t /= P.O1;
      r1 = (int)t;
    }
    const double* w = P.W + o1 * P.wo1 + o2 * P.wo2;
    const double* x = P.in + r1 * P.ir1 + r2 * P.ir2;
    double s = 0.0;
    for (int s1 = 0; s1 < P.S1; ++s1)
      for (int s2 = 0; s2 < P.S2; ++s2) {
        const double wv = __ldg(w + s1 * P.ws1 + s2 * P.ws2);
        if (wv != 0.0) s = fma(wv, x[s1 * P.is1 + s2 * P.is2], s);
      }
    P.out[o1 * P.oo1 + o2 * P.oo2 + r1 * P.or1 + r2 * P.or2] = s;
  }
}
void launch_mpoc(const MpocProb& p, cudaStream_t st) {
  const i64 total = (i64)p.O1 * p.O2 * p.R1 * p.R2;
  if (total <= 0) return;
  int blocks = (int)std::min<i64>((total + 255) / 256, 148 * 8);
  QttProf prof(QK_MOVE, st, 8.0 * (double)total * (1.0 + p.S1 * p.S2));
  qtt_mpoc_kernel<<<blocks, 256, 0, st>>>(p);
  QTT_CU(cudaGetLastError());
}

// out[0] = sum_i x[i] * y[i], one block, fixed summation order (deterministic)
__global__ void __launch_bounds__(1024) qtt_dot_kernel(const double* x, const double* y, i64 n, double* out) {
  __shared__ double red[32];
  double s = 0.0;
  for (i64 i = threadIdx.x; i < n; i += 1024) s = fma(x[i], y[i], s);
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x < 32) {
    s = red[threadIdx.x];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) out[0] = s;
  }
}
// y <- a x + b y
__global__ void qtt_axpby_kernel(double a, const double* x, double b, double* y, i64 n) {
  for (i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (i64)gridDim.x * blockDim.x)
    y[i] = fma(a, x[i], b * y[i]);
}

struct Stage {
  qtt_ctx* ctx;
  cudaStream_t st;
  int n;
  double h, mu;
  // the trial state: cores of capacity r0[k] x 4 x r0[k+1]; the bonds can only shrink when the centre moves
  std::vector<int> r[2];
  std::vector<double*> V[2];
  View g[2];                       // a_i - h B_i
  std::vector<int> Dw[2][2];       // bonds of the product MPOs D_i D_j
  std::vector<const double*> W[2][2];
  std::vector<double*> LH[2][2], RH[2][2], LG[2], RG[2];
  double* hostpin = nullptr;       // 2 doubles of pinned host memory for the scalar read-backs
  double* dscal = nullptr;         // 2 device doubles

  void gemms(std::vector<GemmProb>& v) {
    if (v.empty()) return;
    QTT_CU(qtt_launch_gemm(v.data(), (int)v.size(), st));
    v.clear();
  }
  double dot(const double* x, const double* y, i64 nn) {
    {
      QttProf prof(QK_MOVE, st, 16.0 * (double)nn);
      qtt_dot_kernel<<<1, 1024, 0, st>>>(x, y, nn, dscal);
    }
    QTT_CU(cudaGetLastError());
    QTT_CU(cudaMemcpyAsync(hostpin, dscal, sizeof(double), cudaMemcpyDeviceToHost, st));
    QTT_CU(cudaStreamSynchronize(st));
    return hostpin[0];
  }
  void axpby(double a, const double* x, double b, double* y, i64 nn) {
    int blocks = (int)std::min<i64>((nn + 255) / 256, 148 * 4);
    QttProf prof(QK_MOVE, st, 24.0 * (double)nn);
    qtt_axpby_kernel<<<blocks, 256, 0, st>>>(a, x, b, y, nn);
    QTT_CU(cudaGetLastError());
  }

  // contraction of the MPO core of D_i D_j at site k with T1: the summed pair is (left MPO bond, its physical index)
  // [from_left] or (right MPO bond, its physical index); strides of `in` and `out` are given for (s1, s2, r1, r2) / (o1, o2, r1, r2)
  void mpoc(int i, int j, int k, bool sum_left, const double* in, double* out, int R1, int R2, i64 is1, i64 is2, i64 ir1,
            i64 ir2, i64 oo1, i64 oo2, i64 or1, i64 or2) {
    const int Dm = Dw[i][j][k], Dn = Dw[i][j][k + 1];
    MpocProb p;
    p.W = W[i][j][k]; p.in = in; p.out = out;
    p.R1 = R1; p.R2 = R2;
    p.is1 = is1; p.is2 = is2; p.ir1 = ir1; p.ir2 = ir2;
    p.oo1 = oo1; p.oo2 = oo2; p.or1 = or1; p.or2 = or2;
    // W[m][w][x][n]: strides 16 Dn, 4 Dn, Dn, 1
    if (sum_left) {  // sum over (m, w), output (n, x)
      p.S1 = Dm; p.S2 = 4; p.O1 = Dn; p.O2 = 4;
      p.ws1 = 16 * (i64)Dn; p.ws2 = 4 * (i64)Dn; p.wo1 = 1; p.wo2 = Dn;
    } else {         // sum over (n, x), output (m, w)
      p.S1 = Dn; p.S2 = 4; p.O1 = Dm; p.O2 = 4;
      p.ws1 = 1; p.ws2 = Dn; p.wo1 = 16 * (i64)Dn; p.wo2 = 4 * (i64)Dn;
    }
    launch_mpoc(p, st);
  }

  // environments left of site k+1 from those left of site k (site k of both states is left-orthonormal)
  void upd_left(int k) {
    const size_t mark = ctx->arena.hi;
    std::vector<GemmProb> gq;
    double* T1[2][2];
    double* T2[2][2];
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int a = r[i][k], b = r[i][k + 1], c = r[j][k], m = Dw[i][j][k];
        T1[i][j] = ctx->arena.tmp((size_t)m * c * 4 * b);
        // T1[(m,c),(w,b)] = sum_a LH[a,(m,c)] V_i[a,(w,b)]
        gq.push_back(gemm_tn(LH[i][j][k], (i64)m * c, V[i][k], 4 * (i64)b, T1[i][j], 4 * (i64)b, m * c, 4 * b, a));
      }
    gemms(gq);
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int b = r[i][k + 1], c = r[j][k], nn = Dw[i][j][k + 1];
        T2[i][j] = ctx->arena.tmp((size_t)b * nn * c * 4);
        // T2[b][n][c][x] = sum_{m,w} W[m,w,x,n] T1[m][c][w][b]
        mpoc(i, j, k, true, T1[i][j], T2[i][j], b, c, (i64)c * 4 * b, b, 1, 4 * (i64)b, (i64)c * 4, 1, (i64)nn * c * 4, 4);
      }
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int b = r[i][k + 1], c = r[j][k], d = r[j][k + 1], nn = Dw[i][j][k + 1];
        // LH'[(b,n),d] = sum_{(c,x)} T2[(b,n),(c,x)] V_j[(c,x),d]
        gq.push_back(gemm_nn(T2[i][j], 4 * (i64)c, V[j][k], d, LH[i][j][k + 1], d, b * nn, d, 4 * c));
      }
    gemms(gq);
    double* T[2];
    for (int i = 0; i < 2; ++i) {
      const int a = r[i][k], b = r[i][k + 1], c = g[i].r[k];
      T[i] = ctx->arena.tmp((size_t)c * 4 * b);
      gq.push_back(gemm_tn(LG[i][k], c, V[i][k], 4 * (i64)b, T[i], 4 * (i64)b, c, 4 * b, a));
    }
    gemms(gq);
    for (int i = 0; i < 2; ++i) {
      const int b = r[i][k + 1], c = g[i].r[k], d = g[i].r[k + 1];
      // LG'[b,d] = sum_{(c,w)} T[(c,w),b] g[(c,w),d]
      gq.push_back(gemm_tn(T[i], b, g[i].core[k], d, LG[i][k + 1], d, b, d, 4 * c));
    }
    gemms(gq);
    ctx->arena.hi = mark;
  }

  // environments right of site k-1 from those right of site k (site k of both states is right-orthonormal)
  void upd_right(int k) {
    const size_t mark = ctx->arena.hi;
    std::vector<GemmProb> gq;
    double* T1[2][2];
    double* T2[2][2];
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int b = r[i][k + 1], c = r[j][k], d = r[j][k + 1], nn = Dw[i][j][k + 1];
        T1[i][j] = ctx->arena.tmp((size_t)b * nn * c * 4);
        // T1[(b,n),(c,x)] = sum_d RH[(b,n),d] V_j[(c,x),d]
        gq.push_back(gemm_nt(RH[i][j][k + 1], d, V[j][k], d, T1[i][j], 4 * (i64)c, b * nn, 4 * c, d));
      }
    gemms(gq);
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int b = r[i][k + 1], c = r[j][k], m = Dw[i][j][k], nn = Dw[i][j][k + 1];
        T2[i][j] = ctx->arena.tmp((size_t)4 * b * m * c);
        // T2[w][b][m][c] = sum_{n,x} W[m,w,x,n] T1[b][n][c][x]
        mpoc(i, j, k, false, T1[i][j], T2[i][j], b, c, (i64)c * 4, 1, (i64)nn * c * 4, 4, c, (i64)b * m * c, (i64)m * c, 1);
      }
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int a = r[i][k], b = r[i][k + 1], c = r[j][k], m = Dw[i][j][k];
        // RH[a,(m,c)] = sum_{(w,b)} V_i[a,(w,b)] T2[(w,b),(m,c)]
        gq.push_back(gemm_nn(V[i][k], 4 * (i64)b, T2[i][j], (i64)m * c, RH[i][j][k], (i64)m * c, a, m * c, 4 * b));
      }
    gemms(gq);
    double* T[2];
    for (int i = 0; i < 2; ++i) {
      const int a = r[i][k], b = r[i][k + 1], d = g[i].r[k + 1];
      T[i] = ctx->arena.tmp((size_t)a * 4 * d);
      // T[(a,w),d] = V_i[(a,w),b] RG'[b,d]
      gq.push_back(gemm_nn(V[i][k], b, RG[i][k + 1], d, T[i], d, 4 * a, d, b));
    }
    gemms(gq);
    for (int i = 0; i < 2; ++i) {
      const int a = r[i][k], c = g[i].r[k], d = g[i].r[k + 1];
      // RG[a,c] = sum_{(w,d)} T[a,(w,d)] g[c,(w,d)]
      gq.push_back(gemm_nt(T[i], 4 * (i64)d, g[i].core[k], 4 * (i64)d, RG[i][k], c, a, c, 4 * d));
    }
    gemms(gq);
    ctx->arena.hi = mark;
  }

  i64 off1(int d) const { return (i64)r[0][d] * 4 * r[0][d + 1]; }
  i64 len(int d) const { return off1(d) + (i64)r[1][d] * 4 * r[1][d + 1]; }

  // y <- x - mu h^2 sum_j P_i^T D_i D_j P_j x_j  (the operator of Eq. B23-B24 at site d); x, y: [component 0 | component 1]
  void op(int d, const double* x, double* y) {
    const size_t mark = ctx->arena.hi;
    const i64 nn = len(d);
    QTT_CU(cudaMemcpyAsync(y, x, sizeof(double) * nn, cudaMemcpyDeviceToDevice, st));
    std::vector<GemmProb> gq;
    double* T1[2][2];
    double* T2[2][2];
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int b = r[i][d + 1], c = r[j][d], dd = r[j][d + 1], n2 = Dw[i][j][d + 1];
        T1[i][j] = ctx->arena.tmp((size_t)b * n2 * c * 4);
        const double* xj = x + (j ? off1(d) : 0);
        gq.push_back(gemm_nt(RH[i][j][d + 1], dd, xj, dd, T1[i][j], 4 * (i64)c, b * n2, 4 * c, dd));
      }
    gemms(gq);
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) {
        const int b = r[i][d + 1], c = r[j][d], m = Dw[i][j][d], n2 = Dw[i][j][d + 1];
        T2[i][j] = ctx->arena.tmp((size_t)m * c * 4 * b);
        // T2[m][c][w][b] = sum_{n,x} W[m,w,x,n] T1[b][n][c][x]
        mpoc(i, j, d, false, T1[i][j], T2[i][j], b, c, (i64)c * 4, 1, (i64)n2 * c * 4, 4, (i64)c * 4 * b, b, 1, 4 * (i64)b);
      }
    for (int j = 0; j < 2; ++j) {  // the two j accumulate into the same y_i: one launch per j
      for (int i = 0; i < 2; ++i) {
        const int a = r[i][d], b = r[i][d + 1], c = r[j][d], m = Dw[i][j][d];
        double* yi = y + (i ? off1(d) : 0);
        GemmProb p = gemm_nn(LH[i][j][d], (i64)m * c, T2[i][j], 4 * (i64)b, yi, 4 * (i64)b, a, 4 * b, m * c);
        p.alpha = -mu * h * h;
        p.beta = 1.0;
        gq.push_back(p);
      }
      gemms(gq);
    }
    ctx->arena.hi = mark;
  }

  // right-hand side <basis_i| g_i> at site d
  void rhs(int d, double* out) {
    const size_t mark = ctx->arena.hi;
    std::vector<GemmProb> gq;
    double* T[2];
    for (int i = 0; i < 2; ++i) {
      const int a = r[i][d], c = g[i].r[d], dd = g[i].r[d + 1];
      T[i] = ctx->arena.tmp((size_t)a * 4 * dd);
      gq.push_back(gemm_nn(LG[i][d], c, g[i].core[d], 4 * (i64)dd, T[i], 4 * (i64)dd, a, 4 * dd, c));
    }
    gemms(gq);
    for (int i = 0; i < 2; ++i) {
      const int a = r[i][d], b = r[i][d + 1], dd = g[i].r[d + 1];
      gq.push_back(gemm_nt(T[i], dd, RG[i][d + 1], dd, out + (i ? off1(d) : 0), b, 4 * a, b, dd));
    }
    gemms(gq);
    ctx->arena.hi = mark;
  }

  // conjugate gradients on the centre tensors of site d; returns the iterations used
  int solve_site(int d, int cg_maxit, double cg_tol) {
    const size_t mark = ctx->arena.hi;
    const i64 nn = len(d);
    double* x = ctx->arena.tmp((size_t)nn);
    double* b = ctx->arena.tmp((size_t)nn);
    double* rr_ = ctx->arena.tmp((size_t)nn);
    double* p = ctx->arena.tmp((size_t)nn);
    double* Ap = ctx->arena.tmp((size_t)nn);
    QTT_CU(cudaMemcpyAsync(x, V[0][d], sizeof(double) * off1(d), cudaMemcpyDeviceToDevice, st));
    QTT_CU(cudaMemcpyAsync(x + off1(d), V[1][d], sizeof(double) * (nn - off1(d)), cudaMemcpyDeviceToDevice, st));
    rhs(d, b);
    op(d, x, Ap);
    QTT_CU(cudaMemcpyAsync(rr_, b, sizeof(double) * nn, cudaMemcpyDeviceToDevice, st));
    axpby(-1.0, Ap, 1.0, rr_, nn);  // r = b - A x
    QTT_CU(cudaMemcpyAsync(p, rr_, sizeof(double) * nn, cudaMemcpyDeviceToDevice, st));
    double rr = dot(rr_, rr_, nn);
    const double bnorm = std::sqrt(dot(b, b, nn));
    int its = 0;
    while (its < cg_maxit && std::sqrt(rr) > cg_tol * bnorm) {
      op(d, p, Ap);
      const double pAp = dot(p, Ap, nn);
      const double alpha = rr / pAp;
      axpby(alpha, p, 1.0, x, nn);
      axpby(-alpha, Ap, 1.0, rr_, nn);
      const double rr_new = dot(rr_, rr_, nn);
      const double beta = rr_new / rr;
      axpby(1.0, rr_, beta, p, nn);  // p = r + beta p
      rr = rr_new;
      ++its;
    }
    QTT_CU(cudaMemcpyAsync(V[0][d], x, sizeof(double) * off1(d), cudaMemcpyDeviceToDevice, st));
    QTT_CU(cudaMemcpyAsync(V[1][d], x + off1(d), sizeof(double) * (nn - off1(d)), cudaMemcpyDeviceToDevice, st));
    ctx->arena.hi = mark;
    return its;
  }

  // centre d -> d - 1: site d becomes right-orthonormal (rows of its right unfolding), the rest goes into site d - 1
  void shift_left(int d) {
    for (int i = 0; i < 2; ++i) {
      const size_t mark = ctx->arena.hi;
      const int r0 = r[i][d], r1 = r[i][d + 1], q = 4 * r1, p0 = r[i][d - 1];
      const int rn = std::min(r0, q);
      double* M = ctx->arena.tmp((size_t)r0 * q);
      double* Vt = ctx->arena.tmp((size_t)rn * q);
      double* Cc = ctx->arena.tmp((size_t)r0 * rn);
      double* Ln = ctx->arena.tmp((size_t)p0 * 4 * rn);
      QTT_CU(cudaMemcpyAsync(M, V[i][d], sizeof(double) * (size_t)r0 * q, cudaMemcpyDeviceToDevice, st));
      qtt_row_space_basis(ctx, M, r0, q, Vt);
      std::vector<GemmProb> gq;
      gq.push_back(gemm_nt(V[i][d], q, Vt, q, Cc, rn, r0, rn, q));  // carry = core Vt^T
      gemms(gq);
      gq.push_back(gemm_nn(V[i][d - 1], r0, Cc, rn, Ln, rn, 4 * p0, rn, r0));
      gemms(gq);
      QTT_CU(cudaMemcpyAsync(V[i][d], Vt, sizeof(double) * (size_t)rn * q, cudaMemcpyDeviceToDevice, st));
      QTT_CU(cudaMemcpyAsync(V[i][d - 1], Ln, sizeof(double) * (size_t)p0 * 4 * rn, cudaMemcpyDeviceToDevice, st));
      r[i][d] = rn;
      ctx->arena.hi = mark;
    }
  }
  // centre d -> d + 1: site d becomes left-orthonormal (columns of its left unfolding)
  void shift_right(int d) {
    for (int i = 0; i < 2; ++i) {
      const size_t mark = ctx->arena.hi;
      const int r0 = r[i][d], r1 = r[i][d + 1], m = 4 * r0, r2 = r[i][d + 2];
      const int rn = std::min(r1, m);
      double* Xt = ctx->arena.tmp((size_t)r1 * m);
      double* Ut = ctx->arena.tmp((size_t)rn * m);
      double* Cc = ctx->arena.tmp((size_t)rn * r1);
      double* Nn = ctx->arena.tmp((size_t)rn * 4 * r2);
      QTT_CU(qtt_launch_transpose(V[i][d], m, r1, r1, Xt, m, st));
      qtt_row_space_basis(ctx, Xt, r1, m, Ut);
      std::vector<GemmProb> gq;
      gq.push_back(gemm_nn(Ut, m, V[i][d], r1, Cc, r1, rn, r1, m));  // carry = U^T core
      gemms(gq);
      gq.push_back(gemm_nn(Cc, r1, V[i][d + 1], 4 * (i64)r2, Nn, 4 * (i64)r2, rn, 4 * r2, r1));
      gemms(gq);
      QTT_CU(qtt_launch_transpose(Ut, rn, m, m, V[i][d], rn, st));
      QTT_CU(cudaMemcpyAsync(V[i][d + 1], Nn, sizeof(double) * (size_t)rn * 4 * r2, cudaMemcpyDeviceToDevice, st));
      r[i][d + 1] = rn;
      ctx->arena.hi = mark;
    }
  }
  double norm2() {
    double s = 0.0;
    for (int i = 0; i < 2; ++i) s += dot(V[i][0], V[i][0], (i64)4 * r[i][1]);
    return s;
  }
};

}  // namespace

// Host cores of the product MPO W1 W2 (W1 acts after W2): [(m1,m2)][w][w''][(m1',m2')]
static void mpo_product_host(const std::vector<std::vector<double>>& A, const std::vector<int>& Da,
                             const std::vector<std::vector<double>>& B, const std::vector<int>& Db,
                             std::vector<std::vector<double>>& out, std::vector<int>& Dout) {
  const int n = (int)A.size();
  out.resize(n);
  Dout.resize(n + 1);
  for (int k = 0; k <= n; ++k) Dout[k] = Da[k] * Db[k];
  for (int k = 0; k < n; ++k) {
    const int a0 = Da[k], a1 = Da[k + 1], b0 = Db[k], b1 = Db[k + 1];
    out[k].assign((size_t)a0 * b0 * 16 * a1 * b1, 0.0);
    for (int a = 0; a < a0; ++a)
      for (int o = 0; o < 4; ++o)
        for (int p = 0; p < 4; ++p)
          for (int b = 0; b < a1; ++b) {
            const double av = A[k][(((size_t)a * 4 + o) * 4 + p) * a1 + b];
            if (av == 0.0) continue;
            for (int c = 0; c < b0; ++c)
              for (int q = 0; q < 4; ++q)
                for (int d = 0; d < b1; ++d) {
                  const double bv = B[k][(((size_t)c * 4 + p) * 4 + q) * b1 + d];
                  if (bv == 0.0) continue;
                  out[k][((((size_t)(a * b0 + c)) * 4 + o) * 4 + q) * (a1 * b1) + (b * b1 + d)] += av * bv;
                }
          }
  }
}

void qtt_variational_stage_impl(qtt_ctx* ctx, const View v0[2], const View a[2], const View Bm[2], const MpoData* D1,
                                const MpoData* D2, double h, double mu, int max_sweeps, double sweep_tol, int cg_maxit,
                                double cg_tol, OutMps out[2], int* sweeps_out, long long* cg_total, int* cg_max) {
  Stage S;
  S.ctx = ctx;
  S.st = ctx->stream;
  S.n = v0[0].n;
  S.h = h;
  S.mu = mu;
  const int n = S.n;
  if (n < 2) QTT_THROW(QTT_INVALID_ARG, "the variational stage needs at least two sites");
  const MpoData* Dm[2] = {D1, D2};
  for (int i = 0; i < 2; ++i)
    if (v0[i].n != n || a[i].n != n || Bm[i].n != n || Dm[i]->n != n) QTT_THROW(QTT_SHAPE_MISMATCH, "operands differ in length");
  QTT_CU(cudaMallocHost(reinterpret_cast<void**>(&S.hostpin), 2 * sizeof(double)));
  struct PinGuard {
    double* p;
    ~PinGuard() { cudaFreeHost(p); }
  } guard{S.hostpin};
  S.dscal = ctx->arena.keep(2);
  // ---- product MPOs D_i D_j (host: the cores are tiny), uploaded once
  std::vector<std::vector<double>> Hc[2];
  for (int i = 0; i < 2; ++i) {
    Hc[i].resize(n);
    for (int k = 0; k < n; ++k) {
      Hc[i][k].resize((size_t)Dm[i]->D[k] * 16 * Dm[i]->D[k + 1]);
      QTT_CU(cudaMemcpyAsync(Hc[i][k].data(), Dm[i]->core[k], Hc[i][k].size() * sizeof(double), cudaMemcpyDeviceToHost, S.st));
    }
  }
  QTT_CU(cudaStreamSynchronize(S.st));
  std::vector<std::vector<double>> Hp[2][2];
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 2; ++j) {
      mpo_product_host(Hc[i], Dm[i]->D, Hc[j], Dm[j]->D, Hp[i][j], S.Dw[i][j]);
      S.W[i][j].resize(n);
      for (int k = 0; k < n; ++k) {
        double* dptr = ctx->arena.keep(Hp[i][j][k].size());
        QTT_CU(cudaMemcpyAsync(dptr, Hp[i][j][k].data(), Hp[i][j][k].size() * sizeof(double), cudaMemcpyHostToDevice, S.st));
        S.W[i][j][k] = dptr;
      }
    }
  QTT_CU(cudaStreamSynchronize(S.st));  // (the host vectors may now go)
  // ---- g_i = a_i - h B_i (exact direct sum), working copy of v
  for (int i = 0; i < 2; ++i) {
    std::vector<std::vector<std::pair<double, View>>> terms{{{1.0, a[i]}, {-h, Bm[i]}}};
    std::vector<View> o;
    qtt_concat_batch(ctx, terms, o);
    S.g[i] = o[0];
    S.r[i] = v0[i].r;
    S.V[i].resize(n);
    for (int k = 0; k < n; ++k) {
      const size_t sz = (size_t)v0[i].r[k] * 4 * v0[i].r[k + 1];
      S.V[i][k] = ctx->arena.keep(sz);
      QTT_CU(cudaMemcpyAsync(S.V[i][k], v0[i].core[k], sz * sizeof(double), cudaMemcpyDeviceToDevice, S.st));
    }
  }
  // ---- right-canonical form with the centre on site 1 (PAPER.md:498-518 Eq. B15-B19)
  for (int k = n - 1; k >= 1; --k) S.shift_left(k);
  // ---- environments (sized for the bonds as they are now: they can only shrink further)
  for (int i = 0; i < 2; ++i) {
    S.LG[i].assign(n + 1, nullptr);
    S.RG[i].assign(n + 1, nullptr);
    for (int k = 0; k <= n; ++k) {
      S.LG[i][k] = ctx->arena.keep((size_t)S.r[i][k] * S.g[i].r[k]);
      S.RG[i][k] = ctx->arena.keep((size_t)S.r[i][k] * S.g[i].r[k]);
    }
    for (int j = 0; j < 2; ++j) {
      S.LH[i][j].assign(n + 1, nullptr);
      S.RH[i][j].assign(n + 1, nullptr);
      for (int k = 0; k <= n; ++k) {
        const size_t sz = (size_t)S.r[i][k] * S.Dw[i][j][k] * S.r[j][k];
        S.LH[i][j][k] = ctx->arena.keep(sz);
        S.RH[i][j][k] = ctx->arena.keep(sz);
      }
      QTT_CU(qtt_launch_fill(S.LH[i][j][0], 1, 1.0, S.st));
      QTT_CU(qtt_launch_fill(S.RH[i][j][n], 1, 1.0, S.st));
    }
    QTT_CU(qtt_launch_fill(S.LG[i][0], 1, 1.0, S.st));
    QTT_CU(qtt_launch_fill(S.RG[i][n], 1, 1.0, S.st));
  }
  for (int k = n - 1; k >= 1; --k) S.upd_right(k);

  long long tot = 0;
  int mx = 0, sweeps = 0;
  auto solve = [&](int d) {
    const int its = S.solve_site(d, cg_maxit, cg_tol);
    tot += its;
    mx = std::max(mx, its);
  };
  double prev = S.norm2();
  for (sweeps = 1; sweeps <= max_sweeps; ++sweeps) {
    for (int d = 0; d < n - 1; ++d) {
      solve(d);
      S.shift_right(d);
      S.upd_left(d);
    }
    solve(n - 1);
    for (int d = n - 1; d >= 1; --d) {
      S.shift_left(d);
      S.upd_right(d);
      solve(d - 1);
    }
    const double cur = S.norm2();
    const double change = std::fabs(cur - prev) / std::max(cur, 1e-300);
    prev = cur;
    if (change < sweep_tol) break;
  }
  if (sweeps > max_sweeps) sweeps = max_sweeps;
  for (int i = 0; i < 2; ++i) {
    out[i].r = S.r[i];
    for (int k = 0; k < n; ++k)
      QTT_CU(cudaMemcpyAsync(out[i].core[k], S.V[i][k], sizeof(double) * (size_t)S.r[i][k] * 4 * S.r[i][k + 1],
                             cudaMemcpyDeviceToDevice, S.st));
  }
  QTT_CU(cudaStreamSynchronize(S.st));
  if (sweeps_out) *sweeps_out = sweeps;
  if (cg_total) *cg_total = tot;
  if (cg_max) *cg_max = mx;
}

// Theta (Eq. B6): exact MPS sums, norms from an orthogonalisation sweep.  (The overlap formula <s|s> is no use here: with
// v close to a, the residual (v - a) / h + B is a difference of terms 1 / h times larger than itself and the transfer-matrix
// contraction cancels catastrophically -- measured: a relative 4e-5 of Theta at h = 5e-5; reading 19.)
double qtt_variational_cost_impl(qtt_ctx* ctx, const View v[2], const View a[2], const View Bm[2], const MpoData* D1,
                                 const MpoData* D2, double h, double mu) {
  std::vector<const MpoData*> W{D1, D2};
  std::vector<View> X{v[0], v[1]}, ex;
  qtt_expand_apply_batch(ctx, W, X, ex);
  std::vector<std::vector<std::pair<double, View>>> terms;
  terms.push_back({{1.0, ex[0]}, {1.0, ex[1]}});
  for (int i = 0; i < 2; ++i) terms.push_back({{1.0 / h, v[i]}, {-1.0 / h, a[i]}, {1.0, Bm[i]}});
  std::vector<View> s;
  qtt_concat_batch(ctx, terms, s);
  const int n = s[0].n;
  const int big = 1 << 30;
  std::vector<OutMps> outs(3);
  for (int t = 0; t < 3; ++t) {
    outs[t].n = n;
    outs[t].rcap = qtt_round_caps(s[t].r, big);
    outs[t].core.resize(n);
    for (int k = 0; k < n; ++k) outs[t].core[k] = ctx->arena.keep((size_t)outs[t].rcap[k] * 4 * outs[t].rcap[k + 1]);
  }
  SigmaCapture sc;
  qtt_round_dense_batch(ctx, s, big, 0.0, outs, &sc);
  double nrm2[3];
  for (int t = 0; t < 3; ++t) {
    const int c = sc.count[t][n - 1];
    std::vector<double> sv(c);
    QTT_CU(cudaMemcpyAsync(sv.data(), sc.sigma[t][n - 1], sizeof(double) * c, cudaMemcpyDeviceToHost, ctx->stream));
    QTT_CU(cudaStreamSynchronize(ctx->stream));
    double acc = 0.0;
    for (int i = c - 1; i >= 0; --i) acc += sv[i] * sv[i];
    nrm2[t] = acc;
  }
  return mu * nrm2[0] + nrm2[1] + nrm2[2];
}
