// Rank-revealing preconditioner of the row-Jacobi SVD:
// Householder QR with column pivoting, in place,
//
//   X (p x q)  <-  Q^T X,      Q orthogonal (p x p), never formed.
//
// Left multiplication keeps the row space, so the right singular vectors and the singular values of X are
// unchanged (they are what the truncated-SVD step of the rounding sweep needs), but the rows of the result
// are graded like the singular values: row j is what is left of the largest remaining column after j
// reflections.  One-sided Jacobi on such rows converges in 7-9 sweeps instead of 20-45 on the raw site
// matrices (the scaled Gram matrix of the rows is well conditioned; this is the Drmac-Veselic
// preconditioning).  Columns are NOT physically permuted -- the Jacobi dot products do not care about the
// column order -- so the singular vectors come out in the original column order.
//
// The factorisation stops when the largest remaining column norm is below 8 eps ||X||_F: the rows from there
// on are rounding noise of an (exactly or numerically) rank-deficient matrix -- MPO-expanded and direct-sum
// cores are rank-deficient by construction -- and are written out as exact zeros.  The number of non-zero rows
// (the numerical rank) goes to rank_out, and the Jacobi kernel only rotates that many rows.
//
// One thread-block cluster per matrix.  The columns are cut into slices, one per CTA, resident in shared
// memory column-major, so a reflector needs no cross-CTA reduction: per step ONE cluster barrier carries the
// pivot candidates; every CTA then pulls the pivot column from its owner through distributed shared memory and
// derives the (bit-identical) reflector itself.
#include <cooperative_groups.h>

#include "common.cuh"
namespace cg = cooperative_groups;

namespace {

constexpr int QNT = 512;
constexpr int QNW = QNT / 32;
constexpr int MAXC = 16;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// dynamic shared memory (doubles): Xs [w][pp] | vb [pp] | red [QNW] | wval [QNW] | candv [2][MAXC] | nrm [w]
//                                  | diag [w] | xfro [MAXC] || ints: wcol [QNW] | candc [2][MAXC] | stepidx [w]
__global__ void __launch_bounds__(QNT) qtt_qrcp_kernel(const __grid_constant__ QrcpGroup g) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = g.cluster;
  const int rank = (C > 1) ? (int)cluster.block_rank() : 0;
  const QrcpProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int p = P.p, q = P.q;
  const int w = g.w, pp = g.pp;

  extern __shared__ __align__(16) double sm[];
  double* Xs = sm;
  double* vb = Xs + (size_t)w * pp;
  double* red = vb + pp;
  double* wval = red + QNW;
  double* candv = wval + QNW;
  double* nrm = candv + 2 * MAXC;
  double* diag = nrm + w;
  double* xfro = diag + w;
  int* wcol = reinterpret_cast<int*>(xfro + MAXC);
  int* candc = wcol + QNW;
  int* stepidx = candc + 2 * MAXC;

  // this CTA's columns: [cs, cs + wc); per-problem slice width so that small problems spread over the cluster too
  const int wq = (q + C - 1) / C;
  const int cs = rank * wq;
  const int wc = max(0, min(q, cs + wq) - cs);

  for (int idx = tid; idx < p * wc; idx += QNT) {
    const int r = idx / wc, x = idx - r * wc;
    Xs[(size_t)x * pp + r] = P.X[(i64)r * P.ld + cs + x];
  }
  __syncthreads();
  // column norms and the Frobenius norm
  double fro = 0.0;
  for (int c = warp; c < wc; c += QNW) {
    double s = 0.0;
    for (int i = lane; i < p; i += 32) {
      const double v = Xs[(size_t)c * pp + i];
      s += v * v;
    }
    s = warp_sum(s);
    if (lane == 0) {
      nrm[c] = s;
      stepidx[c] = -1;
      diag[c] = 0.0;
    }
    fro += s;
  }
  if (lane == 0) red[warp] = fro;
  __syncthreads();
  if (tid == 0) {
    double s = 0.0;
    for (int i = 0; i < QNW; ++i) s += red[i];
    red[0] = s;
  }
  __syncthreads();
  const double myfro = red[0];
  __syncthreads();
  if (C > 1) {
    if (tid < C) {
      double* remote = cluster.map_shared_rank(xfro, tid);
      remote[rank] = myfro;
    }
    cluster.sync();
  } else if (tid == 0) {
    xfro[0] = myfro;
  }
  __syncthreads();
  double fro2 = 0.0;
  for (int c2 = 0; c2 < C; ++c2) fro2 += xfro[c2];
  // (8 eps)^2 ||X||_F^2
  const double thresh2 = 3.1554436208840472e-30 * fro2;

  const int rmax = min(p, q);
  int nsteps = 0;
  for (int j = 0; j < rmax; ++j) {
    const int par = j & 1;
    // ---- pivot candidate of this CTA
    {
      double bv = -1.0;
      int bc = 0x7fffffff;
      for (int c = warp; c < wc; c += QNW) {
        const double v = (stepidx[c] < 0) ? nrm[c] : -1.0;
        if (v > bv) {
          bv = v;
          bc = cs + c;
        }
      }
      if (lane == 0) {
        wval[warp] = bv;
        wcol[warp] = bc;
      }
    }
    __syncthreads();
    double gval = -1.0;
    int gcol = 0x7fffffff;
    if (C > 1) {
      if (tid < C) {
        double bv = -1.0;
        int bc = 0x7fffffff;
        for (int i = 0; i < QNW; ++i)
          if (wval[i] > bv || (wval[i] == bv && wcol[i] < bc)) {
            bv = wval[i];
            bc = wcol[i];
          }
        double* rv = cluster.map_shared_rank(candv, tid);
        int* rc = cluster.map_shared_rank(candc, tid);
        rv[par * MAXC + rank] = bv;
        rc[par * MAXC + rank] = bc;
      }
      cluster.sync();
      for (int i = 0; i < C; ++i) {
        const double v = candv[par * MAXC + i];
        const int c = candc[par * MAXC + i];
        if (v > gval || (v == gval && c < gcol)) {
          gval = v;
          gcol = c;
        }
      }
    } else {
      for (int i = 0; i < QNW; ++i)
        if (wval[i] > gval || (wval[i] == gval && wcol[i] < gcol)) {
          gval = wval[i];
          gcol = wcol[i];
        }
    }
    if (!(gval > thresh2)) break;  // what is left is rounding noise (uniform over the cluster)
    nsteps = j + 1;
    // ---- pull the pivot column (rows j..p-1) from its owner
    const int owner = gcol / wq, lc = gcol - owner * wq;
    {
      const double* src = (C > 1) ? cluster.map_shared_rank(Xs + (size_t)lc * pp, owner) : Xs + (size_t)lc * pp;
      for (int i = j + tid; i < p; i += QNT) vb[i] = src[i];
    }
    __syncthreads();
    // ---- reflector H = I - tau v v^T, v_j = 1, v_i = x_i * scale (i > j); every CTA derives the same numbers
    {
      double s = 0.0;
      for (int i = j + 1 + tid; i < p; i += QNT) s += vb[i] * vb[i];
      s = warp_sum(s);
      if (lane == 0) red[warp] = s;
    }
    __syncthreads();
    double sigma = 0.0;
#pragma unroll
    for (int i = 0; i < QNW; ++i) sigma += red[i];
    const double alpha = vb[j];
    double beta = alpha, tau = 0.0, scale = 0.0;
    if (sigma > 0.0) {
      beta = -copysign(sqrt(alpha * alpha + sigma), alpha);
      tau = (beta - alpha) / beta;
      scale = 1.0 / (alpha - beta);
    }
    if (rank == owner && tid == 0) {
      diag[lc] = beta;
      stepidx[lc] = j;
    }
    // ---- apply to the remaining columns of this slice; new norms over rows > j
    for (int c = warp; c < wc; c += QNW) {
      if (stepidx[c] >= 0 || (rank == owner && c == lc)) continue;
      double* col = Xs + (size_t)c * pp;
      double dot = 0.0;
      for (int i = j + lane; i < p; i += 32) {
        const double v = (i == j) ? 1.0 : vb[i] * scale;
        dot += v * col[i];
      }
      dot = warp_sum(dot) * tau;
      double nn = 0.0;
      for (int i = j + lane; i < p; i += 32) {
        const double v = (i == j) ? 1.0 : vb[i] * scale;
        const double x = col[i] - dot * v;
        col[i] = x;
        if (i > j) nn += x * x;
      }
      nn = warp_sum(nn);
      if (lane == 0) nrm[c] = nn;
    }
    __syncthreads();
  }
  __syncthreads();
  // ---- write out Q^T X: rows >= nsteps are zero; a column pivoted at step s is (R entries, beta, zeros)
  for (int idx = tid; idx < p * wc; idx += QNT) {
    const int r = idx / wc, x = idx - r * wc;
    const int s = stepidx[x];
    double v = 0.0;
    if (r < nsteps) {
      if (s < 0 || r < s) v = Xs[(size_t)x * pp + r];
      else if (r == s) v = diag[x];
    }
    P.X[(i64)r * P.ld + cs + x] = v;
  }
  if (rank == 0 && tid == 0 && P.rank_out) P.rank_out[0] = nsteps;
  // no CTA may leave while a peer can still read its shared memory
  if (C > 1) cluster.sync();
}

size_t qrcp_smem_bytes(int w, int pp) {
  const size_t doubles = (size_t)w * pp + pp + QNW + QNW + 2 * MAXC + 2 * (size_t)w + MAXC;
  const size_t ints = QNW + 2 * MAXC + (size_t)w;
  return doubles * sizeof(double) + ints * sizeof(int) + 16;
}

}  // namespace

bool qtt_qrcp_fits(int p, int q) {
  if (p < 1 || q < 1) return false;
  int C = (q + 15) / 16;
  C = C < 1 ? 1 : (C > MAXC ? MAXC : C);
  const int w = (q + C - 1) / C;
  return qrcp_smem_bytes(w, p | 1) <= 220 * 1024;
}

cudaError_t qtt_launch_qrcp(const QrcpProb* probs, int n, cudaStream_t stream) {
  static bool attr_done = false;
  if (!attr_done) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_qrcp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_qrcp_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    attr_done = true;
  }
  for (int b0 = 0; b0 < n; b0 += QTT_QRCP_MAX_BATCH) {
    QrcpGroup g;
    g.nprob = 0;
    int pmax = 0, qmax = 0;
    double flops = 0.0;
    for (int i = b0; i < n && g.nprob < QTT_QRCP_MAX_BATCH; ++i) {
      if (probs[i].p < 1 || probs[i].q < 1) return cudaErrorInvalidValue;
      g.p[g.nprob++] = probs[i];
      pmax = probs[i].p > pmax ? probs[i].p : pmax;
      qmax = probs[i].q > qmax ? probs[i].q : qmax;
      const double a = probs[i].p, b = probs[i].q, r = a < b ? a : b;
      flops += 4.0 * a * b * r - 2.0 * (a + b) * r * r + (4.0 / 3.0) * r * r * r;  // Householder QR count
    }
    int C = (qmax + 15) / 16;
    C = C < 1 ? 1 : (C > MAXC ? MAXC : C);
    // cluster sizes must divide the grid; any size 1..16 is legal with the non-portable attribute, keep powers of two
    int c2 = 1;
    while (c2 < C) c2 *= 2;
    C = c2 > MAXC ? MAXC : c2;
    g.cluster = C;
    g.w = (qmax + C - 1) / C;
    g.pp = pmax | 1;
    const size_t smem = qrcp_smem_bytes(g.w, g.pp);
    if (smem > 224 * 1024) return cudaErrorInvalidConfiguration;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C * g.nprob);
    cfg.blockDim = dim3(QNT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    {
      QttProf prof(QK_QRCP, stream, flops, pmax, qmax, g.nprob, C);
      QTT_CHECK_CUDA(cudaLaunchKernelEx(&cfg, qtt_qrcp_kernel, g));
    }
  }
  return cudaSuccess;
}
