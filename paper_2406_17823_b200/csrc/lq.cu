// Batched Q-less LQ factorisation by blocked Householder reflections acting on contiguous ROWS
// (the L->R orthogonalisation sweep; row a6: the zip-up factorisation).
//
//   Y (k x m, k <= m)  =  L * Q,   Q never formed; only the triangular factor is kept.
//
// Panel factorisation: one thread-block cluster per matrix.  The NB panel rows are cut into column
// slices, one per CTA, resident in shared memory; per reflector ONE cluster-wide exchange carries all
// the inner products the step needs (row j against rows j..NB-1, plus the pivot column), reduced with
// warp shuffles inside a CTA and all-to-all through distributed shared memory between CTAs.
// Trailing update: a separate grid, one warp per pair of rows, Y2 <- Y2 - (Y2 V^T) (T V), compact WY.
#include <cooperative_groups.h>
#include <cstring>
#include <vector>

#include "common.cuh"
namespace cg = cooperative_groups;

namespace {

constexpr int NB = QTT_LQ_NB;
constexpr int PANEL_NT = 256;
constexpr int MAXC = 16;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// dynamic shared memory layout (doubles):
//   Ps   [NB][wp]          panel slice
//   msg  [2][MAXC][2*NB]   per-reflector exchange (double buffered)
//   smsg [MAXC][NB*NB]     V V^T exchange
//   st   [NB*NB]           staging / totals
//   tot  [2*NB], S[NB*NB], T[NB*NB], tau[NB], beta[NB], scl[NB]
__global__ void __launch_bounds__(PANEL_NT) qtt_lq_panel_kernel(const __grid_constant__ LqGroup g, int wp) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = cluster.num_blocks();
  const int rank = cluster.block_rank();
  const LqProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = PANEL_NT / 32;

  extern __shared__ __align__(16) double sm[];
  double* Ps = sm;
  double* msg = Ps + NB * wp;
  double* smsg = msg + 2 * MAXC * 2 * NB;
  double* st = smsg + MAXC * NB * NB;
  double* tot = st + NB * NB;
  double* S = tot + 2 * NB;
  double* T = S + NB * NB;
  double* tau = T + NB * NB;
  double* beta = tau + NB;
  double* scl = beta + NB;

  const int p0 = g.p0;
  const int k = P.k, m = P.m, ld = P.ld;
  const int nbp = (p0 < k) ? min(NB, k - p0) : 0;  // uniform over the cluster
  const int mw = m - p0;
  int w = (mw + C - 1) / C;
  w = (w + 1) & ~1;
  const int cs = p0 + rank * w;
  const int wc = max(0, min(m, cs + w) - cs);

  for (int idx = tid; idx < nbp * wc; idx += PANEL_NT) {
    int j = idx / wc, x = idx - j * wc;
    Ps[j * wp + x] = P.Y[(i64)(p0 + j) * ld + cs + x];
  }
  __syncthreads();

  for (int j = 0; j < nbp; ++j) {
    const int par = j & 1;
    const int colj = p0 + j;
    const int xj = max(0, colj - cs);
    // partial inner products of row j with rows j..nbp-1 over this slice's tail columns
    for (int i = j + warp; i < nbp; i += NW) {
      double s = 0.0;
#pragma unroll 4
      for (int x = xj + lane; x < wc; x += 32) s += Ps[j * wp + x] * Ps[i * wp + x];
      s = warp_sum(s);
      if (lane == 0) {
        st[i] = s;
        st[NB + i] = (colj >= cs && colj < cs + wc) ? Ps[i * wp + (colj - cs)] : 0.0;
      }
    }
    __syncthreads();
    for (int t = tid; t < C * 2 * NB; t += PANEL_NT) {
      int dst = t / (2 * NB), idx = t - dst * (2 * NB);
      int i = idx < NB ? idx : idx - NB;
      if (i >= j && i < nbp) {
        double* remote = cluster.map_shared_rank(msg, dst);
        remote[(par * MAXC + rank) * 2 * NB + idx] = st[idx];
      }
    }
    cluster.sync();
    if (tid < 2 * NB) {
      int i = tid < NB ? tid : tid - NB;
      double s = 0.0;
      if (i >= j && i < nbp)
        for (int src = 0; src < C; ++src) s += msg[(par * MAXC + src) * 2 * NB + tid];
      tot[tid] = s;
    }
    __syncthreads();
    const double gjj = tot[j], yjj = tot[NB + j];
    double bet = 0.0, ta = 0.0, sc = 0.0;
    if (gjj > 0.0) {
      bet = -copysign(sqrt(gjj), yjj);
      ta = (bet - yjj) / bet;
      sc = 1.0 / (yjj - bet);
    } else {
      bet = yjj;
    }
    if (tid == 0) {
      tau[j] = ta;
      beta[j] = bet;
      scl[j] = sc;
    }
    if (ta != 0.0) {
      for (int i = j + 1 + warp; i < nbp; i += NW) {
        const double gji = tot[i], yij = tot[NB + i];
        const double si = yij + sc * (gji - yjj * yij);  // v_j . y_i
        const double f = ta * si;
        const double fs = f * sc;
#pragma unroll 4
        for (int x = xj + lane; x < wc; x += 32) {
          int col = cs + x;
          if (col == colj)
            Ps[i * wp + x] -= f;
          else
            Ps[i * wp + x] -= fs * Ps[j * wp + x];
        }
      }
    }
    __syncthreads();
  }

  // ---- write the L part of the panel rows, then turn Ps into clean reflector rows V
  for (int idx = tid; idx < nbp * wc; idx += PANEL_NT) {
    int j = idx / wc, x = idx - j * wc;
    int col = cs + x, colj = p0 + j;
    double v = Ps[j * wp + x];
    double vv;
    if (col < colj) {
      P.Y[(i64)(p0 + j) * ld + col] = v;
      vv = 0.0;
    } else if (col == colj) {
      P.Y[(i64)(p0 + j) * ld + col] = beta[j];
      vv = 1.0;
    } else {
      vv = v * scl[j];
    }
    Ps[j * wp + x] = vv;
  }
  __syncthreads();
  // ---- S = V V^T (strict upper part), exchanged once
  for (int pr = warp; pr < NB * NB; pr += NW) {
    int a = pr / NB, b = pr - a * NB;
    if (a < b && b < nbp) {
      double s = 0.0;
#pragma unroll 4
      for (int x = lane; x < wc; x += 32) s += Ps[a * wp + x] * Ps[b * wp + x];
      s = warp_sum(s);
      if (lane == 0) st[pr] = s;
    } else if (lane == 0) {
      st[pr] = 0.0;
    }
  }
  __syncthreads();
  for (int t = tid; t < C * NB * NB; t += PANEL_NT) {
    int dst = t / (NB * NB), idx = t - dst * (NB * NB);
    double* remote = cluster.map_shared_rank(smsg, dst);
    remote[rank * NB * NB + idx] = st[idx];
  }
  cluster.sync();
  for (int idx = tid; idx < NB * NB; idx += PANEL_NT) {
    double s = 0.0;
    for (int src = 0; src < C; ++src) s += smsg[src * NB * NB + idx];
    S[idx] = s;
    T[idx] = 0.0;
  }
  __syncthreads();
  // ---- T (upper triangular, forward product H_0 H_1 ... = I - V^T T V for row vectors)
  if (warp == 0) {
    for (int j = 0; j < nbp; ++j) {
      if (lane < j) {
        double s = 0.0;
        for (int l = lane; l < j; ++l) s += T[lane * NB + l] * S[l * NB + j];
        T[lane * NB + j] = -tau[j] * s;
      } else if (lane == j) {
        T[j * NB + j] = tau[j];
      }
      __syncwarp();
    }
  }
  __syncthreads();
  // ---- publish V and T V for the trailing update
  for (int idx = tid; idx < nbp * wc; idx += PANEL_NT) {
    int i = idx / wc, x = idx - i * wc;
    double s = 0.0;
    for (int l = i; l < nbp; ++l) s += T[i * NB + l] * Ps[l * wp + x];
    P.V[(i64)i * m + cs + x] = Ps[i * wp + x];
    P.TV[(i64)i * m + cs + x] = s;
  }
}

// W[0..n) <- sum_z W[z * n + ..): the K-chunks of the skinny first product of the trailing update, fixed order
struct SumProb { double* W; int n, Z; };
struct SumGroup { int nprob; SumProb p[QTT_LQ_MAX_BATCH]; };
__global__ void qtt_sum_partials_kernel(const __grid_constant__ SumGroup g) {
  const SumProb& P = g.p[blockIdx.y];
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= P.n || P.Z <= 1) return;
  double s = P.W[idx];
  for (int z = 1; z < P.Z; ++z) s += P.W[(i64)z * P.n + idx];
  P.W[idx] = s;
}

__global__ void qtt_extract_tri_kernel(const __grid_constant__ TriGroup g) {
  const TriProb& P = g.p[blockIdx.y];
  const i64 n = (i64)P.k * P.k;
  for (i64 idx = (i64)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (i64)gridDim.x * blockDim.x) {
    int i = (int)(idx / P.k), j = (int)(idx - (i64)i * P.k);
    double v;
    if (g.mode == 0)  // R = L^T: R[i][j] = L[j][i], j >= i
      v = (j >= i) ? P.Y[(i64)j * P.ld + i] : 0.0;
    else
      v = (j <= i) ? P.Y[(i64)i * P.ld + j] : 0.0;
    P.dst[(i64)i * P.ldr + j] = v;
  }
}

size_t panel_smem_doubles(int wp) {
  return (size_t)NB * wp + 2 * MAXC * 2 * NB + (size_t)MAXC * NB * NB + NB * NB + 2 * NB + 2 * NB * NB + 3 * NB;
}

int pick_cluster(int mw) {
  // slices of ~256 columns per CTA (measured: 80 us per 16-row panel of 4096 columns with 16 CTAs, 95 us with 8)
  int c = 1;
  while (c < MAXC && (mw + c - 1) / c > 256) c *= 2;
  return c;
}

}  // namespace


namespace {

// One target of a compact-WY update  X <- X - (X V^T)(TV)  over the columns [col0, m):  X is rows x mw (ld), V and TV
// are nv x mw (leading dimension m), W is scratch for the rows x nv product and its K-chunk partials.
struct UpdTarget {
  double* X;
  i64 ld;
  int rows;
  const double* V;
  const double* TV;
  int m, nv, mw;
  double* W;
  i64 wcap;  // doubles available at W
};

// Grouped DMMA GEMMs.  The first product is skinny (nv <= 64 columns) with a long contraction (the row length): it
// is cut into up to 8 K-chunks (one GEMM problem each, so that enough CTAs work on it), whose partial results a small
// kernel adds up in a fixed order.
cudaError_t apply_updates(const std::vector<UpdTarget>& ts, cudaStream_t stream) {
  if (ts.empty()) return cudaSuccess;
  std::vector<GemmProb> g1, g2;
  std::vector<SumProb> sums;
  for (const UpdTarget& t : ts) {
    if (t.rows <= 0 || t.nv <= 0 || t.mw <= 0) continue;
    int Z = t.mw / 512;
    Z = Z > 8 ? 8 : Z;
    const i64 per = (i64)t.rows * t.nv;
    if ((i64)Z * per > t.wcap) Z = (int)(t.wcap / per);
    Z = Z < 1 ? 1 : Z;
    int chunk = (t.mw + Z - 1) / Z;
    chunk = (chunk + 15) & ~15;
    int zused = 0;
    for (int z = 0; z < Z; ++z) {
      const int k0 = z * chunk, kz = (t.mw - k0 < chunk) ? t.mw - k0 : chunk;
      if (kz <= 0) break;
      GemmProb a;
      memset(&a, 0, sizeof(a));
      a.nbatch = 1;
      a.alpha = 1.0; a.beta = 0.0;
      a.A = t.X + k0; a.a_lo = t.ld; a.a_k = 1;
      a.B = t.V + k0; a.b_k = 1; a.b_n = t.m;
      a.C = t.W + (i64)z * per; a.c_lo = t.nv; a.c_n = 1;
      a.M = t.rows; a.N = t.nv; a.K = kz;
      g1.push_back(a);
      ++zused;
    }
    sums.push_back(SumProb{t.W, (int)per, zused});
    GemmProb b;
    memset(&b, 0, sizeof(b));
    b.nbatch = 1;
    b.alpha = -1.0; b.beta = 1.0;
    b.A = t.W; b.a_lo = t.nv; b.a_k = 1;
    b.B = t.TV; b.b_k = t.m; b.b_n = 1;
    b.C = t.X; b.c_lo = t.ld; b.c_n = 1;
    b.M = t.rows; b.N = t.mw; b.K = t.nv;
    g2.push_back(b);
  }
  if (g2.empty()) return cudaSuccess;
  QTT_CHECK_CUDA(qtt_launch_gemm(g1.data(), (int)g1.size(), stream, QK_LQ_UPDATE));
  for (size_t s0 = 0; s0 < sums.size(); s0 += QTT_LQ_MAX_BATCH) {
    SumGroup sg;
    sg.nprob = 0;
    bool any = false;
    int nmax = 0;
    for (size_t i = s0; i < sums.size() && sg.nprob < QTT_LQ_MAX_BATCH; ++i) {
      sg.p[sg.nprob++] = sums[i];
      any = any || sums[i].Z > 1;
      nmax = sums[i].n > nmax ? sums[i].n : nmax;
    }
    if (any) {
      QttProf prof(QK_LQ_UPDATE, stream, 0.0, 0, 0, sg.nprob, -1);
      qtt_sum_partials_kernel<<<dim3((nmax + 255) / 256, sg.nprob), 256, 0, stream>>>(sg);
      QTT_CHECK_CUDA(cudaGetLastError());
    }
  }
  return qtt_launch_gemm(g2.data(), (int)g2.size(), stream, QK_LQ_UPDATE);
}

constexpr int NS_MAX = 4;          // sub-panels per super-panel (scratch is sized for this)
constexpr int SP_MAX = NS_MAX * NB;

}  // namespace

size_t qtt_lq_scratch_doubles(int m) { return (size_t)SP_MAX * m; }

// Two-level blocking.  A super-panel is 4 sub-panels of 16 rows.  After each sub-panel (panel kernel: reflector rows
// V_s and T_s V_s) only the rest of the super-panel is updated -- and the rows A = T_agg V_agg accumulated so far, which
// transform exactly like trailing rows: (I - V_1..k^T A_k)(I - V_{k+1}^T TV_{k+1}) = I - V_1..k+1^T [A_k Q_{k+1}; TV_{k+1}].
// The rows below the super-panel then get ONE update with 64 reflectors, so the big trailing matrix (0.5 GB per operand
// at chi = 128: HBM-bound) is streamed once per 64 rows instead of once per 16.  Batches that fit the L2 (config 3: 67 MB)
// keep one-level blocking: there the extra small updates cost more than the saved passes.
cudaError_t qtt_launch_lq(const LqProb* probs, int n, cudaStream_t stream) {
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_lq_panel_kernel))) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_lq_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_lq_panel_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  }
  for (int b0 = 0; b0 < n; b0 += QTT_LQ_MAX_BATCH) {
    const int nb = n - b0 < QTT_LQ_MAX_BATCH ? n - b0 : QTT_LQ_MAX_BATCH;
    int kmax = 0;
    double bytes = 0.0;
    for (int i = 0; i < nb; ++i) {
      if (probs[b0 + i].k > probs[b0 + i].m) return cudaErrorInvalidValue;
      kmax = probs[b0 + i].k > kmax ? probs[b0 + i].k : kmax;
      bytes += (double)probs[b0 + i].k * probs[b0 + i].m * sizeof(double);
    }
    const int NS = bytes > 96e6 ? NS_MAX : 1;
    const int SP = NS * NB;
    for (int P0 = 0; P0 < kmax; P0 += SP) {
      // the reflector rows of a sub-panel start at its own first column: zero what lies before it inside the super-panel
      for (int i = 0; i < nb && NS > 1; ++i) {
        const LqProb& p = probs[b0 + i];
        if (p.k <= P0) continue;
        const size_t wbytes = (size_t)((p.m - P0 < SP) ? p.m - P0 : SP) * sizeof(double);
        QTT_CHECK_CUDA(cudaMemset2DAsync(p.V + P0, (size_t)p.m * sizeof(double), 0, wbytes, SP, stream));
        QTT_CHECK_CUDA(cudaMemset2DAsync(p.TV + P0, (size_t)p.m * sizeof(double), 0, wbytes, SP, stream));
      }
      for (int s = 0; s < NS; ++s) {
        const int p0 = P0 + s * NB;
        if (p0 >= kmax) break;
        LqGroup grp;
        grp.nprob = 0;
        grp.p0 = p0;
        int mwmax = 0;
        std::vector<UpdTarget> small;
        double fp = 0.0;
        for (int i = 0; i < nb; ++i) {
          const LqProb& p = probs[b0 + i];
          if (p.k <= p0) continue;
          LqProb q = p;
          q.V = p.V + (size_t)s * NB * p.m;
          q.TV = p.TV + (size_t)s * NB * p.m;
          grp.p[grp.nprob++] = q;
          const int mw = p.m - p0, nbp = (p.k - p0 < NB) ? p.k - p0 : NB;
          mwmax = mw > mwmax ? mw : mwmax;
          fp += 2.0 * nbp * nbp * (double)mw;
          const int pend = (P0 + SP < p.k) ? P0 + SP : p.k;
          const int r0 = p0 + nbp;
          const i64 half = (i64)SP_MAX * p.m / 2;
          if (pend > r0)  // the rest of the super-panel
            small.push_back(UpdTarget{p.Y + (i64)r0 * p.ld + p0, p.ld, pend - r0, q.V + p0, q.TV + p0, p.m, nbp, mw, p.W, half});
          if (s > 0 && p.k > pend)  // the accumulated T V rows (only needed if rows remain below the super-panel)
            small.push_back(UpdTarget{p.TV + p0, p.m, s * NB, q.V + p0, q.TV + p0, p.m, nbp, mw, p.W + half, half});
        }
        if (grp.nprob == 0) break;
        const int C = pick_cluster(mwmax);
        int w = (mwmax + C - 1) / C;
        w = (w + 1) & ~1;
        const int wp = w + 1;
        const size_t smem = panel_smem_doubles(wp) * sizeof(double);
        if (smem > 200 * 1024) return cudaErrorInvalidConfiguration;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(C * grp.nprob);
        cfg.blockDim = dim3(PANEL_NT);
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
          QttProf prof(QK_LQ_PANEL, stream, fp, grp.p[0].k, grp.p[0].m, grp.nprob, p0);
          QTT_CHECK_CUDA(cudaLaunchKernelEx(&cfg, qtt_lq_panel_kernel, grp, wp));
        }
        QTT_CHECK_CUDA(apply_updates(small, stream));
      }
      // ---- the rows below the super-panel: one update with all its reflectors
      std::vector<UpdTarget> big;
      for (int i = 0; i < nb; ++i) {
        const LqProb& p = probs[b0 + i];
        const int pend = (P0 + SP < p.k) ? P0 + SP : p.k;
        if (p.k <= P0 || p.k <= pend) continue;
        big.push_back(UpdTarget{p.Y + (i64)pend * p.ld + P0, p.ld, p.k - pend, p.V + P0, p.TV + P0, p.m, pend - P0, p.m - P0,
                                p.W, (i64)SP_MAX * p.m});
      }
      QTT_CHECK_CUDA(apply_updates(big, stream));
    }
  }
  return cudaSuccess;
}

cudaError_t qtt_launch_extract_tri(const TriProb* probs, int n, int mode, cudaStream_t stream) {
  for (int b0 = 0; b0 < n; b0 += QTT_LQ_MAX_BATCH) {
    TriGroup g;
    g.nprob = n - b0 < QTT_LQ_MAX_BATCH ? n - b0 : QTT_LQ_MAX_BATCH;
    g.mode = mode;
    int kmax = 1;
    for (int i = 0; i < g.nprob; ++i) {
      g.p[i] = probs[b0 + i];
      kmax = g.p[i].k > kmax ? g.p[i].k : kmax;
    }
    int bx = (int)(((i64)kmax * kmax + 255) / 256);
    bx = bx > 256 ? 256 : bx;
    {
      QttProf prof(QK_MOVE, stream, 16.0 * kmax * kmax * g.nprob);
      qtt_extract_tri_kernel<<<dim3(bx, g.nprob), 256, 0, stream>>>(g);
    }
    QTT_CHECK_CUDA(cudaGetLastError());
  }
  return cudaSuccess;
}
