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

// Problems that still have rows below the current panel (their trailing update is done by grouped GEMMs).

struct UpdGroup {
  int nprob, p0;
  LqProb p[QTT_LQ_MAX_BATCH];
};

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

size_t qtt_lq_scratch_doubles(int m) { return (size_t)NB * m; }

cudaError_t qtt_launch_lq(const LqProb* probs, int n, cudaStream_t stream) {
  static bool attr_done = false;
  if (!attr_done) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_lq_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_lq_panel_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    attr_done = true;
  }
  for (int b0 = 0; b0 < n; b0 += QTT_LQ_MAX_BATCH) {
    int nb = n - b0 < QTT_LQ_MAX_BATCH ? n - b0 : QTT_LQ_MAX_BATCH;
    int kmax = 0;
    for (int i = 0; i < nb; ++i) {
      if (probs[b0 + i].k > probs[b0 + i].m) return cudaErrorInvalidValue;
      kmax = probs[b0 + i].k > kmax ? probs[b0 + i].k : kmax;
    }
    for (int p0 = 0; p0 < kmax; p0 += NB) {
      LqGroup grp;
      UpdGroup ug;
      grp.nprob = 0;
      grp.p0 = p0;
      ug.nprob = 0;
      ug.p0 = p0;
      int mwmax = 0, ctas = 0;
      for (int i = 0; i < nb; ++i) {
        const LqProb& p = probs[b0 + i];
        if (p.k <= p0) continue;
        grp.p[grp.nprob++] = p;
        mwmax = (p.m - p0) > mwmax ? (p.m - p0) : mwmax;
        int rem = p.k - (p0 + (p.k - p0 < NB ? p.k - p0 : NB));
        if (rem > 0) {
          ug.p[ug.nprob++] = p;
          ctas += 1;
        }
      }
      if (grp.nprob == 0) break;
      int C = pick_cluster(mwmax);
      int w = (mwmax + C - 1) / C;
      w = (w + 1) & ~1;
      int wp = w + 1;
      size_t smem = panel_smem_doubles(wp) * sizeof(double);
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
      // Householder count of this panel step: panel 2 nb^2 mw, trailing update 4 nb mw rows_below
      double fp = 0.0, fu = 0.0;
      for (int i = 0; i < grp.nprob; ++i) {
        const double mw = grp.p[i].m - p0, nbp = (grp.p[i].k - p0 < NB) ? grp.p[i].k - p0 : NB;
        fp += 2.0 * nbp * nbp * mw;
        fu += 4.0 * nbp * mw * (grp.p[i].k - p0 - nbp);
      }
      {
        QttProf prof(QK_LQ_PANEL, stream, fp, grp.p[0].k, grp.p[0].m, grp.nprob, p0);
        QTT_CHECK_CUDA(cudaLaunchKernelEx(&cfg, qtt_lq_panel_kernel, grp, wp));
      }
      if (ctas > 0) {
        // trailing update of the rows below the panel, Y2 <- Y2 - (Y2 V^T)(T V), as grouped DMMA GEMMs.  The first
        // product is skinny (16 columns) with a long contraction (the row length): it is cut into up to 8 K-chunks
        // (one GEMM problem each, so that enough CTAs work on it), whose partial results a small kernel adds up in
        // a fixed order.
        std::vector<GemmProb> g1;
        GemmProb g2[QTT_LQ_MAX_BATCH];
        SumGroup sg;
        sg.nprob = 0;
        for (int i = 0; i < ug.nprob; ++i) {
          const LqProb& p = ug.p[i];
          const int nbp = (p.k - p0 < NB) ? p.k - p0 : NB;
          const int r0 = p0 + nbp, rem = p.k - r0, mw = p.m - p0;
          int Z = mw / 512;
          Z = Z > 8 ? 8 : Z;
          if (Z > p.m / rem) Z = p.m / rem;  // the partials live in the NB x m scratch W
          Z = Z < 1 ? 1 : Z;
          int chunk = (mw + Z - 1) / Z;
          chunk = (chunk + 15) & ~15;
          for (int z = 0; z < Z; ++z) {
            const int k0 = z * chunk, kz = (mw - k0 < chunk) ? mw - k0 : chunk;
            GemmProb a;
            memset(&a, 0, sizeof(a));
            a.nbatch = 1;
            a.alpha = 1.0; a.beta = 0.0;
            a.A = p.Y + (i64)r0 * p.ld + p0 + k0; a.a_lo = p.ld; a.a_k = 1;
            a.B = p.V + p0 + k0; a.b_k = 1; a.b_n = p.m;
            a.C = p.W + (i64)z * rem * NB; a.c_lo = NB; a.c_n = 1;
            a.M = rem; a.N = nbp; a.K = kz > 0 ? kz : 0;
            if (a.K > 0) g1.push_back(a);
            else {  // (cannot happen with chunk >= 16, kept for safety: an empty chunk contributes zeros)
              Z = z;
              break;
            }
          }
          sg.p[sg.nprob].W = p.W;
          sg.p[sg.nprob].n = rem * NB;
          sg.p[sg.nprob].Z = Z;
          ++sg.nprob;
          GemmProb b;
          memset(&b, 0, sizeof(b));
          b.nbatch = 1;
          b.alpha = -1.0; b.beta = 1.0;
          b.A = p.W; b.a_lo = NB; b.a_k = 1;
          b.B = p.TV + p0; b.b_k = p.m; b.b_n = 1;
          b.C = p.Y + (i64)r0 * p.ld + p0; b.c_lo = p.ld; b.c_n = 1;
          b.M = rem; b.N = mw; b.K = nbp;
          g2[i] = b;
        }
        QTT_CHECK_CUDA(qtt_launch_gemm(g1.data(), (int)g1.size(), stream, QK_LQ_UPDATE));
        {
          bool any = false;
          int nmax = 0;
          for (int i = 0; i < sg.nprob; ++i) {
            any = any || sg.p[i].Z > 1;
            nmax = sg.p[i].n > nmax ? sg.p[i].n : nmax;
          }
          if (any) {
            QttProf prof(QK_LQ_UPDATE, stream, 0.0, 0, 0, sg.nprob, -1);
            qtt_sum_partials_kernel<<<dim3((nmax + 255) / 256, sg.nprob), 256, 0, stream>>>(sg);
            QTT_CHECK_CUDA(cudaGetLastError());
          }
        }
        QTT_CHECK_CUDA(qtt_launch_gemm(g2, ug.nprob, stream, QK_LQ_UPDATE));
        (void)fu;
      }
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
