// Cluster-resident Householder QR, two uses:
//
//  (1) pivot = 1: rank-revealing preconditioner of the row-Jacobi SVD, in place,
//        X (p x q)  <-  Q^T X,      Q orthogonal (p x p), never formed.
//      Left multiplication keeps the row space, so the right singular vectors and the singular values of X
//      are unchanged (they are what the truncated-SVD step of the rounding sweep needs), but the rows of the
//      result are graded like the singular values: row j is what is left of the largest remaining column after
//      j reflections.  One-sided Jacobi on such rows converges in 6-10 sweeps instead of 20-45 on the raw site
//      matrices (the scaled Gram matrix of the rows is well conditioned; Drmac-Veselic preconditioning).
//      Columns are NOT physically permuted -- the Jacobi dot products do not care about the column order -- so
//      the singular vectors come out in the original column order.  The factorisation stops when the largest
//      remaining column norm is below 8 eps ||X||_F: the rows from there on are rounding noise of an (exactly
//      or numerically) rank-deficient matrix -- MPO-expanded and direct-sum cores are rank-deficient by
//      construction -- and are written out as exact zeros.  The number of non-zero rows (the numerical rank)
//      goes to rank_out, and the Jacobi kernel only rotates that many rows.
//
//  (2) pivot = 0: the Q-less triangular factor of the L->R orthogonalisation sweep, X = Q R, R (q x q upper
//      triangular) written to a separate array; X may be given transposed (as the k x m matrix Y = X^T whose
//      LQ factor L = R^T is wanted).
//
// One thread-block cluster per matrix.  The columns are cut into slices, one per CTA, resident in shared
// memory column-major, so a reflector needs no cross-CTA reduction: per step ONE cluster barrier (which carries
// the pivot candidates when pivoting); every CTA then pulls the pivot column from its owner through distributed
// shared memory and derives the (bit-identical) reflector itself.
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
// argmax over each group of 16 lanes of (val, col): larger val wins, ties go to the smaller col.  The values are
// squared norms (>= 0) or -1 for "none", handled as their bit patterns: non-negative doubles order like int64.
__device__ __forceinline__ long long norm_key(double v) { return v >= 0.0 ? __double_as_longlong(v) : -1ll; }
__device__ __forceinline__ void warp_argmax16(long long& v, int& c) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) {
    const long long ov = __shfl_xor_sync(0xffffffffu, v, o);
    const int oc = __shfl_xor_sync(0xffffffffu, c, o);
    if (ov > v || (ov == v && oc < c)) {
      v = ov;
      c = oc;
    }
  }
}

// dynamic shared memory (doubles): Xs [w][pp] | vb [pp] | red [QNW] | nrm [w] | ref [w] | diag [w] | xfro [MAXC]
//                       || 64-bit: wval [QNW] | candv [2][MAXC] || ints: wcol [QNW] | candc [2][MAXC] | stepidx [w]
// Column c of the matrix lives in CTA c % C (slot c / C): cyclic, so that the CTAs run out of columns together.
// EPL > 0: rows per lane of the register-cached update (p <= 32 * EPL); EPL = 0: any p, passes over shared memory.
template <int EPL>
__global__ void __launch_bounds__(QNT) qtt_qrcp_kernel(const __grid_constant__ QrcpGroup g) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = g.cluster;
  const int rank = (C > 1) ? (int)cluster.block_rank() : 0;
  const QrcpProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int p = P.p, q = P.q;
  const int w = g.w, pp = g.pp;
  const bool pivot = g.pivot != 0;

  extern __shared__ __align__(16) double sm[];
  double* Xs = sm;
  double* vb = Xs + (size_t)w * pp;
  double* red = vb + pp;
  double* nrm = red + QNW;
  double* ref = nrm + w;
  double* diag = ref + w;
  double* xfro = diag + w;
  long long* wval = reinterpret_cast<long long*>(xfro + MAXC);
  long long* candv = wval + QNW;
  int* wcol = reinterpret_cast<int*>(candv + 2 * MAXC);
  int* candc = wcol + QNW;
  int* stepidx = candc + 2 * MAXC;
  // staging of pivot-column chunks: [2][MAXC sources][chm rows]; CTA k stages rows [k ch, (k+1) ch)
  const int chm = g.chm;
  double* stage = reinterpret_cast<double*>(stepidx + ((w + 1) & ~1));
  const int ch = (p + C - 1) / C;

  const int wc = (q - rank + C - 1) / C;  // columns rank, rank + C, ... < q   (0 if rank >= q)

  if (P.transposed) {  // X[r][c] = Y[c * ld + r]
    for (int idx = tid; idx < p * wc; idx += QNT) {
      const int x = idx / p, r = idx - x * p;
      Xs[(size_t)x * pp + r] = P.X[(i64)(rank + C * x) * P.ld + r];
    }
  } else {
    for (int idx = tid; idx < p * wc; idx += QNT) {
      const int r = idx / wc, x = idx - r * wc;
      Xs[(size_t)x * pp + r] = P.X[(i64)r * P.ld + rank + C * x];
    }
  }
  for (int c = tid; c < wc; c += QNT) {
    stepidx[c] = -1;
    diag[c] = 0.0;
  }
  __syncthreads();
  // column norms and the Frobenius norm (pivoting only)
  double thresh2 = -1.0;
  if (pivot) {
    double fro = 0.0;
    for (int c = warp; c < wc; c += QNW) {
      double s = 0.0;
#pragma unroll 4
      for (int i = lane; i < p; i += 32) {
        const double v = Xs[(size_t)c * pp + i];
        s += v * v;
      }
      s = warp_sum(s);
      if (lane == 0) {
        nrm[c] = s;
        ref[c] = s;
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
    thresh2 = 3.1554436208840472e-30 * fro2;  // (8 eps)^2 ||X||_F^2
  }
  __syncthreads();

  const int rmax = min(p, q);
  int nsteps = 0;
  for (int j = 0; j < rmax; ++j) {
    const int par = j & 1;
    int gcol = j;  // without pivoting the columns are taken in order
    if (pivot) {
      // ---- pivot candidate of this CTA
      {
        long long bv = -1;
        int bc = 0x7fffffff;
        for (int c = warp; c < wc; c += QNW) {
          const long long v = (stepidx[c] < 0) ? norm_key(nrm[c]) : -1ll;
          if (v > bv) {
            bv = v;
            bc = rank + C * c;
          }
        }
        if (lane == 0) {
          wval[warp] = bv;
          wcol[warp] = bc;
        }
      }
      __syncthreads();
      // every warp derives the CTA's candidate; its column is staged chunk-wise in the peers BEFORE the barrier,
      // so that afterwards nobody has to pull a whole column out of one CTA (the owner's shared-memory port
      // would serialise 15 pulls)
      long long bv = wval[lane & 15];
      int bc = wcol[lane & 15];
      warp_argmax16(bv, bc);
      long long gval;
      if (C > 1) {
        if (warp == 0 && lane < C) {
          long long* rv = cluster.map_shared_rank(candv, lane);
          int* rc = cluster.map_shared_rank(candc, lane);
          rv[par * MAXC + rank] = bv;
          rc[par * MAXC + rank] = bc;
        }
        if (bv >= 0) {
          const double* col = Xs + (size_t)(bc / C) * pp;
          for (int i = j + tid; i < p; i += QNT) {
            const int k = i / ch;
            double* dst = cluster.map_shared_rank(stage, k);
            dst[(size_t)(par * MAXC + rank) * chm + (i - k * ch)] = col[i];
          }
        }
        cluster.sync();
        gval = (lane & 15) < C ? candv[par * MAXC + (lane & 15)] : -1ll;
        gcol = (lane & 15) < C ? candc[par * MAXC + (lane & 15)] : 0x7fffffff;
        warp_argmax16(gval, gcol);
      } else {
        gval = bv;
        gcol = bc;
      }
      if (gval < 0 || !(__longlong_as_double(gval) > thresh2)) break;  // what is left is rounding noise (uniform)
    } else if (C > 1) {
      if (rank == j % C) {  // the owner stages column j
        const double* col = Xs + (size_t)(j / C) * pp;
        for (int i = j + tid; i < p; i += QNT) {
          const int k = i / ch;
          double* dst = cluster.map_shared_rank(stage, k);
          dst[(size_t)(par * MAXC + rank) * chm + (i - k * ch)] = col[i];
        }
      }
      cluster.sync();
    }
    nsteps = j + 1;
    // ---- gather the pivot column (rows j..p-1) from the staged chunks; sum of squares of the rows below j on the way
    const int owner = gcol % C, lc = gcol / C;
    {
      double s = 0.0;
      if (C > 1) {
        for (int i = j + tid; i < p; i += QNT) {
          const int k = i / ch;
          const double* src = cluster.map_shared_rank(stage, k);
          const double x = src[(size_t)(par * MAXC + owner) * chm + (i - k * ch)];
          vb[i] = x;
          if (i > j) s += x * x;
        }
      } else {
        const double* src = Xs + (size_t)lc * pp;
        for (int i = j + tid; i < p; i += QNT) {
          const double x = src[i];
          vb[i] = x;
          if (i > j) s += x * x;
        }
      }
      s = warp_sum(s);
      if (lane == 0) red[warp] = s;
    }
    __syncthreads();
    // ---- reflector H = I - tau v v^T, v_j = 1, v_i = x_i * scale (i > j); every CTA derives the same numbers:
    //      nrm = sqrt(alpha^2 + sigma), beta = -sign(alpha) nrm, tau = 1 + |alpha| / nrm, scale = sign(alpha) / (|alpha| + nrm)
    double sigma = red[lane & 15];
    sigma += __shfl_xor_sync(0xffffffffu, sigma, 8);
    sigma += __shfl_xor_sync(0xffffffffu, sigma, 4);
    sigma += __shfl_xor_sync(0xffffffffu, sigma, 2);
    sigma += __shfl_xor_sync(0xffffffffu, sigma, 1);
    const double alpha = vb[j];
    double beta = alpha, tau = 0.0, scale = 0.0;
    if (sigma > 0.0) {
      const double n2 = alpha * alpha + sigma;
      double r = rsqrt(n2);
      r = r * (1.5 - 0.5 * n2 * r * r);
      double nr = n2 * r;
      nr = nr + 0.5 * r * (n2 - nr * nr);  // sqrt(n2) to full accuracy
      const double aa = fabs(alpha);
      beta = -copysign(nr, alpha);
      tau = 1.0 + aa * r;
      scale = copysign(1.0 / (aa + nr), alpha);
    }
    if (rank == owner && tid == 0) {
      diag[lc] = beta;
      stepidx[lc] = j;
    }
    // ---- apply to the remaining columns of this slice, two columns per warp at a time:
    //      dot = col[j] + scale * sum_{i>j} vb[i] col[i];  col[j] -= tau dot;  col[i] -= (tau dot scale) vb[i];
    //      squared norms over the rows > j are downdated by col[j]^2 and recomputed when they have lost 8 digits
    if (tau != 0.0 || pivot) {
      for (int c0 = warp; c0 < wc; c0 += 2 * QNW) {
        const int c1 = c0 + QNW;
        const bool on0 = stepidx[c0] < 0 && !(rank == owner && c0 == lc);
        const bool on1 = c1 < wc && stepidx[c1] < 0 && !(rank == owner && c1 == lc);
        if (!on0 && !on1) continue;
        double* col0 = Xs + (size_t)(on0 ? c0 : c1) * pp;  // (an inactive partner aliases the active one, unused)
        double* col1 = Xs + (size_t)(on1 ? c1 : c0) * pp;
        if constexpr (EPL > 0) {
          double x0[EPL], x1[EPL];
          double da = 0.0, db = 0.0, dc = 0.0, dd = 0.0;
#pragma unroll
          for (int e = 0; e < EPL; ++e) {
            const int i = lane + 32 * e;
            x0[e] = 0.0;
            x1[e] = 0.0;
            if (32 * e + 31 > j && 32 * e < p) {  // warp-uniform: rows of this slab are still live
              const bool on = i > j && i < p;
              const double v = on ? vb[i] : 0.0;
              x0[e] = on ? col0[i] : 0.0;
              x1[e] = on ? col1[i] : 0.0;
              if (e & 1) {
                db += v * x0[e];
                dd += v * x1[e];
              } else {
                da += v * x0[e];
                dc += v * x1[e];
              }
            }
          }
          double dot0 = da + db, dot1 = dc + dd;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            dot0 += __shfl_xor_sync(0xffffffffu, dot0, o);
            dot1 += __shfl_xor_sync(0xffffffffu, dot1, o);
          }
          const double cj0 = col0[j], cj1 = col1[j];
          const double d0 = (cj0 + scale * dot0) * tau, d1 = (cj1 + scale * dot1) * tau;
          const double ds0 = d0 * scale, ds1 = d1 * scale;
          const double nj0 = cj0 - d0, nj1 = cj1 - d1;
          bool re0 = false, re1 = false;
          double nn0 = 0.0, nn1 = 0.0;
          if (pivot) {
            nn0 = nrm[on0 ? c0 : c1] - nj0 * nj0;
            nn1 = nrm[on1 ? c1 : c0] - nj1 * nj1;
            re0 = !(nn0 > 1.5e-8 * ref[on0 ? c0 : c1]);
            re1 = !(nn1 > 1.5e-8 * ref[on1 ? c1 : c0]);
          }
          double s0 = 0.0, s1 = 0.0;
#pragma unroll
          for (int e = 0; e < EPL; ++e) {
            const int i = lane + 32 * e;
            if (32 * e + 31 > j && 32 * e < p) {
              const bool on = i > j && i < p;
              const double v = on ? vb[i] : 0.0;
              const double y0 = x0[e] - ds0 * v, y1 = x1[e] - ds1 * v;
              if (on && on0) col0[i] = y0;
              if (on && on1) col1[i] = y1;
              s0 += y0 * y0;
              s1 += y1 * y1;
            }
          }
          if (lane == 0) {
            if (on0) col0[j] = nj0;
            if (on1) col1[j] = nj1;
          }
          if (pivot) {
            if (re0 || re1) {  // warp-uniform
#pragma unroll
              for (int o = 16; o > 0; o >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, o);
                s1 += __shfl_xor_sync(0xffffffffu, s1, o);
              }
            }
            if (lane == 0) {
              if (on0) {
                nrm[c0] = re0 ? s0 : nn0;
                if (re0) ref[c0] = s0;
              }
              if (on1) {
                nrm[c1] = re1 ? s1 : nn1;
                if (re1) ref[c1] = s1;
              }
            }
          }
        } else {
          double dot0 = 0.0, dot1 = 0.0;
#pragma unroll 4
          for (int i = j + 1 + lane; i < p; i += 32) {
            const double v = vb[i];
            dot0 += v * col0[i];
            dot1 += v * col1[i];
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            dot0 += __shfl_xor_sync(0xffffffffu, dot0, o);
            dot1 += __shfl_xor_sync(0xffffffffu, dot1, o);
          }
          const double cj0 = col0[j], cj1 = col1[j];
          const double d0 = (cj0 + scale * dot0) * tau, d1 = (cj1 + scale * dot1) * tau;
          const double ds0 = d0 * scale, ds1 = d1 * scale;
          const double nj0 = cj0 - d0, nj1 = cj1 - d1;
          bool re0 = false, re1 = false;
          double nn0 = 0.0, nn1 = 0.0;
          if (pivot) {
            nn0 = nrm[on0 ? c0 : c1] - nj0 * nj0;
            nn1 = nrm[on1 ? c1 : c0] - nj1 * nj1;
            re0 = !(nn0 > 1.5e-8 * ref[on0 ? c0 : c1]);
            re1 = !(nn1 > 1.5e-8 * ref[on1 ? c1 : c0]);
          }
          double s0 = 0.0, s1 = 0.0;
          if (on0 && on1) {
#pragma unroll 4
            for (int i = j + 1 + lane; i < p; i += 32) {
              const double v = vb[i];
              const double y0 = col0[i] - ds0 * v, y1 = col1[i] - ds1 * v;
              col0[i] = y0;
              col1[i] = y1;
              s0 += y0 * y0;
              s1 += y1 * y1;
            }
          } else {  // one live column (col0 and col1 alias it)
            const double dsa = on0 ? ds0 : ds1;
            double* cola = on0 ? col0 : col1;
#pragma unroll 4
            for (int i = j + 1 + lane; i < p; i += 32) {
              const double y = cola[i] - dsa * vb[i];
              cola[i] = y;
              s0 += y * y;
            }
            s1 = s0;
          }
          if (lane == 0) {
            if (on0) col0[j] = nj0;
            if (on1) col1[j] = nj1;
          }
          if (pivot) {
            if (re0 || re1) {
#pragma unroll
              for (int o = 16; o > 0; o >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, o);
                s1 += __shfl_xor_sync(0xffffffffu, s1, o);
              }
            }
            if (lane == 0) {
              if (on0) {
                nrm[c0] = re0 ? s0 : nn0;
                if (re0) ref[c0] = s0;
              }
              if (on1) {
                nrm[c1] = re1 ? s1 : nn1;
                if (re1) ref[c1] = s1;
              }
            }
          }
        }
      }
    }
    __syncthreads();
  }
  __syncthreads();
  if (P.R_out) {
    // ---- R (q x q upper triangular, ld = q) of X = Q R: column c was reflected at step c
    for (int idx = tid; idx < q * wc; idx += QNT) {
      const int r = idx / wc, x = idx - r * wc;
      const int s = stepidx[x];
      double v = 0.0;
      if (r < nsteps) {
        if (s < 0 || r < s) v = Xs[(size_t)x * pp + r];
        else if (r == s) v = diag[x];
      }
      P.R_out[(i64)r * q + rank + C * x] = v;
    }
  } else {
    // ---- write out Q^T X: rows >= nsteps are zero; a column pivoted at step s is (R entries, beta, zeros)
    for (int idx = tid; idx < p * wc; idx += QNT) {
      const int r = idx / wc, x = idx - r * wc;
      const int s = stepidx[x];
      double v = 0.0;
      if (r < nsteps) {
        if (s < 0 || r < s) v = Xs[(size_t)x * pp + r];
        else if (r == s) v = diag[x];
      }
      P.X[(i64)r * P.ld + rank + C * x] = v;
    }
  }
  if (rank == 0 && tid == 0 && P.rank_out) P.rank_out[0] = nsteps;
  // no CTA may leave while a peer can still read its shared memory
  if (C > 1) cluster.sync();
}

// ------------------------------------------------------------------------------------------------
// Register-resident variant for p <= 32 * EPL rows and <= 32 columns per CTA: warp wi owns the local columns wi and
// wi + 16 and keeps them in REGISTERS for the whole factorisation (lane l holds rows l, l + 32, ...), so a step
// costs one shared-memory read of the reflector per row slab and four DFMA per element pair; shared memory only
// carries the reflector, the pivot candidates and the staged pivot column.  The generic kernel above is
// issue-bound at ~15k warp instructions per step and CTA (ncu, profiles/); this one executes about a third.
// The step loop is unrolled over the 32-row slabs (JB = j / 32 is a compile-time constant inside the body), so
// finished slabs cost nothing and the "diagonal" element is reached with a static register index.
// Pivot-column slabs are staged round-robin: slab e goes to CTA e % C at offset (e / C) * 32 + lane.
template <int EPL>
__global__ void __launch_bounds__(QNT) qtt_qrcp_reg_kernel(const __grid_constant__ QrcpGroup g) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = g.cluster;
  const int rank = (C > 1) ? (int)cluster.block_rank() : 0;
  const QrcpProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int p = P.p, q = P.q;
  const int w = g.w, pp = g.pp;
  const bool pivot = g.pivot != 0;

  extern __shared__ __align__(16) double sm[];
  double* Xs = sm;
  double* vb = Xs + (size_t)w * pp;  // 32 * EPL
  double* red = vb + 32 * EPL;
  double* diag = red + QNW;
  double* xfro = diag + w;
  long long* wval = reinterpret_cast<long long*>(xfro + MAXC);
  long long* candv = wval + QNW;
  int* wcol = reinterpret_cast<int*>(candv + 2 * MAXC);
  int* candc = wcol + QNW;
  int* stepidx = candc + 2 * MAXC;
  const int chm = g.chm;
  double* stage = reinterpret_cast<double*>(stepidx + ((w + 1) & ~1));  // [2][MAXC sources][chm]
  auto stage_of = [&](int k) { return (C > 1) ? cluster.map_shared_rank(stage, k) : stage; };
  auto barrier = [&]() {
    if (C > 1) cluster.sync();
    else __syncthreads();
  };

  const int wc = (q - rank + C - 1) / C;  // columns rank, rank + C, ... < q
  if (P.transposed) {
    for (int idx = tid; idx < p * wc; idx += QNT) {
      const int x = idx / p, r = idx - x * p;
      Xs[(size_t)x * pp + r] = P.X[(i64)(rank + C * x) * P.ld + r];
    }
  } else {
    for (int idx = tid; idx < p * wc; idx += QNT) {
      const int r = idx / wc, x = idx - r * wc;
      Xs[(size_t)x * pp + r] = P.X[(i64)r * P.ld + rank + C * x];
    }
  }
  for (int i = tid; i < 32 * EPL; i += QNT) vb[i] = 0.0;
  __syncthreads();
  // ---- my two columns into registers
  const bool has0 = warp < wc, has1 = warp + QNW < wc;
  const int col0g = rank + C * warp, col1g = rank + C * (warp + QNW);
  double x0[EPL], x1[EPL];
  double n0 = 0.0, n1 = 0.0;
#pragma unroll
  for (int e = 0; e < EPL; ++e) {
    const int i = lane + 32 * e;
    x0[e] = (has0 && i < p) ? Xs[(size_t)warp * pp + i] : 0.0;
    x1[e] = (has1 && i < p) ? Xs[(size_t)(warp + QNW) * pp + i] : 0.0;
    n0 += x0[e] * x0[e];
    n1 += x1[e] * x1[e];
  }
  int step0 = -1, step1 = -1;
  double diag0 = 0.0, diag1 = 0.0, r0 = 0.0, r1 = 0.0;
  double thresh2 = -1.0;
  if (pivot) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      n0 += __shfl_xor_sync(0xffffffffu, n0, o);
      n1 += __shfl_xor_sync(0xffffffffu, n1, o);
    }
    r0 = n0;
    r1 = n1;
    if (lane == 0) red[warp] = n0 + n1;
    __syncthreads();
    double myfro = 0.0;
    for (int i = 0; i < QNW; ++i) myfro += red[i];
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
    thresh2 = 3.1554436208840472e-30 * fro2;  // (8 eps)^2 ||X||_F^2
  }
  __syncthreads();

  const int rmax = min(p, q);
  int nsteps = 0;
  bool stop = false;
#pragma unroll
  for (int JB = 0; JB < EPL; ++JB) {
    if (stop || 32 * JB >= rmax) break;
    for (int jj = 0; jj < 32; ++jj) {
      const int j = 32 * JB + jj;
      if (j >= rmax) {
        stop = true;
        break;
      }
      const int par = j & 1;
      const bool live0 = has0 && step0 < 0, live1 = has1 && step1 < 0;
      int gcol = j;
      int stage_col = -1;  // global column this CTA stages before the barrier
      if (pivot) {
        long long bv = live0 ? norm_key(n0) : -1ll;
        int bc = live0 ? col0g : 0x7fffffff;
        const long long v1 = live1 ? norm_key(n1) : -1ll;
        if (v1 > bv) {
          bv = v1;
          bc = col1g;
        }
        if (lane == 0) {
          wval[warp] = bv;
          wcol[warp] = bc;
        }
        __syncthreads();
        bv = wval[lane & 15];
        bc = wcol[lane & 15];
        warp_argmax16(bv, bc);
        if (C > 1 && warp == 0 && lane < C) {
          long long* rv = cluster.map_shared_rank(candv, lane);
          int* rc = cluster.map_shared_rank(candc, lane);
          rv[par * MAXC + rank] = bv;
          rc[par * MAXC + rank] = bc;
        }
        if (bv >= 0) stage_col = bc;
        gcol = bc;
        // (the global winner is known after the barrier)
        if (C == 1 && (bv < 0 || !(__longlong_as_double(bv) > thresh2))) {
          stop = true;
          break;
        }
      } else if (rank == j % C) {
        stage_col = j;
      }
      // ---- stage the column (rows >= j) slab by slab in the peers: warp e pushes slab e from the shared-memory
      //      copy (kept current by the write-through of the update below); one warp pushing all slabs would
      //      serialise ~250 cycles per remote store
      if (!pivot) __syncthreads();  // (with pivoting the barrier above orders the write-through)
      if (stage_col >= 0 && warp >= JB && 32 * warp < p && warp < EPL) {
        const double* col = Xs + (size_t)(stage_col / C) * pp;
        double* dst = stage_of(warp % C);
        const int i = 32 * warp + lane;
        dst[(size_t)(par * MAXC + rank) * chm + (warp / C) * 32 + lane] = (i < p) ? col[i] : 0.0;
      }
      barrier();
      if (pivot && C > 1) {
        long long gval = (lane & 15) < C ? candv[par * MAXC + (lane & 15)] : -1ll;
        gcol = (lane & 15) < C ? candc[par * MAXC + (lane & 15)] : 0x7fffffff;
        warp_argmax16(gval, gcol);
        if (gval < 0 || !(__longlong_as_double(gval) > thresh2)) {  // what is left is rounding noise (uniform)
          stop = true;
          break;
        }
      }
      nsteps = j + 1;
      const int owner = gcol % C, lc = gcol / C;
      // ---- gather the pivot column (one row per thread); sum of squares of the rows below j on the way
      {
        double s = 0.0;
        const int i = tid;  // slab = warp
        if (i >= j && i < p) {
          const double* src = stage_of(warp % C);
          const double x = src[(size_t)(par * MAXC + owner) * chm + (warp / C) * 32 + lane];
          vb[i] = x;
          if (i > j) s = x * x;
        }
        s = warp_sum(s);
        if (lane == 0) red[warp] = s;
      }
      __syncthreads();
      double sigma = red[lane & 15];
      sigma += __shfl_xor_sync(0xffffffffu, sigma, 8);
      sigma += __shfl_xor_sync(0xffffffffu, sigma, 4);
      sigma += __shfl_xor_sync(0xffffffffu, sigma, 2);
      sigma += __shfl_xor_sync(0xffffffffu, sigma, 1);
      const double alpha = vb[j];
      double beta = alpha, tau = 0.0, scale = 0.0;
      if (sigma > 0.0) {
        const double n2 = alpha * alpha + sigma;
        double r = rsqrt(n2);
        r = r * (1.5 - 0.5 * n2 * r * r);
        double nr = n2 * r;
        nr = nr + 0.5 * r * (n2 - nr * nr);  // sqrt(n2) to full accuracy
        const double aa = fabs(alpha);
        beta = -copysign(nr, alpha);
        tau = 1.0 + aa * r;
        scale = copysign(1.0 / (aa + nr), alpha);
      }
      bool upd0 = live0, upd1 = live1;
      if (rank == owner) {
        if (live0 && col0g == gcol) {
          step0 = j;
          diag0 = beta;
          upd0 = false;
        }
        if (live1 && col1g == gcol) {
          step1 = j;
          diag1 = beta;
          upd1 = false;
        }
      }
      (void)lc;
      // ---- apply:  dot = col[j] + scale * sum_{i>j} v_i col_i;  col[j] -= tau dot;  col_i -= (tau dot scale) v_i
      if ((upd0 || upd1) && (tau != 0.0 || pivot)) {
        double dot0 = 0.0, dot1 = 0.0;
#pragma unroll
        for (int e = JB; e < EPL; ++e) {
          double v = vb[lane + 32 * e];
          if (e == JB && lane <= jj) v = 0.0;
          dot0 += v * x0[e];
          dot1 += v * x1[e];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          dot0 += __shfl_xor_sync(0xffffffffu, dot0, o);
          dot1 += __shfl_xor_sync(0xffffffffu, dot1, o);
        }
        const double cj0 = __shfl_sync(0xffffffffu, x0[JB], jj), cj1 = __shfl_sync(0xffffffffu, x1[JB], jj);
        const double d0 = upd0 ? (cj0 + scale * dot0) * tau : 0.0, d1 = upd1 ? (cj1 + scale * dot1) * tau : 0.0;
        const double ds0 = d0 * scale, ds1 = d1 * scale;
        const double nj0 = cj0 - d0, nj1 = cj1 - d1;
        double s0 = 0.0, s1 = 0.0;
#pragma unroll
        for (int e = JB; e < EPL; ++e) {
          double v = vb[lane + 32 * e];
          if (e == JB && lane <= jj) v = 0.0;
          x0[e] -= ds0 * v;
          x1[e] -= ds1 * v;
          if (!(e == JB && lane <= jj)) {
            s0 += x0[e] * x0[e];
            s1 += x1[e] * x1[e];
          }
        }
        if (lane == jj) {
          if (upd0) x0[JB] = nj0;
          if (upd1) x1[JB] = nj1;
        }
        // write-through: the shared-memory copy of my columns is what gets staged when one of them is the pivot
#pragma unroll
        for (int e = JB; e < EPL; ++e) {
          const int i = lane + 32 * e;
          if (i < p) {
            if (upd0) Xs[(size_t)warp * pp + i] = x0[e];
            if (upd1) Xs[(size_t)(warp + QNW) * pp + i] = x1[e];
          }
        }
        if (pivot) {
          if (upd0) n0 -= nj0 * nj0;
          if (upd1) n1 -= nj1 * nj1;
          const bool re0 = upd0 && !(n0 > 1.5e-8 * r0), re1 = upd1 && !(n1 > 1.5e-8 * r1);
          if (re0 || re1) {  // warp-uniform: the downdated norm has lost 8 digits, take the exact one
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
              s0 += __shfl_xor_sync(0xffffffffu, s0, o);
              s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            }
            if (re0) n0 = r0 = s0;
            if (re1) n1 = r1 = s1;
          }
        }
      }
    }
  }
  // ---- registers -> shared memory, then the coalesced write-out
  __syncthreads();
#pragma unroll
  for (int e = 0; e < EPL; ++e) {
    const int i = lane + 32 * e;
    if (has0 && i < p) Xs[(size_t)warp * pp + i] = x0[e];
    if (has1 && i < p) Xs[(size_t)(warp + QNW) * pp + i] = x1[e];
  }
  if (lane == 0) {
    if (has0) {
      stepidx[warp] = step0;
      diag[warp] = diag0;
    }
    if (has1) {
      stepidx[warp + QNW] = step1;
      diag[warp + QNW] = diag1;
    }
  }
  __syncthreads();
  if (P.R_out) {
    for (int idx = tid; idx < q * wc; idx += QNT) {
      const int r = idx / wc, x = idx - r * wc;
      const int s = stepidx[x];
      double v = 0.0;
      if (r < nsteps) {
        if (s < 0 || r < s) v = Xs[(size_t)x * pp + r];
        else if (r == s) v = diag[x];
      }
      P.R_out[(i64)r * q + rank + C * x] = v;
    }
  } else {
    for (int idx = tid; idx < p * wc; idx += QNT) {
      const int r = idx / wc, x = idx - r * wc;
      const int s = stepidx[x];
      double v = 0.0;
      if (r < nsteps) {
        if (s < 0 || r < s) v = Xs[(size_t)x * pp + r];
        else if (r == s) v = diag[x];
      }
      P.X[(i64)r * P.ld + rank + C * x] = v;
    }
  }
  if (rank == 0 && tid == 0 && P.rank_out) P.rank_out[0] = nsteps;
  if (C > 1) cluster.sync();  // no CTA may leave while a peer can still read its shared memory
}

size_t qrcp_reg_smem_bytes(int w, int pp, int epl, int chm) {
  const size_t doubles = (size_t)w * pp + 32 * (size_t)epl + QNW + (size_t)w + MAXC + QNW + 2 * MAXC;
  const size_t ints = QNW + 2 * MAXC + (((size_t)w + 1) & ~(size_t)1);
  return (doubles + 2 * MAXC * (size_t)chm) * sizeof(double) + ints * sizeof(int) + 16;
}

size_t qrcp_smem_bytes(int w, int pp, int chm) {
  const size_t doubles = (size_t)w * pp + pp + QNW + 3 * (size_t)w + MAXC + QNW + 2 * MAXC;  // incl. the 64-bit keys
  const size_t ints = QNW + 2 * MAXC + (((size_t)w + 1) & ~(size_t)1);
  return (doubles + 2 * MAXC * (size_t)chm) * sizeof(double) + ints * sizeof(int) + 16;
}

int qrcp_cluster(int q) {
  int C = (q + 15) / 16;
  C = C < 1 ? 1 : (C > MAXC ? MAXC : C);
  int c2 = 1;
  while (c2 < C) c2 *= 2;
  return c2 > MAXC ? MAXC : c2;
}

template <class K>
cudaError_t launch_qrcp(K kern, const QrcpGroup& g, size_t smem, double flops, int pmax, int qmax, cudaStream_t stream) {
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(kern))) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(g.cluster * g.nprob);
  cfg.blockDim = dim3(QNT);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = g.cluster;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  QttProf prof(g.pivot ? QK_QRCP : QK_LQ_PANEL, stream, flops, pmax, qmax, g.nprob, g.pivot ? g.cluster : -g.cluster);
  return cudaLaunchKernelEx(&cfg, kern, g);
}

}  // namespace

bool qtt_qrcp_fits(int p, int q) {
  if (p < 1 || q < 1) return false;
  const int C = qrcp_cluster(q);
  const int w = (q + C - 1) / C;
  return qrcp_smem_bytes(w, p | 1, (p + C - 1) / C) <= 220 * 1024;
}

cudaError_t qtt_launch_qrcp(const QrcpProb* probs, int n, int pivot, cudaStream_t stream) {
  for (int b0 = 0; b0 < n; b0 += QTT_QRCP_MAX_BATCH) {
    QrcpGroup g;
    g.nprob = 0;
    g.pivot = pivot;
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
    const int C = qrcp_cluster(qmax);
    g.cluster = C;
    g.w = (qmax + C - 1) / C;
    g.pp = pmax | 1;
    cudaError_t e;
    if (pmax <= 512 && g.w <= 2 * QNW) {
      // register-resident columns
      const int epl = pmax <= 128 ? 4 : (pmax <= 256 ? 8 : 16);
      g.chm = 32 * ((epl + C - 1) / C);
      const size_t smem = qrcp_reg_smem_bytes(g.w, g.pp, epl, g.chm);
      if (smem > 224 * 1024) return cudaErrorInvalidConfiguration;
      if (epl == 4) e = launch_qrcp(qtt_qrcp_reg_kernel<4>, g, smem, flops, pmax, qmax, stream);
      else if (epl == 8) e = launch_qrcp(qtt_qrcp_reg_kernel<8>, g, smem, flops, pmax, qmax, stream);
      else e = launch_qrcp(qtt_qrcp_reg_kernel<16>, g, smem, flops, pmax, qmax, stream);
    } else {
      g.chm = (pmax + C - 1) / C;
      const size_t smem = qrcp_smem_bytes(g.w, g.pp, g.chm);
      if (smem > 224 * 1024) return cudaErrorInvalidConfiguration;
      e = launch_qrcp(qtt_qrcp_kernel<0>, g, smem, flops, pmax, qmax, stream);
    }
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}
