// Batched one-sided (Hestenes) Jacobi on the ROWS of X (the truncated-SVD
// step of the R->L rounding sweep; row a6: the SVD of the zip-up's triangular factor): the dispatcher
// (qtt_launch_rowjacobi: bj2.cu for p, q <= 512, sbj.cu up to 2048 columns, the column-sliced kernel below as the
// last resort) and the rank selection.
//
//   X (p x q)  <-  J X,   J orthogonal, rows of the result mutually orthogonal:  J X = Sigma V^T.
//
// The right singular vectors are the normalised rows and the singular values are the row norms, so
// no rotation is ever accumulated.  One thread-block cluster per matrix: the columns are cut into
// slices, one per CTA, resident in (distributed) shared memory when they fit; per round-robin round
// the p/2 disjoint row pairs need (a.a, b.b, a.b), reduced with warp shuffles inside a CTA and
// exchanged all-to-all through distributed shared memory, so every CTA derives bit-identical
// rotations and applies them to its own slice.
#include <cooperative_groups.h>

#include "common.cuh"
#include "jacobi_rot.cuh"
namespace cg = cooperative_groups;

namespace {

constexpr int JNT = 512;
constexpr int MAXC = 16;

// dynamic shared memory (doubles): slice [p][wp] (if resident) | part [2][C][3*np2] | rot [2*np2]
//                                  | order (ints) [p_even] | counters
__global__ void __launch_bounds__(JNT) qtt_rowjacobi_kernel(const __grid_constant__ JacGroup g, int pmax, int wp) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = g.cluster;
  const int rank = cluster.block_rank();
  const JacProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x;
  int p = P.p;
  if (P.p_dev) p = min(p, P.p_dev[0]);
  if (p < 2) return;  // uniform over the cluster
  const int q = P.q;
  const int pe = (p + 1) & ~1;  // players in the tournament (one bye if p is odd)
  const int np2 = pe / 2;
  const int pe_max = (pmax + 1) & ~1, np2_max = pe_max / 2;

  extern __shared__ __align__(16) double sm[];
  double* slice_sm = sm;
  double* part = sm + (g.use_smem ? (size_t)pmax * wp : 0);
  double* rot = part + 2 * C * 3 * np2_max;
  int* flags = reinterpret_cast<int*>(rot + 2 * np2_max);  // [0] rotations this sweep
  // Largest squared row norm seen so far, identical in every CTA of the cluster (it is derived from the
  // exchanged totals only): [0] accumulates during phase B1, [1] is the value phase B1 reads.
  unsigned long long* nmax = reinterpret_cast<unsigned long long*>(flags + 2);

  const int w = g.wslice;
  const int cs = rank * w;
  const int wc = max(0, min(q, cs + w) - cs);
  double* S;
  i64 rs;  // row stride of the working slice
  if (g.use_smem) {
    S = slice_sm;
    rs = wp;
    for (int idx = tid; idx < p * wc; idx += JNT) {
      int r = idx / wc, x = idx - r * wc;
      S[(i64)r * rs + x] = P.X[(i64)r * P.ld + cs + x];
    }
  } else {
    S = P.X + cs;
    rs = P.ld;
  }
  if (tid == 0) {
    flags[0] = 0;
    nmax[0] = nmax[1] = 0ull;
  }
  __syncthreads();

  // threads per pair: power of two, chosen so one pass covers all pairs when possible
  int tpp = 32;
  while (tpp > 1 && np2 * tpp > JNT) tpp >>= 1;
  const int ngrp = JNT / tpp;
  const int grp = tid / tpp, gl = tid % tpp;
  const double tol = 2.220446049250313e-16 * sqrt((double)q);

  int sweep = 0, hit_limit = 0;
  unsigned par = 0;
  for (; sweep < g.max_sweeps; ++sweep) {
    for (int round = 0; round < pe - 1; ++round) {
      // ---- phase A: partial (aa, bb, ab) of every pair over this slice
      for (int k0 = 0; k0 < np2; k0 += ngrp) {  // uniform trip count: the shuffles below need full warps
        const int k = k0 + grp;
        int ia = p, ib = p;
        if (k < np2) {
          if (k == 0) {
            ia = pe - 1;
            ib = round;
          } else {
            ia = (round + k) % (pe - 1);
            ib = (round - k + (pe - 1)) % (pe - 1);
          }
        }
        double aa = 0.0, bb = 0.0, ab = 0.0;
        if (ia < p && ib < p) {
          const double* ra = S + (i64)ia * rs;
          const double* rb = S + (i64)ib * rs;
          for (int x = gl; x < wc; x += tpp) {
            double a = ra[x], b = rb[x];
            aa += a * a;
            bb += b * b;
            ab += a * b;
          }
        }
        for (int o = tpp >> 1; o > 0; o >>= 1) {
          aa += __shfl_xor_sync(0xffffffffu, aa, o);
          bb += __shfl_xor_sync(0xffffffffu, bb, o);
          ab += __shfl_xor_sync(0xffffffffu, ab, o);
        }
        if (k < np2) {
          for (int dst = gl; dst < C; dst += tpp) {
            double* remote = (C > 1) ? cluster.map_shared_rank(part, dst) : part;
            double* slot = remote + ((size_t)(par * C + rank) * np2_max + k) * 3;
            slot[0] = aa;
            slot[1] = bb;
            slot[2] = ab;
          }
        }
      }
      if (C > 1)
        cluster.sync();
      else
        __syncthreads();
      // ---- phase B1: one thread per pair derives the rotation
      for (int k = tid; k < np2; k += JNT) {
        double aa = 0.0, bb = 0.0, ab = 0.0;
        for (int src = 0; src < C; ++src) {
          const double* slot = part + ((size_t)(par * C + src) * np2_max + k) * 3;
          aa += slot[0];
          bb += slot[1];
          ab += slot[2];
        }
        double c = 1.0, s = 0.0;
        const double lim = tol * sqrt(aa) * sqrt(bb);
        // rows below eps * (largest row norm) are zero to working accuracy: rotating them against each
        // other never terminates when p > rank (they cannot all be mutually orthogonal); the selection
        // step writes such rows out as exact zeros
        const double floor2 = 4.930380657631324e-32 * __longlong_as_double((long long)nmax[1]);
        atomicMax(&nmax[0], (unsigned long long)__double_as_longlong(fmax(aa, bb)));
        if (fabs(ab) > lim && lim > 0.0 && aa > floor2 && bb > floor2) {
          const double zeta = (bb - aa) / (2.0 * ab);
          const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
          c = 1.0 / sqrt(1.0 + t * t);
          s = c * t;
          if (s != 0.0) atomicAdd(&flags[0], 1);
        }
        rot[2 * k] = c;
        rot[2 * k + 1] = s;
      }
      __syncthreads();
      // ---- phase B2: apply  a' = c a - s b,  b' = s a + c b  on this slice
      for (int k = grp; k < np2; k += ngrp) {
        const double c = rot[2 * k], s = rot[2 * k + 1];
        if (s == 0.0) continue;
        int ia, ib;
        if (k == 0) {
          ia = pe - 1;
          ib = round;
        } else {
          ia = (round + k) % (pe - 1);
          ib = (round - k + (pe - 1)) % (pe - 1);
        }
        double* ra = S + (i64)ia * rs;
        double* rb = S + (i64)ib * rs;
        for (int x = gl; x < wc; x += tpp) {
          double a = ra[x], b = rb[x];
          ra[x] = c * a - s * b;
          rb[x] = s * a + c * b;
        }
      }
      par ^= 1u;
      if (tid == 0) nmax[1] = nmax[0];
      __syncthreads();
    }
    const int nrot = flags[0];
    __syncthreads();
    if (tid == 0) flags[0] = 0;
    __syncthreads();
    if (nrot == 0) {
      ++sweep;
      break;
    }
    if (sweep + 1 == g.max_sweeps) hit_limit = 1;
  }
  if (g.use_smem) {
    for (int idx = tid; idx < p * wc; idx += JNT) {
      int r = idx / wc, x = idx - r * wc;
      P.X[(i64)r * P.ld + cs + x] = S[(i64)r * rs + x];
    }
  }
  if (rank == 0 && tid == 0 && P.status) {
    atomicMax(&P.status[0], sweep);
    if (hit_limit) atomicAdd(&P.status[1], 1);
  }
  // no CTA may leave while a peer can still write into its shared memory
  if (C > 1) cluster.sync();
}

// ------------------------------------------------------------------------------------------------
// select: sort rows by norm (bitonic in shared memory), rank rule, normalised top rows.
constexpr int SNT = 256;
constexpr int SEL_MAXP = 16384;  // rows whose sort keys fit the opt-in shared memory (12 bytes per padded row)

// dynamic shared memory: key [np] doubles | idx [np] ints, np = rows padded to a power of two
// One cluster of S CTAs per matrix (S = 1 for small ones): the squared row norms are computed by slices of rows, one
// slice per CTA, and all-gathered through distributed shared memory (a single CTA reading a 2 MB matrix out of L2 was
// most of this kernel's time); every CTA then sorts the keys itself and writes its share of the output rows.
__global__ void __launch_bounds__(SNT) qtt_select_kernel(const __grid_constant__ SelGroup g, int npmax, int S) {
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = S > 1 ? (int)cluster.block_rank() : 0;
  const SelProb& P = g.p[blockIdx.x / S];
  extern __shared__ __align__(16) double sel_sm[];
  double* key = sel_sm;
  int* idx = reinterpret_cast<int*>(sel_sm + npmax);
  __shared__ int s_rank;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int p = P.p, q = P.q;
  int np = 1;
  while (np < p) np <<= 1;
  for (int r = tid; r < np; r += SNT) idx[r] = r;
  const int per = (np + S - 1) / S;
  const int r_end = min(np, (crank + 1) * per);
  for (int r = crank * per + warp; r < r_end; r += SNT / 32) {
    double s = 0.0;
    if (r < p)
#pragma unroll 4
      for (int x = lane; x < q; x += 32) {
        double v = P.X[(i64)r * P.ld + x];
        s += v * v;
      }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const double kv = (r < p) ? s : -1.0;
    if (S > 1) {
      if (lane < S) cluster.map_shared_rank(key, lane)[r] = kv;
    } else if (lane == 0) {
      key[r] = kv;
    }
  }
  if (S > 1) cluster.sync();
  __syncthreads();
  // bitonic sort, descending by key (ties: lower row index first, for determinism)
  for (int k2 = 2; k2 <= np; k2 <<= 1)
    for (int j = k2 >> 1; j > 0; j >>= 1) {
      for (int i = tid; i < np; i += SNT) {
        int l = i ^ j;
        if (l > i) {
          bool desc = ((i & k2) == 0);
          double ki = key[i], kl = key[l];
          int ii = idx[i], il = idx[l];
          bool i_before_l = (ki > kl) || (ki == kl && ii < il);
          if (desc ? !i_before_l : i_before_l) {
            key[i] = kl; key[l] = ki;
            idx[i] = il; idx[l] = ii;
          }
        }
      }
      __syncthreads();
    }
  if (tid == 0) {
    const int mn = p < q ? p : q;
    int r = P.chi_max < mn ? P.chi_max : mn;
    double tot = 0.0;
    if (P.delta_out)  // (only the first SVD of an eps > 0 sweep needs ||X||_F)
      for (int i = p - 1; i >= 0; --i) tot += key[i];
    if (P.delta_out && crank == 0) *P.delta_out = P.delta_scale * sqrt(tot);
    double delta = -1.0;
    if (P.delta_ptr) delta = *P.delta_ptr;
    else if (P.delta_out) delta = P.delta_scale * sqrt(tot);
    if (P.delta_ptr || (P.delta_out && P.delta_scale > 0.0)) {
      // smallest r with sqrt(sum_{i >= r} sigma_i^2) <= delta
      double tail = 0.0;
      int rr = mn;
      for (int i = p - 1; i >= mn; --i) tail += key[i];
      for (int cand = mn; cand >= 0; --cand) {
        // tail = sum_{i >= cand} key[i]
        if (sqrt(tail) <= delta) rr = cand; else break;
        if (cand > 0) tail += key[cand - 1];
      }
      r = rr;
      if (r > P.chi_max) r = P.chi_max;
      if (r > mn) r = mn;
      if (r < 1) r = 1;
    }
    if (r > P.r_cap) r = P.r_cap;
    if (r < 1) r = 1;
    s_rank = r;
    if (P.rank && crank == 0) P.rank[0] = r;
  }
  __syncthreads();
  const int r = s_rank;
  if (P.sigma && crank == 0)
    for (int i = tid; i < p; i += SNT) P.sigma[i] = sqrt(fmax(key[i], 0.0));
  for (int j = crank * (SNT / 32) + warp; j < P.r_cap; j += S * (SNT / 32)) {
    double inv = 0.0;
    int src = 0;
    if (j < r) {
      src = idx[j];
      double s2 = key[j];
      // rows below 4 eps sigma_1 were not orthogonalised (see the row-Jacobi floor): exact zeros
      inv = (s2 > 1e-290 && s2 > 7.888609052210118e-31 * key[0]) ? rsqrt(s2) : 0.0;
      // one Newton step: rsqrt() is accurate to ~1 ulp in fp64, keep the normalisation at full precision
      inv = inv * (1.5 - 0.5 * s2 * inv * inv);
    }
#pragma unroll 4
    for (int x = lane; x < q; x += 32)
      P.out[(i64)j * P.out_ld + x] = (inv != 0.0) ? P.X[(i64)src * P.ld + x] * inv : 0.0;
  }
}

}  // namespace

cudaError_t qtt_launch_rowjacobi(const JacProb* probs, int n, cudaStream_t stream) {
  // production path: the register-blocked cluster block Jacobi (bj2.cu); problems of one call (the operands of one
  // site, similar shapes) share launches
  {
    bool all_fit = true;
    for (int i = 0; i < n && all_fit; ++i) {
      int EPL, BR, C;
      if (probs[i].p >= 2 && probs[i].q >= 1 && !qtt_bj2_config(probs[i].p, probs[i].q, EPL, BR, C)) all_fit = false;
    }
    if (all_fit) {
      int done = 0;
      while (done < n) {
        JacGroup grp;
        grp.nprob = 0;
        int pmax = 0, qmax = 0;
        double flops = 0.0;
        while (done < n && grp.nprob < QTT_JAC_MAX_BATCH) {
          const JacProb& pr = probs[done];
          if (pr.p >= 2 && pr.q >= 1) {
            grp.p[grp.nprob++] = pr;
            pmax = pr.p > pmax ? pr.p : pmax;
            qmax = pr.q > qmax ? pr.q : qmax;
            double a = pr.p > pr.q ? pr.p : pr.q, bb = pr.p > pr.q ? pr.q : pr.p;
            flops += 6.0 * a * bb * bb + 20.0 * bb * bb * bb;
          }
          ++done;
        }
        if (grp.nprob == 0) continue;
        QTT_CHECK_CUDA(qtt_launch_bj2(grp, pmax, qmax, flops, stream));
      }
      return cudaSuccess;
    }
  }
  // too large for a cluster's shared memory: the L2-streamed block Jacobi (sbj.cu) if the rows are short enough
  {
    bool ok = true;
    for (int i = 0; i < n && ok; ++i)
      if (probs[i].p >= 2 && probs[i].q >= 1 && !(probs[i].work && qtt_sbj_fits(probs[i].p, probs[i].q))) ok = false;
    if (ok) return qtt_launch_sbj(probs, n, stream);
  }
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_rowjacobi_kernel))) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_rowjacobi_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_rowjacobi_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  }
  for (int b0 = 0; b0 < n; b0 += QTT_JAC_MAX_BATCH) {
    JacGroup grp;
    grp.nprob = 0;
    int pmax = 0, qmax = 0;
    for (int i = b0; i < n && grp.nprob < QTT_JAC_MAX_BATCH; ++i) {
      if (probs[i].p < 2 || probs[i].q < 1) continue;  // a single row is already "orthogonal"
      grp.p[grp.nprob++] = probs[i];
      pmax = probs[i].p > pmax ? probs[i].p : pmax;
      qmax = probs[i].q > qmax ? probs[i].q : qmax;
    }
    if (grp.nprob == 0) continue;
    const int pe = (pmax + 1) & ~1;
    // exchange buffers [2][c][3 * pairs] + rotations: they grow with the cluster size c
    auto fixed_for = [&](int c) { return ((size_t)2 * c * 3 * (pe / 2) + 2 * (pe / 2) + 8) * sizeof(double); };
    const size_t budget = 216 * 1024;
    // smallest cluster whose slice fits in shared memory, with at least ~16 columns per CTA
    int C = 1, use_smem = 0, w = 0, wp = 0;
    for (int c = 1; c <= MAXC; c *= 2) {
      int ww = (qmax + c - 1) / c;
      ww = (ww + 3) & ~3;
      int wpp = ww | 1;
      size_t need = fixed_for(c) + (size_t)pmax * wpp * sizeof(double);
      if (need <= budget) {
        C = c; use_smem = 1; w = ww; wp = wpp;
        break;
      }
    }
    if (use_smem) {
      // more CTAs when there is enough work per round: aim at <= ~8k slice elements per CTA
      while (C < MAXC && (size_t)pmax * w > 8192 && w >= 32) {
        const int c2 = C * 2;
        int ww = (qmax + c2 - 1) / c2;
        ww = (ww + 3) & ~3;
        if (fixed_for(c2) + (size_t)pmax * (ww | 1) * sizeof(double) > budget) break;
        C = c2;
        w = ww;
        wp = w | 1;
      }
    } else {
      // the matrix stays in global memory (L2): the largest cluster whose exchange buffers fit
      C = MAXC;
      while (C > 1 && fixed_for(C) > budget) C /= 2;
      if (fixed_for(C) > budget) return cudaErrorInvalidConfiguration;
      w = (qmax + C - 1) / C;
      w = (w + 3) & ~3;
      wp = 0;
    }
    const size_t fixed = fixed_for(C);
    grp.cluster = C;
    grp.use_smem = use_smem;
    grp.wslice = w;
    grp.max_sweeps = 60;
    size_t smem = fixed + (use_smem ? (size_t)pmax * wp * sizeof(double) : 0);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C * grp.nprob);
    cfg.blockDim = dim3(JNT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    double flops = 0.0;  // nominal SVD count 6 a b^2 + 20 b^3, a >= b (kernels)
    for (int i = 0; i < grp.nprob; ++i) {
      double a = grp.p[i].p > grp.p[i].q ? grp.p[i].p : grp.p[i].q, b = grp.p[i].p > grp.p[i].q ? grp.p[i].q : grp.p[i].p;
      flops += 6.0 * a * b * b + 20.0 * b * b * b;
    }
    {
      QttProf prof(QK_JACOBI, stream, flops, pmax, qmax, grp.nprob, -C);
      QTT_CHECK_CUDA(cudaLaunchKernelEx(&cfg, qtt_rowjacobi_kernel, grp, pmax, wp));
    }
  }
  return cudaSuccess;
}

int qtt_select_max_rows() { return SEL_MAXP; }

cudaError_t qtt_launch_select(const SelProb* probs, int n, cudaStream_t stream) {
  for (int b0 = 0; b0 < n; b0 += QTT_SEL_MAX_BATCH) {
    SelGroup g;
    g.nprob = n - b0 < QTT_SEL_MAX_BATCH ? n - b0 : QTT_SEL_MAX_BATCH;
    int npmax = 2;
    for (int i = 0; i < g.nprob; ++i) {
      g.p[i] = probs[b0 + i];
      if (g.p[i].p > SEL_MAXP) return cudaErrorInvalidValue;  // callers check qtt_select_max_rows() first
      while (npmax < g.p[i].p) npmax <<= 1;
    }
    const size_t smem = (size_t)npmax * (sizeof(double) + sizeof(int));
    if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_select_kernel)))
      QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)((size_t)SEL_MAXP * (sizeof(double) + sizeof(int)))));
    double bytes = 0.0;
    for (int i = 0; i < g.nprob; ++i) bytes += 8.0 * ((double)g.p[i].p * g.p[i].q + (double)g.p[i].r_cap * g.p[i].q);
    int pmaxrows = 0;
    for (int i = 0; i < g.nprob; ++i) pmaxrows = g.p[i].p > pmaxrows ? g.p[i].p : pmaxrows;
    const int S = pmaxrows >= 64 ? 8 : 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(g.nprob * S);
    cfg.blockDim = dim3(SNT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = S;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    {
      QttProf prof(QK_SELECT, stream, bytes, g.p[0].p, g.p[0].q, g.nprob, 0);
      QTT_CHECK_CUDA(cudaLaunchKernelEx(&cfg, qtt_select_kernel, g, npmax, S));
    }
  }
  return cudaSuccess;
}
