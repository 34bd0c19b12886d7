// Register-blocked cluster block Jacobi: the production one-sided (Hestenes)
// Jacobi SVD for matrices of up to 512 rows and 512 columns,
//
//   X (p x q)  <-  J X,   J orthogonal, rows of the result mutually orthogonal:  J X = Sigma V^T.
//
// What bounded the first version of this kernel (jacobi.cu, profiles/r1_blockjacobi_full.md) was not the fp64 pipe
// but shared memory: one warp per row pair kept ONE row in registers and read the other row twice and wrote it
// once per meeting (3 x 4 KB of shared-memory traffic per pair at 512 columns: ~1500 of the ~2100 cycles of a
// round), and the block exchange through distributed shared memory ran at ~17 B/clk (~15k cycles per round).  Here
//  * a warp keeps TWO "top" rows in registers for a whole block meeting and pulls TWO "bottom" rows into registers
//    per super-round: four pair rotations per round trip through shared memory (a 2 x 2 register block), done as two
//    dependent sub-steps of two INDEPENDENT rotations each, so the inner-product reductions and the rotation
//    arithmetic of the two pairs overlap (instruction-level parallelism instead of stalls);
//  * the matrix lives in global memory (L2: at most 2 MB per operand) between block meetings: every CTA stores its
//    two blocks and loads the next two, ordered by ONE cluster barrier per meeting (release / acquire at cluster
//    scope; the loads bypass L1).  L2 serves a CTA at ~50 B/clk, three times the distributed-shared-memory rate,
//    and no slot relabelling is needed: the round-robin schedule is a pure function of (round, CTA rank).
// One cluster per matrix, 2 Ce blocks of BR rows, Ce = ceil(rows / 2 BR) CTAs take part (the number of rows is read
// on the device: the numerical rank found by the pivoted-QR preconditioner).  A sweep = pairs inside every block
// + 2 Ce - 1 block meetings; every pair of rows meets exactly once per sweep, as in the cyclic Jacobi method.
// Squared row norms are recomputed from the data whenever a block is loaded and updated in closed form inside a
// meeting (aa' = aa - t ab, bb' = bb + t ab).  Convergence: a sweep without a pair of cos^2 > 1e-15.
#include <cooperative_groups.h>

#include "common.cuh"
#include "jacobi_rot.cuh"
namespace cg = cooperative_groups;

namespace {

constexpr int MAXC = 16;

__device__ __forceinline__ void rr_pair(int P, int t, int k, int& ia, int& ib) {
  if (k == 0) {
    ia = P - 1;
    ib = t;
  } else {
    ia = (t + k) % (P - 1);
    ib = (t - k + (P - 1)) % (P - 1);
  }
}

__device__ __forceinline__ void warp_sum2(double& a, double& b) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
}

// A row of up to 64 * E2 columns held by a warp: lane l owns the column pairs (2 l, 2 l + 1) + 64 e, e < E2.
template <int E2>
struct RowRegs {
  double2 v[E2];
};

template <int E2>
__device__ __forceinline__ void load_global(RowRegs<E2>& r, const double* X, i64 ld, int row, int p, int q, bool vec,
                                            int lane) {
#pragma unroll
  for (int e = 0; e < E2; ++e) {
    const int x = 2 * lane + 64 * e;
    double2 t = make_double2(0.0, 0.0);
    if (row < p) {
      const double* src = X + (i64)row * ld + x;
      if (vec && x + 1 < q) {
        t = __ldcg(reinterpret_cast<const double2*>(src));
      } else {
        if (x < q) t.x = __ldcg(src);
        if (x + 1 < q) t.y = __ldcg(src + 1);
      }
    }
    r.v[e] = t;
  }
}
template <int E2>
__device__ __forceinline__ void store_global(const RowRegs<E2>& r, double* X, i64 ld, int row, int p, int q, bool vec,
                                             int lane) {
  if (row >= p) return;
#pragma unroll
  for (int e = 0; e < E2; ++e) {
    const int x = 2 * lane + 64 * e;
    double* dst = X + (i64)row * ld + x;
    if (vec && x + 1 < q) {
      __stcg(reinterpret_cast<double2*>(dst), r.v[e]);
    } else {
      if (x < q) __stcg(dst, r.v[e].x);
      if (x + 1 < q) __stcg(dst + 1, r.v[e].y);
    }
  }
}
template <int E2>
__device__ __forceinline__ void load_shared(RowRegs<E2>& r, const double* row, int lane) {
#pragma unroll
  for (int e = 0; e < E2; ++e) r.v[e] = *reinterpret_cast<const double2*>(row + 2 * lane + 64 * e);
}
template <int E2>
__device__ __forceinline__ void store_shared(const RowRegs<E2>& r, double* row, int lane) {
#pragma unroll
  for (int e = 0; e < E2; ++e) *reinterpret_cast<double2*>(row + 2 * lane + 64 * e) = r.v[e];
}
template <int E2>
__device__ __forceinline__ double dot_partial(const RowRegs<E2>& a, const RowRegs<E2>& b) {
  double s0 = 0.0, s1 = 0.0;
#pragma unroll
  for (int e = 0; e < E2; ++e) {
    s0 = fma(a.v[e].x, b.v[e].x, s0);
    s1 = fma(a.v[e].y, b.v[e].y, s1);
  }
  return s0 + s1;
}
template <int E2>
__device__ __forceinline__ void rotate(RowRegs<E2>& a, RowRegs<E2>& b, double c, double s) {
#pragma unroll
  for (int e = 0; e < E2; ++e) {
    const double ax = a.v[e].x, ay = a.v[e].y, bx = b.v[e].x, by = b.v[e].y;
    a.v[e].x = c * ax - s * bx;
    a.v[e].y = c * ay - s * by;
    b.v[e].x = s * ax + c * bx;
    b.v[e].y = s * ay + c * by;
  }
}

// Two independent pairs (a0, b0) and (a1, b1).  The rotation of pair 0 is computed by the lanes 0-15 and that of pair
// 1 by the lanes 16-31 (the same scalar instructions serve both), then exchanged with three shuffles each -- the
// rotation parameters were two thirds of the instructions of a meeting at 256 columns when every lane computed both.
template <int E2>
__device__ __forceinline__ void meet2(RowRegs<E2>& a0, RowRegs<E2>& b0, double& aa0, double& bb0, RowRegs<E2>& a1,
                                      RowRegs<E2>& b1, double& aa1, double& bb1, double tol2, double floor2, int& big,
                                      int lane) {
  double d0 = dot_partial(a0, b0), d1 = dot_partial(a1, b1);
  warp_sum2(d0, d1);
  const bool up = (lane & 16) != 0;
  const Rot R = jacobi_rotation(up ? aa1 : aa0, up ? bb1 : bb0, up ? d1 : d0, tol2, floor2);
  const unsigned ap = __ballot_sync(0xffffffffu, R.apply), bg = __ballot_sync(0xffffffffu, R.big);
  const double c0 = __shfl_sync(0xffffffffu, R.c, 0), c1 = __shfl_sync(0xffffffffu, R.c, 16);
  const double s0 = __shfl_sync(0xffffffffu, R.s, 0), s1 = __shfl_sync(0xffffffffu, R.s, 16);
  const double t0 = __shfl_sync(0xffffffffu, R.t, 0), t1 = __shfl_sync(0xffffffffu, R.t, 16);
  if (ap & 1u) {
    rotate(a0, b0, c0, s0);
    aa0 = fmax(aa0 - t0 * d0, 0.0);
    bb0 = fmax(bb0 + t0 * d0, 0.0);
    big += (int)(bg & 1u);
  }
  if (ap & 0x10000u) {
    rotate(a1, b1, c1, s1);
    aa1 = fmax(aa1 - t1 * d1, 0.0);
    bb1 = fmax(bb1 + t1 * d1, 0.0);
    big += (int)((bg >> 16) & 1u);
  }
}

// shared memory (doubles): Bs [BR][PITCH] | nB [BR] | xch [2][MAXC] | xfro [MAXC] | cnt (int)
template <int EPL, int BR>
__global__ void __launch_bounds__(BR * 16) qtt_bj2_kernel(const __grid_constant__ JacGroup g) {
  constexpr int NW = BR / 2, NT = NW * 32, E2 = EPL / 2, PITCH = 32 * EPL;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = g.cluster;
  const int rank = (C > 1) ? (int)cluster.block_rank() : 0;
  const JacProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int p = P.p;
  if (P.p_dev) p = min(p, P.p_dev[0]);
  if (p < 2) return;  // uniform over the cluster
  const int Ce = max(1, (p + 2 * BR - 1) / (2 * BR));  // CTAs that take part (<= C by the launch configuration)
  if (rank >= Ce) return;
  const int q = P.q;
  const i64 ld = P.ld;
  double* X = P.X;
  const bool vec = ((ld & 1) == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0);
  const int NBLK = 2 * Ce;

  extern __shared__ __align__(16) double sm[];
  double* Bs = sm;
  double* nB = Bs + (size_t)BR * PITCH;
  double* xch = nB + BR;
  double* xfro = xch + 2 * MAXC;
  int* cnt = reinterpret_cast<int*>(xfro + MAXC);

  // ---- Frobenius norm^2 over the cluster -> noise floor (rows below eps ||X||_F / sqrt(p) are zero to working
  // accuracy; they cannot all be made mutually orthogonal when p > rank)
  double fro = 0.0;
  for (int r = warp; r < 2 * BR; r += NW) {
    const int gr = rank * 2 * BR + r;
    if (gr < p)
#pragma unroll 4
      for (int x = lane; x < q; x += 32) {
        const double v = __ldcg(X + (i64)gr * ld + x);
        fro += v * v;
      }
  }
  fro = warp_sum1(fro);
  if (tid == 0) cnt[0] = 0;
  if (tid < MAXC) xfro[tid] = 0.0;
  __syncthreads();
  if (lane == 0) atomicAdd(&xfro[rank], fro);
  __syncthreads();
  if (Ce > 1) {
    cluster.sync();  // peers have zeroed their xfro
    if (tid < Ce && tid != rank) {
      double* remote = cluster.map_shared_rank(xfro, tid);
      remote[rank] = xfro[rank];
    }
    cluster.sync();
  }
  double fro2 = 0.0;
  for (int c2 = 0; c2 < Ce; ++c2) fro2 += xfro[c2];
  const double floor2 = 4.930380657631324e-32 * fro2 / (double)p;
  const double tol = 2.220446049250313e-16 * sqrt((double)q);
  const double tol2 = tol * tol;
  __syncthreads();

  int sweep = 0, hit_limit = 0, mybig = 0;
  for (; sweep < g.max_sweeps; ++sweep) {
    // ---- pairs inside the blocks: this CTA does blocks rank and rank + Ce
    for (int which = 0; which < 2; ++which) {
      const int blk = rank + which * Ce;
      if (blk * BR >= p) continue;  // uniform over the CTA
      for (int r = warp; r < BR; r += NW) {
        RowRegs<E2> t;
        load_global(t, X, ld, blk * BR + r, p, q, vec, lane);
        store_shared(t, Bs + (size_t)r * PITCH, lane);
        double sq = dot_partial(t, t);
        sq = warp_sum1(sq);
        if (lane == 0) nB[r] = sq;
      }
      __syncthreads();
      for (int round = 0; round < BR - 1; ++round) {
        int ia, ib;
        rr_pair(BR, round, warp, ia, ib);  // NW = BR / 2 pairs per round, one per warp
        RowRegs<E2> a, b;
        load_shared(a, Bs + (size_t)ia * PITCH, lane);
        load_shared(b, Bs + (size_t)ib * PITCH, lane);
        const double aa = nB[ia], bb = nB[ib];
        double ab = warp_sum1(dot_partial(a, b));
        const Rot R = jacobi_rotation(aa, bb, ab, tol2, floor2);
        if (R.apply) {
          rotate(a, b, R.c, R.s);
          store_shared(a, Bs + (size_t)ia * PITCH, lane);
          store_shared(b, Bs + (size_t)ib * PITCH, lane);
          if (lane == 0) {
            nB[ia] = fmax(aa - R.t * ab, 0.0);
            nB[ib] = fmax(bb + R.t * ab, 0.0);
          }
          mybig += R.big ? 1 : 0;
        }
        __syncthreads();
      }
      for (int r = warp; r < BR; r += NW) {
        RowRegs<E2> t;
        load_shared(t, Bs + (size_t)r * PITCH, lane);
        store_global(t, X, ld, blk * BR + r, p, q, vec, lane);
      }
      __syncthreads();
    }
    if (Ce > 1) cluster.sync();
    // ---- round-robin tournament over the 2 Ce blocks: one block meeting per CTA and round
    for (int t = 0; t < NBLK - 1; ++t) {
      int ia, ib;
      rr_pair(NBLK, t, rank, ia, ib);
      const bool live = ia * BR < p && ib * BR < p;  // an empty padding block: nothing to do (uniform over the CTA)
      if (live) {
        RowRegs<E2> t0, t1, b0, b1;
        const int ra = ia * BR + 2 * warp, rb = ib * BR + 2 * warp;
        load_global(t0, X, ld, ra, p, q, vec, lane);
        load_global(t1, X, ld, ra + 1, p, q, vec, lane);
        load_global(b0, X, ld, rb, p, q, vec, lane);
        load_global(b1, X, ld, rb + 1, p, q, vec, lane);
        store_shared(b0, Bs + (size_t)(2 * warp) * PITCH, lane);
        store_shared(b1, Bs + (size_t)(2 * warp + 1) * PITCH, lane);
        double aa0 = dot_partial(t0, t0), aa1 = dot_partial(t1, t1);
        double q0 = dot_partial(b0, b0), q1 = dot_partial(b1, b1);
        warp_sum2(aa0, aa1);
        warp_sum2(q0, q1);
        if (lane == 0) {
          nB[2 * warp] = q0;
          nB[2 * warp + 1] = q1;
        }
        __syncthreads();
        // the two top rows of one warp belong to the same block: they met in the intra-block phase
        for (int s = 0; s < NW; ++s) {
          int j = warp + s;
          j = (j >= NW) ? j - NW : j;
          double* r0 = Bs + (size_t)(2 * j) * PITCH;
          double* r1 = r0 + PITCH;
          if (s > 0) {
            load_shared(b0, r0, lane);
            load_shared(b1, r1, lane);
          }
          double bb0 = nB[2 * j], bb1 = nB[2 * j + 1];
          meet2(t0, b0, aa0, bb0, t1, b1, aa1, bb1, tol2, floor2, mybig, lane);
          meet2(t0, b1, aa0, bb1, t1, b0, aa1, bb0, tol2, floor2, mybig, lane);
          store_shared(b0, r0, lane);
          store_shared(b1, r1, lane);
          if (lane == 0) {
            nB[2 * j] = bb0;
            nB[2 * j + 1] = bb1;
          }
          __syncthreads();
        }
        store_global(t0, X, ld, ra, p, q, vec, lane);
        store_global(t1, X, ld, ra + 1, p, q, vec, lane);
        load_shared(b0, Bs + (size_t)(2 * warp) * PITCH, lane);
        load_shared(b1, Bs + (size_t)(2 * warp + 1) * PITCH, lane);
        store_global(b0, X, ld, rb, p, q, vec, lane);
        store_global(b1, X, ld, rb + 1, p, q, vec, lane);
        __syncthreads();
      }
      if (Ce > 1) cluster.sync();  // release the stores / acquire the peers' stores (global memory, cluster scope)
    }
    // ---- "big" rotations of this sweep over the whole cluster
    if (lane == 0 && mybig) atomicAdd(&cnt[0], mybig);
    mybig = 0;
    __syncthreads();
    int total = cnt[0];
    if (Ce > 1) {
      const int par = sweep & 1;
      if (tid < Ce) {
        double* remote = cluster.map_shared_rank(xch, tid);
        remote[par * MAXC + rank] = (double)cnt[0];
      }
      cluster.sync();
      total = 0;
      for (int c2 = 0; c2 < Ce; ++c2) total += (int)xch[par * MAXC + c2];
    }
    __syncthreads();
    if (tid == 0) cnt[0] = 0;
    __syncthreads();
    if (total == 0) {
      ++sweep;
      break;
    }
    if (sweep + 1 == g.max_sweeps) hit_limit = 1;
  }
  if (rank == 0 && tid == 0 && P.status) {
    atomicMax(&P.status[0], sweep);
    if (hit_limit) atomicAdd(&P.status[1], 1);
  }
  // no CTA may leave while a peer can still write into its shared memory
  if (Ce > 1) cluster.sync();
}

template <int EPL, int BR>
cudaError_t launch_bj2(JacGroup& grp, int pmax, int qmax, double flops, cudaStream_t stream) {
  constexpr int NT = BR * 16;
  const size_t smem = ((size_t)BR * 32 * EPL + BR + 3 * MAXC + 2) * sizeof(double);
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_bj2_kernel<EPL, BR>))) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_bj2_kernel<EPL, BR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_bj2_kernel<EPL, BR>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grp.cluster * grp.nprob);
  cfg.blockDim = dim3(NT);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = grp.cluster;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  QttProf prof(QK_JACOBI, stream, flops, pmax, qmax, grp.nprob, grp.cluster);
  return cudaLaunchKernelEx(&cfg, qtt_bj2_kernel<EPL, BR>, grp);
}

}  // namespace

// Configuration for a group with largest shape pmax x qmax; false if the kernel does not cover it.
bool qtt_bj2_config(int pmax, int qmax, int& EPL, int& BR, int& C) {
  if (qmax <= 128) EPL = 4;
  else if (qmax <= 256) EPL = 8;
  else if (qmax <= 512) EPL = 16;
  else return false;
  // 8-row blocks on up to 16 CTAs for p <= 256 (measured 10-15 % faster than 16-row blocks on half as many CTAs),
  // 16-row blocks beyond
  BR = pmax <= 256 ? 8 : 16;
  C = (pmax + 2 * BR - 1) / (2 * BR);
  C = C < 1 ? 1 : C;
  return C <= MAXC;
}

cudaError_t qtt_launch_bj2(JacGroup& grp, int pmax, int qmax, double flops, cudaStream_t stream) {
  int EPL, BR, C;
  if (!qtt_bj2_config(pmax, qmax, EPL, BR, C)) return cudaErrorInvalidConfiguration;
  grp.cluster = C;
  grp.use_smem = 1;
  grp.wslice = 0;
  grp.max_sweeps = 60;
  if (BR == 8) {
    if (EPL == 4) return launch_bj2<4, 8>(grp, pmax, qmax, flops, stream);
    if (EPL == 8) return launch_bj2<8, 8>(grp, pmax, qmax, flops, stream);
    return launch_bj2<16, 8>(grp, pmax, qmax, flops, stream);
  }
  if (EPL == 4) return launch_bj2<4, 16>(grp, pmax, qmax, flops, stream);
  if (EPL == 8) return launch_bj2<8, 16>(grp, pmax, qmax, flops, stream);
  return launch_bj2<16, 16>(grp, pmax, qmax, flops, stream);
}
