// Batched one-sided (Hestenes) Jacobi on the ROWS of X (the truncated-SVD
// step of the R->L rounding sweep; row a6: the SVD of the zip-up's triangular factor).
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
#include <cstdlib>

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
// Two-level block Jacobi, the production path for every matrix whose row blocks fit in a cluster's shared
// memory.  The p rows are cut into 2C blocks of b rows; every CTA of the cluster (C CTAs) holds two blocks
// with their FULL rows, so a rotation needs no cross-CTA reduction at all:
//   sweep = intra-block pairs of the two resident blocks (b-1 rounds)
//         + 2C-1 outer rounds of a round-robin tournament over the blocks; in each, the CTA meets
//           every row of its "top" block with every row of its "bot" block (b inner rounds of b
//           disjoint pairs, one warp per pair, the top row kept in registers), then the blocks
//           move one seat through distributed shared memory (pull into a spare slot, two
//           cluster.syncs, relabel the slots -- no copy inside a CTA).
// Every pair of rows meets exactly once per sweep, as in the cyclic one-sided Jacobi method.
//  * Squared row norms travel with the rows and are updated in closed form after a rotation
//    (aa' = aa - t ab, bb' = bb + t ab), so a pair costs ONE inner product (a.b) and one warp reduction; they
//    are recomputed from the data once per sweep.
//  * The number of rows is read on the device (numerical rank from the pivoted-QR preconditioner); only
//    Ce = ceil(p / (2 bmax)) CTAs of the cluster take part, the others exit at once (cluster barriers wait
//    for non-exited threads only).
//  * Convergence: a sweep in which no pair had cos^2 > 1e-15 ends the iteration -- Jacobi converges
//    quadratically, so after such a sweep the remaining cosines are O(1e-15).
constexpr int BJ_NT = 512;
constexpr int BJ_G = 32;
constexpr int BJ_NGRP = BJ_NT / BJ_G;

// shared memory: 3 slots of [bmax * pitchmax data | bme norms] | xch [2][MAXC] counts | fro [MAXC] | ints
template <int EPL>
__global__ void __launch_bounds__(BJ_NT) qtt_blockjacobi_kernel(const __grid_constant__ JacGroup g, int bmax,
                                                                 int pitchmax) {
  cg::cluster_group cluster = cg::this_cluster();
  const int C = g.cluster;
  const int rank = (C > 1) ? (int)cluster.block_rank() : 0;
  const JacProb& P = g.p[blockIdx.x / C];
  const int tid = threadIdx.x, lane = tid & 31, grp = tid >> 5;
  // rows to rotate: the numerical rank found by the pivoted-QR preconditioner, if there is one
  int p = P.p;
  if (P.p_dev) p = min(p, P.p_dev[0]);
  if (p < 2) return;  // uniform over the cluster: nothing to orthogonalise
  const int Ce = max(1, (p + 2 * bmax - 1) / (2 * bmax));  // CTAs that take part (<= C)
  if (rank >= Ce) return;
  const int q = P.q;
  constexpr int pitch = BJ_G * EPL;  // every row is zero-padded to the full lane footprint (== pitchmax)
  const int b = (p + 2 * Ce - 1) / (2 * Ce);         // <= bmax

  extern __shared__ __align__(16) double sm[];
  const int bme = (bmax + 1) & ~1;
  const size_t data_sz = (size_t)bmax * pitchmax;
  const size_t slot_sz = data_sz + bme;
  double* xch = sm + 3 * slot_sz;  // [2][MAXC] "big rotation" counts from peers
  double* xfro = xch + 2 * MAXC;   // [MAXC]
  int* cnt = reinterpret_cast<int*>(xfro + MAXC);
  int top_s = 0, bot_s = 1, spare_s = 2;
  auto slot = [&](int sidx) { return sm + (size_t)sidx * slot_sz; };

  // ---- load: block k holds rows [k b, (k+1) b); CTA c starts with top = block c, bot = block 2Ce-1-c
  double fro = 0.0;
  for (int which = 0; which < 2; ++which) {
    const int blk = which == 0 ? rank : 2 * Ce - 1 - rank;
    double* S = slot(which == 0 ? top_s : bot_s);
    for (int idx = tid; idx < b * pitch; idx += BJ_NT) {
      const int r = idx / pitch, x = idx - r * pitch;
      const int gr = blk * b + r;
      double v = 0.0;
      if (gr < p && x < q) v = P.X[(i64)gr * P.ld + x];
      S[idx] = v;
      fro += v * v;
    }
  }
  // Frobenius norm^2 over the cluster -> noise floor (rows below eps * ||X||_F / sqrt(p) are zero to
  // working accuracy; they cannot all be made mutually orthogonal when p > rank)
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

  const int be = b + (b & 1);  // players of the intra-block tournament
  int sweep = 0, hit_limit = 0;
  int mybig = 0;
  for (; sweep < g.max_sweeps; ++sweep) {
    // ---- fresh squared norms of the resident rows
    for (int which = 0; which < 2; ++which) {
      double* S = slot(which == 0 ? top_s : bot_s);
      for (int r = grp; r < b; r += BJ_NGRP) {
        const double* row = S + (size_t)r * pitch + lane;
        double sq = 0.0;
#pragma unroll
        for (int e = 0; e < EPL; ++e)
          sq += row[e * BJ_G] * row[e * BJ_G];
        sq = warp_sum1(sq);
        if (lane == 0) S[data_sz + r] = sq;
      }
    }
    __syncthreads();
    // ---- intra-block pairs of both resident blocks
    for (int round = 0; round < be - 1; ++round) {
      for (int k0 = 0; k0 < be; k0 += BJ_NGRP) {  // be pairs in all: be/2 per block
        const int kk = k0 + grp;
        int ia = b, ib = b;
        double* S = slot(top_s);
        if (kk < be) {
          const int k = kk % (be / 2);
          S = slot(kk < be / 2 ? top_s : bot_s);
          if (k == 0) {
            ia = be - 1;
            ib = round;
          } else {
            ia = (round + k) % (be - 1);
            ib = (round - k + (be - 1)) % (be - 1);
          }
        }
        const bool live = ia < b && ib < b;
        double a[EPL], v[EPL];
        double ab = 0.0, ab2 = 0.0;
        double* ra = S + (size_t)(live ? ia : 0) * pitch + lane;
        double* rb = S + (size_t)(live ? ib : 0) * pitch + lane;
        if (live) {
#pragma unroll
          for (int e = 0; e < EPL; ++e) {
            a[e] = ra[e * BJ_G];
            v[e] = rb[e * BJ_G];
            if (e & 1) ab2 += a[e] * v[e];
            else ab += a[e] * v[e];
          }
          ab += ab2;
        }
        ab = warp_sum1(ab);
        if (live) {
          const double aa = S[data_sz + ia], bb = S[data_sz + ib];
          const Rot R = jacobi_rotation(aa, bb, ab, tol2, floor2);
          if (R.apply) {
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
              ra[e * BJ_G] = R.c * a[e] - R.s * v[e];
              rb[e * BJ_G] = R.s * a[e] + R.c * v[e];
            }
            if (lane == 0) {
              S[data_sz + ia] = fmax(aa - R.t * ab, 0.0);
              S[data_sz + ib] = fmax(bb + R.t * ab, 0.0);
              if (R.big) ++mybig;
            }
          }
        }
      }
      __syncthreads();
    }
    // ---- tournament over the 2Ce blocks
    for (int t = 0; t < 2 * Ce - 1; ++t) {
      double* T = slot(top_s);
      double* B = slot(bot_s);
      for (int i0 = 0; i0 < b; i0 += BJ_NGRP) {
        const int i = i0 + grp;
        const bool have = i < b;
        double a[EPL];
        double aa = 0.0;
        double* rt = T + (have ? i : 0) * pitch + lane;
        if (have) {
#pragma unroll
          for (int e = 0; e < EPL; ++e) a[e] = rt[e * BJ_G];
          aa = T[data_sz + i];
        }
        int j = have ? i : 0;
        for (int r = 0; r < b; ++r) {
          double ab = 0.0, ab2 = 0.0, bb = 0.0;
          double* rb = B + j * pitch + lane;
          if (have) {
            bb = B[data_sz + j];
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
              const double ve = rb[e * BJ_G];
              if (e & 1) ab2 += a[e] * ve;
              else ab += a[e] * ve;
            }
          }
          ab = warp_sum1(ab + ab2);
          if (have) {
            const Rot R = jacobi_rotation(aa, bb, ab, tol2, floor2);
            if (R.apply) {
#pragma unroll
              for (int e = 0; e < EPL; ++e) {  // the bottom row is read again: keeping it live costs spills
                const double ve = rb[e * BJ_G];
                const double an = R.c * a[e] - R.s * ve;
                rb[e * BJ_G] = R.s * a[e] + R.c * ve;
                a[e] = an;
              }
              aa = fmax(aa - R.t * ab, 0.0);
              if (lane == 0) {
                B[data_sz + j] = fmax(bb + R.t * ab, 0.0);
                if (R.big) ++mybig;
              }
            }
          }
          j = (j + 1 == b) ? 0 : j + 1;
          __syncthreads();
        }
        if (have) {
#pragma unroll
          for (int e = 0; e < EPL; ++e) rt[e * BJ_G] = a[e];
          if (lane == 0) T[data_sz + i] = aa;
        }
      }
      __syncthreads();
      if (Ce == 1) break;
      // ---- move the blocks one seat (labels of every peer are a function of the round number only)
      const int tt = sweep * (2 * Ce - 1) + t;  // exchanges done so far
      // peer labelling after tt relabels: CTA 0: top fixed at slot 0, (bot, spare) = tt even ? (1, 2) : (2, 1);
      // CTA c >= 1: (top, bot, spare) = cyclic shifts of (0, 1, 2)
      auto peer_top = [&](int c2) { return c2 == 0 ? 0 : (2 * tt) % 3; };
      auto peer_bot = [&](int c2) { return c2 == 0 ? ((tt & 1) ? 2 : 1) : (2 * tt + 1) % 3; };
      auto pull = [&](double* dst, const double* remote) {
        for (int idx = tid * 2; idx < b * pitch; idx += BJ_NT * 2)
          *reinterpret_cast<double2*>(dst + idx) = *reinterpret_cast<const double2*>(remote + idx);
        for (int idx = tid; idx < b; idx += BJ_NT) dst[data_sz + idx] = remote[data_sz + idx];
      };
      cluster.sync();  // every CTA has finished rotating its blocks
      // phase 1: new top <- old top of the left neighbour (CTA 1: old bot of CTA 0) into my spare slot
      if (rank >= 1) {
        const int src = rank - 1;
        const int ss = (rank == 1) ? peer_bot(0) : peer_top(src);
        pull(slot(spare_s), cluster.map_shared_rank(sm + (size_t)ss * slot_sz, src));
      }
      cluster.sync();
      // phase 2: new bot <- old bot of the right neighbour (last CTA: its own old top, a relabel)
      if (rank <= Ce - 2) {
        const int src = rank + 1;
        pull(slot(rank == 0 ? spare_s : top_s), cluster.map_shared_rank(sm + (size_t)peer_bot(src) * slot_sz, src));
      }
      cluster.sync();
      if (rank == 0) {
        const int ob = bot_s;
        bot_s = spare_s;
        spare_s = ob;
      } else {
        const int ot = top_s, ob = bot_s;
        top_s = spare_s;
        bot_s = ot;
        spare_s = ob;
      }
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
  // ---- after whole sweeps every block is back in its first seat
  for (int which = 0; which < 2; ++which) {
    const int blk = which == 0 ? rank : 2 * Ce - 1 - rank;
    const double* S = slot(which == 0 ? top_s : bot_s);
    for (int idx = tid; idx < b * pitch; idx += BJ_NT) {
      const int r = idx / pitch, x = idx - r * pitch;
      const int gr = blk * b + r;
      if (gr < p && x < q) P.X[(i64)gr * P.ld + x] = S[idx];
    }
  }
  if (rank == 0 && tid == 0 && P.status) {
    atomicMax(&P.status[0], sweep);
    if (hit_limit) atomicAdd(&P.status[1], 1);
  }
  if (Ce > 1) cluster.sync();
}

// ------------------------------------------------------------------------------------------------
// select: sort rows by norm (bitonic in shared memory), rank rule, normalised top rows.
constexpr int SNT = 256;
constexpr int SEL_MAXP = 16384;  // rows whose sort keys fit the opt-in shared memory (12 bytes per padded row)

// dynamic shared memory: key [np] doubles | idx [np] ints, np = rows padded to a power of two
__global__ void __launch_bounds__(SNT) qtt_select_kernel(const __grid_constant__ SelGroup g, int npmax) {
  const SelProb& P = g.p[blockIdx.x];
  extern __shared__ __align__(16) double sel_sm[];
  double* key = sel_sm;
  int* idx = reinterpret_cast<int*>(sel_sm + npmax);
  __shared__ int s_rank;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int p = P.p, q = P.q;
  int np = 1;
  while (np < p) np <<= 1;
  for (int r = warp; r < np; r += SNT / 32) {
    double s = 0.0;
    if (r < p)
      for (int x = lane; x < q; x += 32) {
        double v = P.X[(i64)r * P.ld + x];
        s += v * v;
      }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) {
      key[r] = (r < p) ? s : -1.0;
      idx[r] = r;
    }
  }
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
    for (int i = p - 1; i >= 0; --i) tot += key[i];
    if (P.delta_out) *P.delta_out = P.delta_scale * sqrt(tot);
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
    if (P.rank) P.rank[0] = r;
  }
  __syncthreads();
  const int r = s_rank;
  if (P.sigma)
    for (int i = tid; i < p; i += SNT) P.sigma[i] = sqrt(fmax(key[i], 0.0));
  for (int j = warp; j < P.r_cap; j += SNT / 32) {
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
    for (int x = lane; x < q; x += 32)
      P.out[(i64)j * P.out_ld + x] = (inv != 0.0) ? P.X[(i64)src * P.ld + x] * inv : 0.0;
  }
}

}  // namespace

namespace {
template <int EPL>
cudaError_t launch_blockjacobi(JacGroup& grp, int pmax, int qmax, int b, int pitch, size_t smem, double flops,
                               cudaStream_t stream) {
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_blockjacobi_kernel<EPL>))) {
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_blockjacobi_kernel<EPL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        224 * 1024));
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_blockjacobi_kernel<EPL>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grp.cluster * grp.nprob);
  cfg.blockDim = dim3(BJ_NT);
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
  return cudaLaunchKernelEx(&cfg, qtt_blockjacobi_kernel<EPL>, grp, b, pitch);
}

// Block-Jacobi configuration for a group with largest shape pmax x qmax; false if it does not fit.
// One warp per row pair (EPL = elements per lane); C = ceil(p / 16) CTAs (at most 16) of two blocks of 8 rows each
// for p <= 256 (measured ~10 % faster than 16-row blocks on half as many CTAs: two instead of four warps share an
// fp64 pipe), 16-row blocks on 16 CTAs for p = 512.
bool blockjacobi_config(int pmax, int qmax, int& EPL, int& C, int& b, int& pitch, size_t& smem) {
  if (qmax <= 128) EPL = 4;
  else if (qmax <= 256) EPL = 8;
  else if (qmax <= 512) EPL = 16;
  else return false;
  pitch = BJ_G * EPL;
  C = (pmax + 15) / 16;
  C = C < 1 ? 1 : (C > MAXC ? MAXC : C);
  b = (pmax + 2 * C - 1) / (2 * C);
  smem = ((size_t)3 * ((size_t)b * pitch + ((b + 1) & ~1)) + 3 * MAXC + 2) * sizeof(double);
  return smem <= 220 * 1024;
}
}  // namespace

cudaError_t qtt_launch_rowjacobi(const JacProb* probs, int n, cudaStream_t stream) {
  // production path: the register-blocked cluster block Jacobi (bj2.cu); problems of one call (the operands of one
  // site, similar shapes) share launches
  static const bool use_old = getenv("QTT_OLD_BJ") != nullptr;
  if (!use_old) {
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
  if (use_old) {
    int done = 0;
    bool all_fit = true;
    for (int i = 0; i < n && all_fit; ++i) {
      int EPL, C, b, pitch;
      size_t smem;
      if (probs[i].p >= 2 && probs[i].q >= 1 && !blockjacobi_config(probs[i].p, probs[i].q, EPL, C, b, pitch, smem))
        all_fit = false;
    }
    if (all_fit) {
      while (done < n) {
        JacGroup grp;
        grp.nprob = 0;
        int pmax = 0, qmax = 0;
        double flops = 0.0;
        while (done < n && grp.nprob < QTT_JAC_MAX_BATCH) {
          const JacProb& pr = probs[done];
          if (pr.p >= 2 && pr.q >= 1) {
            const int pm = pr.p > pmax ? pr.p : pmax, qm = pr.q > qmax ? pr.q : qmax;
            int EPL, C, b, pitch;
            size_t smem;
            if (grp.nprob > 0 && !blockjacobi_config(pm, qm, EPL, C, b, pitch, smem)) break;
            grp.p[grp.nprob++] = pr;
            pmax = pm;
            qmax = qm;
            double a = pr.p > pr.q ? pr.p : pr.q, bb = pr.p > pr.q ? pr.q : pr.p;
            flops += 6.0 * a * bb * bb + 20.0 * bb * bb * bb;
          }
          ++done;
        }
        if (grp.nprob == 0) continue;
        int EPL, C, b, pitch;
        size_t smem;
        blockjacobi_config(pmax, qmax, EPL, C, b, pitch, smem);
        grp.cluster = C;
        grp.use_smem = 1;
        grp.wslice = 0;
        grp.max_sweeps = 60;
        cudaError_t e;
        if (EPL == 4) e = launch_blockjacobi<4>(grp, pmax, qmax, b, pitch, smem, flops, stream);
        else if (EPL == 8) e = launch_blockjacobi<8>(grp, pmax, qmax, b, pitch, smem, flops, stream);
        else e = launch_blockjacobi<16>(grp, pmax, qmax, b, pitch, smem, flops, stream);
        if (e != cudaSuccess) return e;
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
    {
      QttProf prof(QK_SELECT, stream, bytes, g.p[0].p, g.p[0].q, g.nprob, 0);
      qtt_select_kernel<<<g.nprob, SNT, smem, stream>>>(g, npmax);
    }
    QTT_CHECK_CUDA(cudaGetLastError());
  }
  return cudaSuccess;
}
