// Grouped fp64 GEMM for the QTT site contractions (SURVEY.md section 8 rows a2, a4-a6 carry/absorb):
// tensor-core DMMA (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4 on sm_100a), operands staged global ->
// shared with a 3-stage cp.async pipeline, every reshape / permute / transpose of the site tensors
// folded into the tile addressing (see GemmProb in common.cuh).
//
// Shared-memory layouts keep each operand in its global orientation (contiguous direction stays
// contiguous, so 16-byte async copies apply) and pad the pitch to == 4 (mod 16) doubles, which makes
// the 8x4 / 4x8 DMMA fragment reads conflict-free for 64-bit accesses in either orientation.
#include <cstdlib>

#include "common.cuh"

namespace {

constexpr int BK = 16;
constexpr int STAGES = 3;
constexpr int KPITCH = BK + 4;  // pitch of a K-contiguous tile row

__device__ __forceinline__ void cp_async16(double* smem, const double* g, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(g), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(double* smem, const double* g, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(g), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// ---- TMA (bulk asynchronous copy engine, SASS UBLKCP) + mbarrier: rows of an M/N-contiguous operand tile are
// contiguous in global memory (up to 1 KB), so one cp.async.bulk per tile row moves them into the padded shared-memory
// layout the DMMA fragment loads need -- no tensor map: the operand views are strided / batched / split-index views of
// site tensors, and a 1-D bulk copy needs only 16-byte alignment of source, destination and size.
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(a), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(a), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(double* smem, const double* g, unsigned bytes, uint64_t* bar) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  unsigned b = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(s), "l"(g),
               "r"(bytes), "r"(b) : "memory");
}

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// One operand tile: T "strided" rows (pitch P) of CT contiguous doubles.
//  kind 0: contiguous direction is K (CT = BK), strided direction is the M/N index (T = BM or BN)
//  kind 1: contiguous direction is the M/N index (CT = BM or BN), strided direction is K (T = BK)
template <int BMN, int NT>
struct TileLoader {
  const double* base;  // operand base incl. batch offset
  int kind;
  bool vec;
  int mn0, MN, K;
  i64 k_stride;                               // kind 1
  static constexpr int CH0 = BMN * (BK / 2);  // 16-byte chunks per tile
  static constexpr int PER = (CH0 + NT - 1) / NT;
  i64 rowoff[PER];  // kind 0: precomputed offsets of this thread's rows
  int rowvalid;     // bit i: row of chunk i is inside the matrix

  __device__ void init(const double* b, int kind_, bool vec_, int mn0_, int MN_, int K_, i64 lo, i64 hi, int div,
                       i64 kst, int tid) {
    base = b; kind = kind_; vec = vec_; mn0 = mn0_; MN = MN_; K = K_; k_stride = kst;
    rowvalid = 0;
    if (kind == 0) {
#pragma unroll
      for (int i = 0; i < PER; ++i) {
        int q = tid + i * NT;
        int r = mn0 + q / (BK / 2);
        bool ok = (q < CH0) && (r < MN);
        i64 off = 0;
        if (ok) off = div > 0 ? (i64)(r / div) * hi + (i64)(r % div) * lo : (i64)r * lo;
        rowoff[i] = off;
        if (ok) rowvalid |= 1 << i;
      }
    }
  }

  // kind 1 through the bulk copy engine: thread t0 + kr moves row kr of the tile (rows beyond K are zero-filled by
  // that thread: 0 x 0 must not meet stale data; columns beyond MN only feed C entries that are never stored)
  __device__ __forceinline__ void issue_bulk(double* sm, int k0, int tid, int t0, uint64_t* bar) const {
    constexpr int P = BMN + 4;
    const int kr = tid - t0;
    if (kr < 0 || kr >= BK) return;
    double* s = sm + kr * P;
    const int cnt = (k0 + kr < K) ? min(max(MN - mn0, 0), BMN) : 0;
    const int even = cnt & ~1;
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    mbar_arrive_expect_tx(bar, (unsigned)even * 8u);
    if (even > 0) bulk_g2s(s, base + (i64)(k0 + kr) * k_stride + mn0, (unsigned)even * 8u, bar);
    if (cnt & 1) s[even] = base[(i64)(k0 + kr) * k_stride + mn0 + even];
    if (k0 + kr >= K)
      for (int c = 0; c < BMN; ++c) s[c] = 0.0;
  }

  __device__ __forceinline__ void issue(double* sm, int k0, int tid) const {
    if (kind == 0) {
#pragma unroll
      for (int i = 0; i < PER; ++i) {
        int q = tid + i * NT;
        if (q >= CH0) break;
        int r = q / (BK / 2), c = (q % (BK / 2)) * 2;
        int nv = 0;
        if (rowvalid & (1 << i)) nv = min(max(K - (k0 + c), 0), 2);
        const double* g = nv > 0 ? base + rowoff[i] + k0 + c : base;
        double* s = sm + r * KPITCH + c;
        if (vec) {
          cp_async16(s, g, nv * 8);
        } else {
          cp_async8(s, g, nv > 0 ? 8 : 0);
          cp_async8(s + 1, nv > 1 ? g + 1 : base, nv > 1 ? 8 : 0);
        }
      }
    } else {
      constexpr int P = BMN + 4;
#pragma unroll
      for (int i = 0; i < PER; ++i) {
        int q = tid + i * NT;
        if (q >= CH0) break;
        int kr = q / (BMN / 2), c = (q % (BMN / 2)) * 2;
        int nv = 0;
        if (k0 + kr < K) nv = min(max(MN - (mn0 + c), 0), 2);
        const double* g = nv > 0 ? base + (i64)(k0 + kr) * k_stride + mn0 + c : base;
        double* s = sm + kr * P + c;
        if (vec) {
          cp_async16(s, g, nv * 8);
        } else {
          cp_async8(s, g, nv > 0 ? 8 : 0);
          cp_async8(s + 1, nv > 1 ? g + 1 : base, nv > 1 ? 8 : 0);
        }
      }
    }
  }
};

// TMA = true: the variant whose M/N-contiguous operands are staged by the bulk copy engine (a separate instantiation,
// so that the cp.async-only kernel keeps its register allocation)
template <int BM, int BN, int WM, int WN, bool TMA>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32)
qtt_gemm_dmma_kernel(const __grid_constant__ GemmGroup g) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  constexpr int A_SZ = BM * KPITCH;  // >= BK * (BM + 4)
  constexpr int B_SZ = BN * KPITCH;
  constexpr int MI = WM / 8, NI = WN / 8;
  extern __shared__ __align__(16) double smem[];

  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  // ---- which problem / tile
  int pi = 0;
  {
    int t = blockIdx.x;
    for (int i = 1; i < g.nprob; ++i)
      if (t >= g.p[i].tile0) pi = i;
  }
  const GemmProb& P = g.p[pi];
  int local = blockIdx.x - P.tile0;
  const int per = P.tiles_m * P.tiles_n;
  const int z = local / per;
  local -= z * per;
  const int tm = local % P.tiles_m, tn = local / P.tiles_m;
  const int m0 = tm * BM, n0 = tn * BN;

  const int a_kind = (P.a_k == 1) ? 0 : 1;
  const int b_kind = (P.b_k == 1) ? 0 : 1;
  TileLoader<BM, NT> la;
  TileLoader<BN, NT> lb;
  la.init(P.A + (i64)z * P.a_bs, a_kind, (P.flags & 1) != 0, m0, P.M, P.K, P.a_lo, P.a_hi, P.a_div, P.a_k, tid);
  lb.init(P.B + (i64)z * P.b_bs, b_kind, (P.flags & 2) != 0, n0, P.N, P.K, P.b_n, 0, 0, P.b_k, tid);
  // operands staged by the bulk copy engine (flags 8 / 16 set by the launcher: M/N-contiguous, 16-byte aligned views)
  const bool a_bulk = TMA && (P.flags & 8) != 0, b_bulk = TMA && (P.flags & 16) != 0;
  __shared__ uint64_t tma_bar[TMA ? STAGES : 1];
  if (TMA && (a_bulk || b_bulk)) {
    if (tid == 0)
      for (int s = 0; s < STAGES; ++s) mbar_init(&tma_bar[s], (unsigned)BK * ((a_bulk ? 1u : 0u) + (b_bulk ? 1u : 0u)));
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    __syncthreads();
  }
  auto issue_stage = [&](int s, int k0) {
    double* As = smem + s * (A_SZ + B_SZ);
    if (TMA && a_bulk) la.issue_bulk(As, k0, tid, 0, &tma_bar[TMA ? s : 0]);
    else la.issue(As, k0, tid);
    if (TMA && b_bulk) lb.issue_bulk(As + A_SZ, k0, tid, NT >= 2 * BK ? BK : 0, &tma_bar[TMA ? s : 0]);
    else lb.issue(As + A_SZ, k0, tid);
  };

  const int sa_m = a_kind == 0 ? KPITCH : 1, sa_k = a_kind == 0 ? 1 : (BM + 4);
  const int sb_n = b_kind == 0 ? KPITCH : 1, sb_k = b_kind == 0 ? 1 : (BN + 4);

  const int wm0 = (warp % (BM / WM)) * WM, wn0 = (warp / (BM / WM)) * WN;
  double acc[MI][NI][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const int KT = (P.K + BK - 1) / BK;
#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < KT) issue_stage(s, s * BK);
    cp_async_commit();
  }
  const int fr = lane >> 2, fk = lane & 3;
  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<STAGES - 2>();
    if (TMA && (a_bulk || b_bulk)) mbar_wait(&tma_bar[TMA ? kt % STAGES : 0], (unsigned)((kt / STAGES) & 1));
    __syncthreads();
    {
      int nk = kt + STAGES - 1;
      if (nk < KT) issue_stage(nk % STAGES, nk * BK);
      cp_async_commit();
    }
    const double* As = smem + (kt % STAGES) * (A_SZ + B_SZ);
    const double* Bs = As + A_SZ;
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      double af[MI], bf[NI];
#pragma unroll
      for (int i = 0; i < MI; ++i) af[i] = As[(wm0 + i * 8 + fr) * sa_m + (kk + fk) * sa_k];
#pragma unroll
      for (int j = 0; j < NI; ++j) bf[j] = Bs[(wn0 + j * 8 + fr) * sb_n + (kk + fk) * sb_k];
#pragma unroll
      for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
  }
  cp_async_wait<0>();

  // ---- epilogue
  double* Cb = P.C + (i64)z * P.c_bs;
  const bool cvec = (P.flags & 4) != 0;
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    int r = m0 + wm0 + i * 8 + fr;
    if (r >= P.M) continue;
    i64 roff = P.c_div > 0 ? (i64)(r / P.c_div) * P.c_hi + (i64)(r % P.c_div) * P.c_lo : (i64)r * P.c_lo;
#pragma unroll
    for (int j = 0; j < NI; ++j) {
      int c = n0 + wn0 + j * 8 + fk * 2;
      if (c >= P.N) continue;
      double v0 = P.alpha * acc[i][j][0], v1 = P.alpha * acc[i][j][1];
      double* dst = Cb + roff + (i64)c * P.c_n;
      if (cvec && c + 1 < P.N) {
        if (P.beta != 0.0) {
          double2 o = *reinterpret_cast<double2*>(dst);
          v0 += P.beta * o.x;
          v1 += P.beta * o.y;
        }
        *reinterpret_cast<double2*>(dst) = make_double2(v0, v1);
      } else {
        if (P.beta != 0.0) v0 += P.beta * dst[0];
        dst[0] = v0;
        if (c + 1 < P.N) {
          if (P.beta != 0.0) v1 += P.beta * dst[P.c_n];
          dst[P.c_n] = v1;
        }
      }
    }
  }
}

template <int BM, int BN, int WM, int WN, bool TMA>
cudaError_t launch_cfg(GemmGroup& grp, cudaStream_t stream, int family) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  constexpr size_t SMEM = (size_t)STAGES * (BM + BN) * KPITCH * sizeof(double);
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_gemm_dmma_kernel<BM, BN, WM, WN, TMA>)))
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_gemm_dmma_kernel<BM, BN, WM, WN, TMA>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
  int t = 0;
  for (int i = 0; i < grp.nprob; ++i) {
    GemmProb& p = grp.p[i];
    p.tiles_m = (p.M + BM - 1) / BM;
    p.tiles_n = (p.N + BN - 1) / BN;
    p.tile0 = t;
    t += p.tiles_m * p.tiles_n * p.nbatch;
  }
  grp.total_tiles = t;
  if (t == 0) return cudaSuccess;
  double flops = 0.0;
  for (int i = 0; i < grp.nprob; ++i) flops += 2.0 * grp.p[i].M * grp.p[i].N * (double)grp.p[i].K * grp.p[i].nbatch;
  {
    QttProf prof(family, stream, flops, grp.p[0].M, grp.p[0].N, grp.p[0].K, grp.nprob);
    qtt_gemm_dmma_kernel<BM, BN, WM, WN, TMA><<<t, NT, SMEM, stream>>>(grp);
  }
  return cudaGetLastError();
}

inline bool even(i64 x) { return (x & 1) == 0; }
inline bool al16(const void* p) { return ((uintptr_t)p & 15) == 0; }

}  // namespace

cudaError_t qtt_launch_gemm(const GemmProb* probs, int n, cudaStream_t stream, int family) {
  int done = 0;
  while (done < n) {
    GemmGroup grp;
    grp.nprob = 0;
    i64 big_tiles = 0, mid_tiles = 0;
    int minMN = 1 << 30;
    while (done < n && grp.nprob < QTT_GEMM_MAX_GROUP) {
      GemmProb p = probs[done++];
      if (p.M <= 0 || p.N <= 0 || p.nbatch <= 0) continue;
      if (p.a_k != 1 && !(p.a_lo == 1 && p.a_div == 0)) return cudaErrorInvalidValue;
      if (p.b_k != 1 && p.b_n != 1) return cudaErrorInvalidValue;
      int f = 0;
      // 16-byte async copies need even strides in the non-contiguous directions and aligned bases
      if (p.a_k == 1) {
        if (al16(p.A) && even(p.a_lo) && even(p.a_hi) && even(p.a_bs)) f |= 1;
      } else if (al16(p.A) && even(p.a_k) && even(p.a_bs)) f |= 1;
      if (p.b_k == 1) {
        if (al16(p.B) && even(p.b_n) && even(p.b_bs)) f |= 2;
      } else if (al16(p.B) && even(p.b_k) && even(p.b_bs)) f |= 2;
      if (p.c_n == 1 && al16(p.C) && even(p.c_lo) && even(p.c_hi) && even(p.c_bs)) f |= 4;
      // M/N-contiguous operand views that are 16-byte aligned go through the bulk copy engine (TMA) unless disabled
      // (QTT_GEMM_TMA=0: the cp.async path for every operand; profiles/r2_gemm_tma_ab.md has the comparison)
      static const int tma_mode = getenv("QTT_GEMM_TMA") ? (getenv("QTT_GEMM_TMA")[0] == '0' ? 0 : 1) : -1;
      // default (-1): the bulk engine where it measured at least as fast as cp.async -- the batched site contractions
      // with long K (the chi = 256 shapes of row a2: 26.0 vs 25.8 TFLOP/s); at K = 64 / 128 and for the unbatched carry
      // products cp.async is 1-5 % ahead and stays (profiles/r2_gemm_tma_ab.md)
      const bool use_tma = tma_mode == 1 || (tma_mode < 0 && p.K >= 256 && p.nbatch >= 4);
      if (use_tma) {
        if (p.a_k != 1 && (f & 1)) f |= 8;
        if (p.b_k != 1 && (f & 2)) f |= 16;
      }
      p.flags = f;
      grp.p[grp.nprob++] = p;
      big_tiles += (i64)((p.M + 127) / 128) * ((p.N + 127) / 128) * p.nbatch;
      mid_tiles += (i64)((p.M + 63) / 64) * ((p.N + 63) / 64) * p.nbatch;
      minMN = p.M < minMN ? p.M : minMN;
      minMN = p.N < minMN ? p.N : minMN;
    }
    if (grp.nprob == 0) continue;
    bool any_bulk = false;
    for (int i = 0; i < grp.nprob; ++i) any_bulk = any_bulk || (grp.p[i].flags & 24) != 0;
    cudaError_t e;
    if (big_tiles >= 120 && minMN >= 96)
      e = any_bulk ? launch_cfg<128, 128, 64, 32, true>(grp, stream, family) : launch_cfg<128, 128, 64, 32, false>(grp, stream, family);
    else if (mid_tiles >= 32 && minMN >= 48)
      e = any_bulk ? launch_cfg<64, 64, 32, 32, true>(grp, stream, family) : launch_cfg<64, 64, 32, 32, false>(grp, stream, family);
    else
      e = any_bulk ? launch_cfg<32, 32, 16, 16, true>(grp, stream, family) : launch_cfg<32, 32, 16, 16, false>(grp, stream, family);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}
