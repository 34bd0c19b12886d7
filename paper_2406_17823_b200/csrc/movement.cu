// Bandwidth-bound data movement of the QTT step (SURVEY.md section 8 rows a1, a3 and the boundary):
// MPO x MPS site expand, direct-sum concatenation, Hadamard (Kronecker) site tensors, the quantics
// bit interleave, transposes and copies.  All grid-stride, coalesced along the innermost index.
#include "common.cuh"

namespace {

constexpr int NT = 256;

inline int grid_for(i64 n) {
  i64 b = (n + NT - 1) / NT;
  const i64 cap = 148 * 16;
  return (int)(b < 1 ? 1 : (b > cap ? cap : b));
}

// out[(al,a), w, (be,b)] = sum_w' W[al,w,w',be] * A[a,w',b]      (MPO bond index major)
// (DP = physical dimension, a compile-time constant so that the index arithmetic stays shifts and the w' loop unrolls)
template <int DP>
__global__ void qtt_expand_kernel(const __grid_constant__ ExpandGroup g) {
  const ExpandProb& P = g.p[blockIdx.y];
  const int Dl = P.Dl, Dr = P.Dr, a = P.a, b = P.b;
  constexpr int d = DP;
  const i64 n = (i64)Dl * a * d * Dr * b;
  const i64 rowlen = (i64)Dr * b;
  for (i64 idx = (i64)blockIdx.x * NT + threadIdx.x; idx < n; idx += (i64)gridDim.x * NT) {
    i64 t = idx;
    int bb = (int)(t % b); t /= b;
    int be = (int)(t % Dr); t /= Dr;
    int w = (int)(t % d); t /= d;
    int aa = (int)(t % a);
    int al = (int)(t / a);
    double s = 0.0;
#pragma unroll
    for (int wp = 0; wp < d; ++wp) {
      double wv = P.W[((al * d + w) * d + wp) * Dr + be];
      if (wv != 0.0) s += wv * P.A[((i64)aa * d + wp) * b + bb];
    }
    P.out[idx] = s;
    (void)rowlen;
  }
}

template <int DP>
__global__ void qtt_concat_kernel(const __grid_constant__ ConcatGroup g) {
  const ConcatProb& P = g.p[blockIdx.y];
  int RL = 0, RR = 0;
  if (P.mode == 0) {
    RL = P.rl[0];
    for (int t = 0; t < P.nterm; ++t) RR += P.rr[t];
  } else if (P.mode == 2) {
    RR = P.rr[0];
    for (int t = 0; t < P.nterm; ++t) RL += P.rl[t];
  } else {
    for (int t = 0; t < P.nterm; ++t) {
      RL += P.rl[t];
      RR += P.rr[t];
    }
  }
  constexpr int d = DP;
  const i64 n = (i64)RL * d * RR;
  for (i64 idx = (i64)blockIdx.x * NT + threadIdx.x; idx < n; idx += (i64)gridDim.x * NT) {
    int c = (int)(idx % RR);
    i64 t2 = idx / RR;
    int w = (int)(t2 % d);
    int r = (int)(t2 / d);
    // locate the term of the row and of the column
    int tr = 0, tc = 0, r_in = r, c_in = c;
    if (P.mode != 0) {
      while (tr < P.nterm - 1 && r_in >= P.rl[tr]) { r_in -= P.rl[tr]; ++tr; }
    }
    if (P.mode != 2) {
      while (tc < P.nterm - 1 && c_in >= P.rr[tc]) { c_in -= P.rr[tc]; ++tc; }
    }
    double v = 0.0;
    if (P.mode == 0) {
      v = P.alpha[tc] * P.src[tc][((i64)r * d + w) * P.rr[tc] + c_in];
    } else if (P.mode == 2) {
      v = P.src[tr][((i64)r_in * d + w) * P.rr[tr] + c];
    } else if (tr == tc) {
      v = P.src[tr][((i64)r_in * d + w) * P.rr[tr] + c_in];
    }
    P.out[idx] = v;
  }
}

// out[(a,b), w, (a2,b2)] = A[a,w,a2] * B[b,w,b2]                  (Eq. 8)
template <int DP>
__global__ void qtt_kron_kernel(const __grid_constant__ KronGroup g) {
  const KronProb& P = g.p[blockIdx.y];
  constexpr int d = DP;
  const i64 n = (i64)P.a * P.b * d * P.a2 * P.b2;
  for (i64 idx = (i64)blockIdx.x * NT + threadIdx.x; idx < n; idx += (i64)gridDim.x * NT) {
    i64 t = idx;
    int bb2 = (int)(t % P.b2); t /= P.b2;
    int aa2 = (int)(t % P.a2); t /= P.a2;
    int w = (int)(t % d); t /= d;
    int bb = (int)(t % P.b);
    int aa = (int)(t / P.b);
    P.out[idx] = P.A[((i64)aa * d + w) * P.a2 + aa2] * P.B[((i64)bb * d + w) * P.b2 + bb2];
  }
}

// Quantics interleave (Eq. 3): tensor index t = (w_1 ... w_n)_4, w_k = 2 x_k + y_k, bit 1
// most significant;  dense index = x * N + y.
__device__ __forceinline__ unsigned compact_even_bits(unsigned long long v) {
  // gathers bits 0,2,4,... of v
  v &= 0x5555555555555555ull;
  v = (v | (v >> 1)) & 0x3333333333333333ull;
  v = (v | (v >> 2)) & 0x0f0f0f0f0f0f0f0full;
  v = (v | (v >> 4)) & 0x00ff00ff00ff00ffull;
  v = (v | (v >> 8)) & 0x0000ffff0000ffffull;
  v = (v | (v >> 16)) & 0x00000000ffffffffull;
  return (unsigned)v;
}
__global__ void qtt_interleave_kernel(const double* __restrict__ src, double* __restrict__ dst, int nbits,
                                      int inverse) {
  const i64 n = 1ll << (2 * nbits);
  for (i64 t = (i64)blockIdx.x * NT + threadIdx.x; t < n; t += (i64)gridDim.x * NT) {
    unsigned y = compact_even_bits((unsigned long long)t);
    unsigned x = compact_even_bits((unsigned long long)t >> 1);
    i64 d = ((i64)x << nbits) | y;
    if (inverse)
      dst[d] = src[t];  // tensor -> dense
    else
      dst[t] = src[d];  // dense -> tensor
  }
}
// Three coordinates (reading 26): t = (w_1 ... w_n)_8, w_k = 4 x_k + 2 y_k + z_k; dense index = (x * N + y) * N + z.
__global__ void qtt_interleave3_kernel(const double* __restrict__ src, double* __restrict__ dst, int nbits,
                                       int inverse) {
  const i64 n = 1ll << (3 * nbits);
  for (i64 t = (i64)blockIdx.x * NT + threadIdx.x; t < n; t += (i64)gridDim.x * NT) {
    i64 x = 0, y = 0, z = 0;
    for (int k = 0; k < nbits; ++k) {
      const i64 w = (t >> (3 * k)) & 7;  // site n - k: bit k of every coordinate
      x |= ((w >> 2) & 1) << k;
      y |= ((w >> 1) & 1) << k;
      z |= (w & 1) << k;
    }
    const i64 d = (((x << nbits) | y) << nbits) | z;
    if (inverse)
      dst[d] = src[t];
    else
      dst[t] = src[d];
  }
}

__global__ void qtt_transpose_kernel(const double* __restrict__ src, int rows, int cols, int lds,
                                     double* __restrict__ dst, int ldd) {
  __shared__ double tile[32][33];
  const int bx = blockIdx.y * 32, by = blockIdx.x * 32;  // x runs over row blocks (the long direction)
  for (int j = threadIdx.y; j < 32; j += 8) {
    int r = by + j, c = bx + threadIdx.x;
    if (r < rows && c < cols) tile[j][threadIdx.x] = src[(i64)r * lds + c];
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += 8) {
    int c = bx + j, r = by + threadIdx.x;  // dst row = c, dst col = r
    if (r < rows && c < cols) dst[(i64)c * ldd + r] = tile[threadIdx.x][j];
  }
}

__global__ void qtt_copy2d_kernel(const double* __restrict__ src, int rows, int cols, int lds,
                                  double* __restrict__ dst, int ldd) {
  const i64 n = (i64)rows * cols;
  for (i64 idx = (i64)blockIdx.x * NT + threadIdx.x; idx < n; idx += (i64)gridDim.x * NT) {
    int r = (int)(idx / cols), c = (int)(idx - (i64)r * cols);
    dst[(i64)r * ldd + c] = src[(i64)r * lds + c];
  }
}

__global__ void qtt_fill_kernel(double* dst, i64 n, double v) {
  for (i64 idx = (i64)blockIdx.x * NT + threadIdx.x; idx < n; idx += (i64)gridDim.x * NT) dst[idx] = v;
}

}  // namespace

cudaError_t qtt_launch_expand(const ExpandProb* probs, int n, cudaStream_t stream) {
  for (int b0 = 0; b0 < n; b0 += QTT_MOVE_MAX_BATCH) {
    ExpandGroup g;
    g.nprob = n - b0 < QTT_MOVE_MAX_BATCH ? n - b0 : QTT_MOVE_MAX_BATCH;
    i64 mx = 1;
    for (int i = 0; i < g.nprob; ++i) {
      g.p[i] = probs[b0 + i];
      if ((g.p[i].d != 4 && g.p[i].d != 8) || g.p[i].d != probs[b0].d) return cudaErrorInvalidValue;
      i64 sz = (i64)g.p[i].Dl * g.p[i].a * g.p[i].d * g.p[i].Dr * g.p[i].b;
      mx = sz > mx ? sz : mx;
    }
    {
      QttProf prof(QK_MOVE, stream, 16.0 * (double)mx * g.nprob);
      if (g.p[0].d == 8)
        qtt_expand_kernel<8><<<dim3(grid_for(mx), g.nprob), NT, 0, stream>>>(g);
      else
        qtt_expand_kernel<4><<<dim3(grid_for(mx), g.nprob), NT, 0, stream>>>(g);
    }
    QTT_CHECK_CUDA(cudaGetLastError());
  }
  return cudaSuccess;
}

cudaError_t qtt_launch_concat(const ConcatProb* probs, int n, cudaStream_t stream) {
  for (int b0 = 0; b0 < n; b0 += QTT_MOVE_MAX_BATCH) {
    ConcatGroup g;
    g.nprob = n - b0 < QTT_MOVE_MAX_BATCH ? n - b0 : QTT_MOVE_MAX_BATCH;
    i64 mx = 1;
    for (int i = 0; i < g.nprob; ++i) {
      g.p[i] = probs[b0 + i];
      if ((g.p[i].d != 4 && g.p[i].d != 8) || g.p[i].d != probs[b0].d) return cudaErrorInvalidValue;
      i64 RL = 0, RR = 0;
      for (int t = 0; t < g.p[i].nterm; ++t) {
        RL += g.p[i].rl[t];
        RR += g.p[i].rr[t];
      }
      i64 sz = RL * g.p[i].d * RR;
      mx = sz > mx ? sz : mx;
    }
    {
      QttProf prof(QK_MOVE, stream, 16.0 * (double)mx * g.nprob);
      if (g.p[0].d == 8)
        qtt_concat_kernel<8><<<dim3(grid_for(mx), g.nprob), NT, 0, stream>>>(g);
      else
        qtt_concat_kernel<4><<<dim3(grid_for(mx), g.nprob), NT, 0, stream>>>(g);
    }
    QTT_CHECK_CUDA(cudaGetLastError());
  }
  return cudaSuccess;
}

cudaError_t qtt_launch_kron(const KronProb* probs, int n, cudaStream_t stream) {
  for (int b0 = 0; b0 < n; b0 += QTT_MOVE_MAX_BATCH) {
    KronGroup g;
    g.nprob = n - b0 < QTT_MOVE_MAX_BATCH ? n - b0 : QTT_MOVE_MAX_BATCH;
    i64 mx = 1;
    for (int i = 0; i < g.nprob; ++i) {
      g.p[i] = probs[b0 + i];
      if ((g.p[i].d != 4 && g.p[i].d != 8) || g.p[i].d != probs[b0].d) return cudaErrorInvalidValue;
      i64 sz = (i64)g.p[i].a * g.p[i].b * g.p[i].d * g.p[i].a2 * g.p[i].b2;
      mx = sz > mx ? sz : mx;
    }
    {
      QttProf prof(QK_MOVE, stream, 8.0 * (double)mx * g.nprob);
      if (g.p[0].d == 8)
        qtt_kron_kernel<8><<<dim3(grid_for(mx), g.nprob), NT, 0, stream>>>(g);
      else
        qtt_kron_kernel<4><<<dim3(grid_for(mx), g.nprob), NT, 0, stream>>>(g);
    }
    QTT_CHECK_CUDA(cudaGetLastError());
  }
  return cudaSuccess;
}

cudaError_t qtt_launch_interleave(const double* src, double* dst, int nbits, int ndim, int inverse,
                                  cudaStream_t stream) {
  if ((ndim != 2 && ndim != 3) || nbits < 1 || ndim * nbits > 40) return cudaErrorInvalidValue;
  const i64 n = 1ll << (ndim * nbits);
  {
    QttProf prof(QK_MOVE, stream, 16.0 * (double)n);
    if (ndim == 3)
      qtt_interleave3_kernel<<<grid_for(n), NT, 0, stream>>>(src, dst, nbits, inverse);
    else
      qtt_interleave_kernel<<<grid_for(n), NT, 0, stream>>>(src, dst, nbits, inverse);
  }
  return cudaGetLastError();
}

cudaError_t qtt_launch_transpose(const double* src, int rows, int cols, int lds, double* dst, int ldd,
                                 cudaStream_t stream) {
  if (rows <= 0 || cols <= 0) return cudaSuccess;
  dim3 grid((rows + 31) / 32, (cols + 31) / 32);
  if (grid.y > 65535) return cudaErrorInvalidValue;
  {
    QttProf prof(QK_MOVE, stream, 16.0 * (double)rows * cols);
    qtt_transpose_kernel<<<grid, dim3(32, 8), 0, stream>>>(src, rows, cols, lds, dst, ldd);
  }
  return cudaGetLastError();
}

cudaError_t qtt_launch_copy2d(const double* src, int rows, int cols, int lds, double* dst, int ldd,
                              cudaStream_t stream) {
  if (rows <= 0 || cols <= 0) return cudaSuccess;
  {
    QttProf prof(QK_MOVE, stream, 16.0 * (double)rows * cols);
    qtt_copy2d_kernel<<<grid_for((i64)rows * cols), NT, 0, stream>>>(src, rows, cols, lds, dst, ldd);
  }
  return cudaGetLastError();
}

cudaError_t qtt_launch_fill(double* dst, i64 n, double value, cudaStream_t stream) {
  if (n <= 0) return cudaSuccess;
  {
    QttProf prof(QK_MOVE, stream, 8.0 * (double)n);
    qtt_fill_kernel<<<grid_for(n), NT, 0, stream>>>(dst, n, value);
  }
  return cudaGetLastError();
}

// Sign vectors of the sketched zip-up (reading 25): probe t carries at site `site` the sign vector
// Core of the random sign tensor train the sketched zip-up probes with (reading 25; oracle sketch_mixers):
// G[c][t] = +-scale, c = w * P + u < 4 P, t < P, minus where the top bit of the splitmix64 finaliser of
// seed * 0x9E3779B97F4A7C15 + site * 0xD1B54A32D192ED03 + c * 2^20 + t (mod 2^64) is set -- the counter-based generator the
// oracle implements too (oracle sketch_signs); scale = 1 / sqrt(P) is one correctly rounded double on both sides, so the
// two sides use bit-identical cores.
__global__ void qtt_sketch_mixers_kernel(unsigned long long base, double* G, i64 n, int P, double scale) {
  for (i64 idx = (i64)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (i64)gridDim.x * blockDim.x) {
    const unsigned long long t = (unsigned long long)(idx % P);
    const unsigned long long c = (unsigned long long)(idx / P);
    unsigned long long z = base + (c << 20) + t;
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    G[idx] = (z >> 63) ? -scale : scale;
  }
}
cudaError_t qtt_launch_sketch_mixers(unsigned long long seed, int site, double* G, int P, cudaStream_t stream) {
  const i64 n = 4ll * P * P;
  if (n <= 0) return cudaSuccess;
  if (P >= (1 << 20)) return cudaErrorInvalidValue;
  const unsigned long long base = seed * 0x9E3779B97F4A7C15ull + (unsigned long long)site * 0xD1B54A32D192ED03ull;
  int blocks = (int)((n + 255) / 256);
  blocks = blocks > 148 * 8 ? 148 * 8 : blocks;
  QttProf prof(QK_MOVE, stream, 8.0 * (double)n);
  qtt_sketch_mixers_kernel<<<blocks, 256, 0, stream>>>(base, G, n, P, 1.0 / sqrt((double)P));
  return cudaGetLastError();
}
