// Turbulent-kinetic-energy spectrum of a velocity field (Eq. 13-15):
//   E(k1, k2) = 1/2 (|u1'^(k1, k2)|^2 + |u2'^(k1, k2)|^2),   E(k) = sum over the shell round(|k|) = k,
// u'^ the Fourier coefficients (1/N^2) sum_x u'(x) exp(-2 pi i k.x) of the fluctuating part u' = u - u_mean on the
// N x N periodic grid.  A diagnostic, not on the time-step path: dense fields (qtt_to_dense), a radix-2 FFT in shared
// memory (one CTA per row, the transform of the other direction after a transpose), shells accumulated in a fixed order
// (no floating-point atomics: the result is bit-reproducible).
#include "common.cuh"

namespace {

constexpr int FNT = 256;

// In-place FFT of every row of a complex N x N array (N = 2^logN <= 4096); if re_in != nullptr the rows are read from
// the real array re_in instead (imaginary part zero).  Decimation in time: bit-reversed load, logN butterfly stages.
__global__ void __launch_bounds__(FNT) qtt_fft_rows_kernel(const double* re_in, double2* data, int N, int logN) {
  extern __shared__ __align__(16) double2 row[];
  const int r = blockIdx.x;
  for (int i = threadIdx.x; i < N; i += FNT) {
    const int j = (int)(__brev((unsigned)i) >> (32 - logN));
    double2 v;
    if (re_in) v = make_double2(re_in[(i64)r * N + i], 0.0);
    else v = data[(i64)r * N + i];
    row[j] = v;
  }
  __syncthreads();
  for (int s = 1; s <= logN; ++s) {
    const int m = 1 << s, half = m >> 1;
    for (int b = threadIdx.x; b < N / 2; b += FNT) {
      const int pos = b & (half - 1);
      const int i0 = ((b >> (s - 1)) << s) + pos, i1 = i0 + half;
      double sn, cs;
      sincospi(-2.0 * (double)pos / (double)m, &sn, &cs);
      const double2 a = row[i0], x = row[i1];
      const double2 t = make_double2(x.x * cs - x.y * sn, x.x * sn + x.y * cs);
      row[i0] = make_double2(a.x + t.x, a.y + t.y);
      row[i1] = make_double2(a.x - t.x, a.y - t.y);
    }
    __syncthreads();
  }
  for (int i = threadIdx.x; i < N; i += FNT) data[(i64)r * N + i] = row[i];
}

__global__ void qtt_ctranspose_kernel(const double2* src, double2* dst, int N) {
  __shared__ double2 tile[16][17];
  const int x = blockIdx.x * 16 + threadIdx.x, y = blockIdx.y * 16 + threadIdx.y;
  if (x < N && y < N) tile[threadIdx.y][threadIdx.x] = src[(i64)y * N + x];
  __syncthreads();
  const int tx = blockIdx.y * 16 + threadIdx.x, ty = blockIdx.x * 16 + threadIdx.y;
  if (tx < N && ty < N) dst[(i64)ty * N + tx] = tile[threadIdx.x][threadIdx.y];
}

// partial[r][b] = sum over the columns c of row r with shell(r, c) == b of  (|U1|^2 + |U2|^2) * scale, columns in
// increasing order; thread t owns the shells t, t + FNT, ...
__global__ void __launch_bounds__(FNT) qtt_tke_rows_kernel(const double2* U1, const double2* U2, int N, int nbins,
                                                           double scale, double* partial) {
  const int r = blockIdx.x;
  const int ka = r < N / 2 ? r : r - N;
  for (int b = threadIdx.x; b < nbins; b += FNT) {
    double s = 0.0;
    // columns whose shell can be b: |kb| in [sqrt((b-.5)^2 - ka^2), sqrt((b+.5)^2 - ka^2)); scanning all keeps it simple
    for (int c = 0; c < N; ++c) {
      const int kb = c < N / 2 ? c : c - N;
      const int shell = (int)floor(sqrt((double)ka * ka + (double)kb * kb) + 0.5);
      if (shell == b) {
        const double2 a = U1[(i64)r * N + c], d = U2[(i64)r * N + c];
        s += (a.x * a.x + a.y * a.y) + (d.x * d.x + d.y * d.y);
      }
    }
    partial[(i64)r * nbins + b] = s * scale;
  }
}

__global__ void qtt_tke_sum_kernel(const double* partial, int N, int nbins, double* E) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nbins) return;
  double s = 0.0;
  for (int r = 0; r < N; ++r) s += partial[(i64)r * nbins + b];
  E[b] = s;
}

}  // namespace

// 2-D DFT of the real N x N field F into out (complex, TRANSPOSED wave-number order out[k2][k1]); tmp: N*N complex.
cudaError_t qtt_launch_fft2_real(const double* F, double* out_c, double* tmp_c, int nbits, cudaStream_t stream) {
  const int N = 1 << nbits;
  if (nbits < 1 || nbits > 12) return cudaErrorInvalidValue;
  double2* out = reinterpret_cast<double2*>(out_c);
  double2* tmp = reinterpret_cast<double2*>(tmp_c);
  const size_t smem = (size_t)N * sizeof(double2);
  if (qtt_first_use_on_device(reinterpret_cast<const void*>(&qtt_fft_rows_kernel)))
    QTT_CHECK_CUDA(cudaFuncSetAttribute(qtt_fft_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 4096 * 16));
  {
    QttProf prof(QK_MOVE, stream, 24.0 * N * N);
    qtt_fft_rows_kernel<<<N, FNT, smem, stream>>>(F, tmp, N, nbits);
  }
  {
    QttProf prof(QK_MOVE, stream, 32.0 * N * N);
    qtt_ctranspose_kernel<<<dim3((N + 15) / 16, (N + 15) / 16), dim3(16, 16), 0, stream>>>(tmp, out, N);
  }
  {
    QttProf prof(QK_MOVE, stream, 32.0 * N * N);
    qtt_fft_rows_kernel<<<N, FNT, smem, stream>>>(nullptr, out, N, nbits);
  }
  return cudaGetLastError();
}

// E[b] = 1/2 sum_{shell(k) = b} (|U1(k)|^2 + |U2(k)|^2) / N^4 from the unnormalised transforms; partial: N * nbins doubles.
cudaError_t qtt_launch_tke_shells(const double* U1_c, const double* U2_c, int nbits, int nbins, double* partial,
                                  double* E_dev, cudaStream_t stream) {
  const int N = 1 << nbits;
  const double n2 = (double)N * (double)N;
  {
    QttProf prof(QK_MOVE, stream, 32.0 * N * N);
    qtt_tke_rows_kernel<<<N, FNT, 0, stream>>>(reinterpret_cast<const double2*>(U1_c),
                                               reinterpret_cast<const double2*>(U2_c), N, nbins, 0.5 / (n2 * n2), partial);
  }
  {
    QttProf prof(QK_MOVE, stream, 8.0 * N * nbins);
    qtt_tke_sum_kernel<<<(nbins + 127) / 128, 128, 0, stream>>>(partial, N, nbins, E_dev);
  }
  return cudaGetLastError();
}
