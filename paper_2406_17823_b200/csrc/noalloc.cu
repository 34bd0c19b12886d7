// qtt_lq_noalloc (include/qtt_diag.h): the Q-less LQ of qtt_diag_lq for callers that cannot allocate device memory
// (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same kernels, same launch
// sequence (lq.cu / qrcp.cu); the only difference is where the scratch of the blocked path (V, T V and the products
// X V^T with their K-chunk partials: 3 x 64 x m doubles per matrix) lives: in the file-scope device array below instead
// of a buffer the caller allocates.
//
// The array is part of the library image: every GPU that loads the library holds its 6 MiB until the process exits.
// In HOST code its name is a host-side stand-in, not a device address -- the device address is taken once per device
// with cudaGetSymbolAddress (that device current) and passed to the kernels like any other pointer.
// All calls share the array and it keeps the last call's contents: the part a call uses is cleared on the call's stream
// first, and two calls that overlap on the GPU (different streams, no dependency) race on it.
#include <cstdio>
#include <mutex>

#include "../../include/qtt_diag.h"
#include "common.cuh"

namespace {

static_assert(QTT_LQ_NOALLOC_MAX_DOUBLES == 3 * 64 * 4096, "the header states the size of the scratch array");
static __device__ __align__(256) double qtt_lq_noalloc_scratch[QTT_LQ_NOALLOC_MAX_DOUBLES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double* g_scratch_ptr[MAX_DEVICES] = {};  // device address of the array, per device, taken at the first call there

// device address of the scratch array on the CURRENT device (no allocation: the array came with the module)
cudaError_t scratch_address(double** out) {
  int dev = -1;
  QTT_CHECK_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    double* p = nullptr;
    QTT_CHECK_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), qtt_lq_noalloc_scratch));
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" int qtt_lq_noalloc(void* stream, double* Y, int batch, int k, int m, int ld, double* R) {
  if (!Y || !R || batch < 1 || batch > QTT_LQ_MAX_BATCH || k < 1 || m < k || ld < m || m > 16384) {
    std::fprintf(stderr, "qtt_lq_noalloc: invalid argument (batch %d in 1..%d, 1 <= k %d <= m %d <= ld %d, m <= 16384)\n",
                 batch, QTT_LQ_MAX_BATCH, k, m, ld);
    return QTT_NOALLOC_BAD_ARG;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (qtt_qrcp_fits(m, k)) {  // the cluster-resident Householder kernel needs no scratch at all
    QrcpProb qp[QTT_LQ_MAX_BATCH];
    for (int i = 0; i < batch; ++i) qp[i] = QrcpProb{Y + (size_t)i * k * ld, m, k, ld, nullptr, 1, R + (size_t)i * k * k};
    return (int)qtt_launch_qrcp(qp, batch, 0, st);
  }
  const size_t s = qtt_lq_scratch_doubles(m);  // per matrix, for each of V, TV and W
  const size_t need = (size_t)batch * 3 * s;
  if (need > (size_t)QTT_LQ_NOALLOC_MAX_DOUBLES) {
    std::fprintf(stderr,
                 "qtt_lq_noalloc: batch %d x m %d needs %zu doubles of scratch, the built-in array holds %d (batch * m <= 4096); "
                 "use qtt_diag_lq with a caller-allocated buffer\n", batch, m, need, (int)QTT_LQ_NOALLOC_MAX_DOUBLES);
    return QTT_NOALLOC_TOO_LARGE;
  }
  double* scratch = nullptr;
  cudaError_t e = scratch_address(&scratch);
  if (e != cudaSuccess) return (int)e;
  // the array keeps the previous call's contents: clear what this call uses (stream-ordered, no allocation)
  e = cudaMemsetAsync(scratch, 0, need * sizeof(double), st);
  if (e != cudaSuccess) return (int)e;
  LqProb probs[QTT_LQ_MAX_BATCH];
  TriProb tris[QTT_LQ_MAX_BATCH];
  for (int i = 0; i < batch; ++i) {
    probs[i] = LqProb{};
    probs[i].Y = Y + (size_t)i * k * ld;
    probs[i].k = k; probs[i].m = m; probs[i].ld = ld;
    probs[i].V = scratch + (size_t)i * 3 * s;
    probs[i].TV = probs[i].V + s;
    probs[i].W = probs[i].TV + s;
    tris[i] = TriProb{probs[i].Y, k, ld, R + (size_t)i * k * k, k};
  }
  e = qtt_launch_lq(probs, batch, st);
  if (e != cudaSuccess) return (int)e;
  return (int)qtt_launch_extract_tri(tris, batch, 0, st);
}
