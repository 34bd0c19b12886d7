// fp64 issue-rate probes (include/qtt_diag.h: qtt_diag_fp64_probe) -- the measured denominators of the
// fp64 roofline (MEASURED_PEAKS.json carries no fp64 figure), the per-context launch
// counter / profiler records and the per-device kernel-attribute bookkeeping.
#include <cstdio>
#include <mutex>
#include <set>
#include <utility>
#include <vector>

#include "../../include/qtt_diag.h"
#include "common.cuh"

namespace {

// 16 independent DMMA.8x8x4 accumulator pairs per warp, 4 rounds per iteration = 64 DMMA per warp-iteration
__global__ void __launch_bounds__(256) qtt_probe_dmma_kernel(int iters, double* sink) {
  double d0[16], d1[16];
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
#pragma unroll
  for (int i = 0; i < 16; ++i) d0[i] = d1[i] = (double)i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int i = 0; i < 16; ++i)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                     : "+d"(d0[i]), "+d"(d1[i])
                     : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += d0[i] + d1[i];
  if (s == 123.456) sink[0] = s;
}

// 16 independent DFMA chains per thread, 4 rounds per iteration = 64 DFMA per thread-iteration
__global__ void __launch_bounds__(256) qtt_probe_dfma_kernel(int iters, double* sink) {
  double d[16];
  double a = 1.0 + threadIdx.x * 1e-12, b = 1e-9 * threadIdx.x;
#pragma unroll
  for (int i = 0; i < 16; ++i) d[i] = (double)i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int i = 0; i < 16; ++i) d[i] = fma(d[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += d[i];
  if (s == 123.456) sink[0] = s;
}

}  // namespace

// ------------------------------------------------------------------------------------------ per-context stats
namespace {
QttStats g_default_stats;
thread_local QttStats* t_stats = nullptr;
std::vector<QttProfRec>& recs_of(QttStats* s) {
  if (!s->recs) s->recs = new std::vector<QttProfRec>();
  return *static_cast<std::vector<QttProfRec>*>(s->recs);
}
std::mutex g_attr_mu;
std::set<std::pair<int, const void*>> g_attr_seen;
}  // namespace

QttStats* qtt_stats_current() { return t_stats ? t_stats : &g_default_stats; }
void qtt_stats_bind(QttStats* s) { t_stats = s; }
void qtt_stats_destroy(QttStats* s) {
  if (!s) return;
  if (s->recs) {
    for (QttProfRec& r : recs_of(s)) {
      cudaEventDestroy(r.e0);
      cudaEventDestroy(r.e1);
    }
    delete static_cast<std::vector<QttProfRec>*>(s->recs);
    s->recs = nullptr;
  }
  if (t_stats == s) t_stats = nullptr;
}

bool qtt_first_use_on_device(const void* key) {
  int dev = 0;
  cudaGetDevice(&dev);
  std::lock_guard<std::mutex> lock(g_attr_mu);
  return g_attr_seen.insert({dev, key}).second;
}

QttProf::QttProf(int family, cudaStream_t stream, double work, int d0, int d1, int d2, int d3)
    : stats(qtt_stats_current()), st(stream), live(false) {
  ++stats->launches;
  if (!stats->prof_on) return;
  QttProfRec r;
  r.fam = family;
  r.work = work;
  r.d[0] = d0; r.d[1] = d1; r.d[2] = d2; r.d[3] = d3;
  if (cudaEventCreate(&r.e0) != cudaSuccess) return;
  if (cudaEventCreate(&r.e1) != cudaSuccess) {
    cudaEventDestroy(r.e0);
    return;
  }
  live = true;
  cudaEventRecord(r.e0, st);
  recs_of(stats).push_back(r);
}
QttProf::~QttProf() {
  if (live) cudaEventRecord(recs_of(stats).back().e1, st);
}
cudaError_t qtt_prof_collect(QttStats* s, double ms[QK_COUNT], double work[QK_COUNT], long long launches[QK_COUNT]) {
  for (int i = 0; i < QK_COUNT; ++i) ms[i] = work[i] = 0.0, launches[i] = 0;
  cudaError_t e = cudaDeviceSynchronize();
  for (QttProfRec& r : recs_of(s)) {
    float t = 0.f;
    if (e == cudaSuccess && cudaEventElapsedTime(&t, r.e0, r.e1) == cudaSuccess) {
      ms[r.fam] += t;
      work[r.fam] += r.work;
      launches[r.fam] += 1;
    }
    cudaEventDestroy(r.e0);
    cudaEventDestroy(r.e1);
  }
  recs_of(s).clear();
  return e;
}

// writes the records of the calling thread's current context (the context of its last qtt_* call)
extern "C" int qtt_diag_profile_dump(const char* path_host) {
  if (!path_host) return (int)cudaErrorInvalidValue;
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) return (int)e;
  FILE* f = fopen(path_host, "w");
  if (!f) return (int)cudaErrorInvalidValue;
  static const char* names[QK_COUNT] = {"gemm", "lq_panel", "lq_update", "rowjacobi", "select", "move", "qrcp"};
  fprintf(f, "family,d0,d1,d2,d3,ms,work\n");
  for (QttProfRec& r : recs_of(qtt_stats_current())) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.e0, r.e1) != cudaSuccess) continue;
    fprintf(f, "%s,%d,%d,%d,%d,%.6f,%.6g\n", names[r.fam], r.d[0], r.d[1], r.d[2], r.d[3], (double)t, r.work);
  }
  fclose(f);
  return 0;
}

extern "C" int qtt_diag_fp64_probe(void* stream, int kind, int ctas, int iters, double* tflops_out) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (ctas < 1 || iters < 1 || !tflops_out) return (int)cudaErrorInvalidValue;
  double* sink = nullptr;
  QTT_CHECK_CUDA(cudaMalloc(&sink, sizeof(double)));
  cudaEvent_t e0, e1;
  QTT_CHECK_CUDA(cudaEventCreate(&e0));
  QTT_CHECK_CUDA(cudaEventCreate(&e1));
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {  // first repetition is the warm-up
    QTT_CHECK_CUDA(cudaEventRecord(e0, st));
    if (kind == 0)
      qtt_probe_dmma_kernel<<<ctas, 256, 0, st>>>(iters, sink);
    else
      qtt_probe_dfma_kernel<<<ctas, 256, 0, st>>>(iters, sink);
    QTT_CHECK_CUDA(cudaGetLastError());
    QTT_CHECK_CUDA(cudaEventRecord(e1, st));
    QTT_CHECK_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    QTT_CHECK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    if (rep > 0 && ms < best) best = ms;
  }
  // DMMA.8x8x4: 8*8*4*2 = 512 flop per warp instruction; DFMA: 2 flop per thread instruction
  const double per_cta_iter = (kind == 0) ? 8.0 * 64.0 * 512.0 : 256.0 * 64.0 * 2.0;
  *tflops_out = per_cta_iter * (double)ctas * (double)iters / ((double)best * 1e-3) * 1e-12;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return 0;
}
