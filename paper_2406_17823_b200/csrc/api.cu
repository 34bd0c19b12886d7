// The qtt_* C ABI (include/qtt.h): handles, lazy results, dispatch to the batched sweeps, and the
// CUDA-graph replay of a whole RK4 step.  No CPU fallback anywhere: every numerical step runs in the
// kernels of this library.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

#include "../../include/qtt_diag.h"
#include "engine.cuh"

// ------------------------------------------------------------------------------------------ bodies
namespace {

void body_release(Body* b);

void mpo_release(MpoData* w) {
  if (!w) return;
  if (--w->refs > 0) return;
  if (w->storage && w->ctx) w->ctx->release(w->storage, w->ctx->user);
  if (w->storage && w->ctx) --w->ctx->live;
  delete w;
}

void body_release(Body* b) {
  if (!b) return;
  if (--b->refs > 0) return;
  if (b->storage && b->ctx) b->ctx->release(b->storage, b->ctx->user);
  if (b->storage && b->ctx) --b->ctx->live;
  mpo_release(b->mpo);
  body_release(b->x);
  body_release(b->a);
  body_release(b->b);
  for (auto& t : b->terms) body_release(t.second);
  delete b;
}

Body* body_retain(Body* b) {
  ++b->refs;
  return b;
}

size_t cores_doubles(const std::vector<int>& r, int d) {
  size_t s = 0;
  for (size_t k = 0; k + 1 < r.size(); ++k) s += (size_t)r[k] * d * r[k + 1];
  return s;
}

// New dense body with slots for the capacity bonds `rcap`, 256-byte aligned slots.
Body* body_new_dense(qtt_ctx* ctx, const std::vector<int>& rcap) {
  Body* b = new Body();
  b->ctx = ctx;
  b->kind = BODY_DENSE;
  b->n = (int)rcap.size() - 1;
  b->r = rcap;
  b->storage_doubles = cores_doubles(rcap, ctx->d);
  b->storage = static_cast<double*>(ctx->alloc(std::max<size_t>(b->storage_doubles, 1) * sizeof(double), ctx->user));
  if (!b->storage) {
    delete b;
    QTT_THROW(QTT_CAPACITY, "alloc callback returned NULL");
  }
  ++ctx->live;
  b->core.resize(b->n);
  size_t off = 0;
  for (int k = 0; k < b->n; ++k) {
    b->core[k] = b->storage + off;
    off += (size_t)rcap[k] * ctx->d * rcap[k + 1];
  }
  b->tight = true;
  return b;
}

OutMps out_of_body(Body* b) {
  OutMps o;
  o.n = b->n;
  o.rcap = b->r;
  o.core = b->core;
  return o;
}
void body_set_bonds(Body* b, const std::vector<int>& r) {
  b->tight = (r == b->r);
  b->r = r;
}

View view_of_body(const Body* b) {
  View v;
  v.n = b->n;
  v.r = b->r;
  v.core.assign(b->core.begin(), b->core.end());
  return v;
}


// Dense view of any body; lazy kinds are materialised in the tmp stack (bounded by the limit).
View materialize(qtt_ctx* ctx, const Body* b) {
  if (b->kind == BODY_DENSE) return view_of_body(b);
  if (cores_doubles(b->r, ctx->d) * sizeof(double) > ctx->mat_limit)
    QTT_THROW(QTT_CAPACITY, "lazy result exceeds the materialisation limit; round it instead");
  if (b->kind == BODY_APPLIED) {
    View x = materialize(ctx, b->x);
    return qtt_expand_apply(ctx, b->mpo, x);
  }
  if (b->kind == BODY_PRODUCT) {
    View a = materialize(ctx, b->a), c = materialize(ctx, b->b);
    return qtt_kron(ctx, a, c);
  }
  // SUM: chunks of at most 5 terms
  std::vector<std::pair<double, View>> terms;
  for (auto& t : b->terms) terms.push_back({t.first, materialize(ctx, t.second)});
  while (terms.size() > 5) {
    std::vector<std::pair<double, View>> head(terms.begin(), terms.begin() + 5);
    std::vector<View> o;
    qtt_concat_batch(ctx, {head}, o);
    terms.erase(terms.begin(), terms.begin() + 5);
    terms.insert(terms.begin(), {1.0, o[0]});
  }
  std::vector<View> o;
  qtt_concat_batch(ctx, {terms}, o);
  return o[0];
}

struct ArenaScope {
  qtt_ctx* ctx;
  size_t lo, hi;
  explicit ArenaScope(qtt_ctx* c) : ctx(c), lo(c->arena.lo), hi(c->arena.hi) {}
  ~ArenaScope() {
    ctx->arena.lo = lo;
    ctx->arena.hi = hi;
  }
};

int fail(qtt_ctx* ctx, const QttError& e) {
  if (ctx) ctx->err = e.msg;
  return e.status;
}

#define QTT_API_BEGIN try {
#define QTT_API_END(ctx)                                         \
  }                                                              \
  catch (const QttError& e) { return fail((ctx), e); }           \
  catch (const std::bad_alloc&) {                                \
    if (ctx) (ctx)->err = "host out of memory";                  \
    return QTT_CAPACITY;                                         \
  }                                                              \
  return QTT_OK;

void set_device(qtt_ctx* ctx) {
  QTT_CU(cudaSetDevice(ctx->device));
  qtt_stats_bind(&ctx->stats);
}

// Jacobi non-convergence is recorded on the device (jac_status[1]).  Calls that synchronise the stream anyway read it
// back and return QTT_NUMERIC once per new hit, so a half-orthogonalised SVD of an earlier asynchronous call (eps == 0,
// graph replay) cannot go unnoticed.  Synchronises the stream.
void check_numeric(qtt_ctx* ctx) {
  int h[2] = {0, 0};
  QTT_CU(cudaMemcpyAsync(h, ctx->jac_status, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
  QTT_CU(cudaStreamSynchronize(ctx->stream));
  if (h[1] > ctx->numeric_seen) {
    ctx->numeric_seen = h[1];
    QTT_THROW(QTT_NUMERIC, "a Jacobi SVD hit its sweep limit (not converged) in this or an earlier call on this context");
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------ RK4 plans
struct Rk4Plan {
  std::vector<int> rin[2], rout[2];
  const MpoData *Dx, *Dy, *Lap;
  double Re, dt;
  int chi, chi_work, skew, sketch;
  unsigned long long sketch_seed;
  double* in_buf[2] = {nullptr, nullptr};
  double* out_buf[2] = {nullptr, nullptr};
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  size_t nodes = 0;
  size_t lo0 = 0, hi0 = 0;
};

namespace {
void plan_free(qtt_ctx* ctx, Rk4Plan* p) {
  if (p->exec) cudaGraphExecDestroy(p->exec);
  if (p->graph) cudaGraphDestroy(p->graph);
  for (int i = 0; i < 2; ++i) {
    if (p->in_buf[i]) ctx->release(p->in_buf[i], ctx->user);
    if (p->out_buf[i]) ctx->release(p->out_buf[i], ctx->user);
  }
  mpo_release(const_cast<MpoData*>(p->Dx));
  mpo_release(const_cast<MpoData*>(p->Dy));
  mpo_release(const_cast<MpoData*>(p->Lap));
  delete p;
}

View packed_view(const std::vector<int>& r, double* base) {
  View v;
  v.n = (int)r.size() - 1;
  v.r = r;
  v.core.resize(v.n);
  size_t off = 0;
  for (int k = 0; k < v.n; ++k) {
    v.core[k] = base + off;
    off += (size_t)r[k] * 4 * r[k + 1];
  }
  return v;
}
OutMps packed_out(const std::vector<int>& r, double* base) {
  OutMps o;
  o.n = (int)r.size() - 1;
  o.rcap = r;
  o.core.resize(o.n);
  size_t off = 0;
  for (int k = 0; k < o.n; ++k) {
    o.core[k] = base + off;
    off += (size_t)r[k] * 4 * r[k + 1];
  }
  return o;
}

// static output bonds of one RK4 step (eps == 0)
void rk4_out_bonds(const std::vector<int> rin[2], const MpoData* Dx, const MpoData* Dy, const MpoData* Lap, int chi,
                   int chi_work, int skew, std::vector<int> rout[2]) {
  auto applied = [&](const MpoData* W, const std::vector<int>& r) {
    std::vector<int> e(r.size());
    for (size_t k = 0; k < r.size(); ++k) e[k] = W->D[k] * r[k];
    return qtt_round_caps(e, chi);
  };
  auto summed = [&](std::vector<std::vector<int>> rs) {
    std::vector<int> e(rs[0].size(), 0);
    for (auto& r : rs)
      for (size_t k = 0; k < r.size(); ++k) e[k] += r[k];
    e.front() = e.back() = 1;
    return qtt_round_caps(e, chi);
  };
  auto rhs_b = [&](const std::vector<int> u[2], std::vector<int> f[2]) {
    for (int i = 0; i < 2; ++i) {
      std::vector<int> g0 = applied(Dx, u[i]), g1 = applied(Dy, u[i]), l = applied(Lap, u[i]);
      std::vector<int> rw, c0, c1;
      qtt_zip_caps(u[0], g0, chi, chi_work, rw, c0);
      qtt_zip_caps(u[1], g1, chi, chi_work, rw, c1);
      if (skew) {
        std::vector<int> p0, p1;
        qtt_zip_caps(u[0], u[i], chi, chi_work, rw, p0);
        qtt_zip_caps(u[i], u[1], chi, chi_work, rw, p1);
        f[i] = summed({c0, c1, applied(Dx, p0), applied(Dy, p1), l});
      } else {
        f[i] = summed({c0, c1, l});
      }
    }
  };
  std::vector<int> k1[2], k2[2], k3[2], k4[2], us[2];
  rhs_b(rin, k1);
  for (int i = 0; i < 2; ++i) us[i] = summed({rin[i], k1[i]});
  rhs_b(us, k2);
  for (int i = 0; i < 2; ++i) us[i] = summed({rin[i], k2[i]});
  rhs_b(us, k3);
  for (int i = 0; i < 2; ++i) us[i] = summed({rin[i], k3[i]});
  rhs_b(us, k4);
  for (int i = 0; i < 2; ++i) rout[i] = summed({rin[i], k1[i], k2[i], k3[i], k4[i]});
}
}  // namespace

// ------------------------------------------------------------------------------------------ context
extern "C" {

qtt_status qtt_ctx_create(qtt_ctx** out, int device, void* cuda_stream, qtt_alloc_fn alloc, qtt_release_fn release,
                          void* user, size_t workspace_bytes) {
  if (!out || !alloc || !release) return QTT_INVALID_ARG;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || count <= 0 || device < 0 || device >= count) return QTT_CUDA;
  if (cudaSetDevice(device) != cudaSuccess) return QTT_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return QTT_CUDA;
  if (prop.major < 10) return QTT_CUDA;  // kernels are sm_100a only
  qtt_ctx* ctx = new (std::nothrow) qtt_ctx();
  if (!ctx) return QTT_CAPACITY;
  ctx->device = device;
  ctx->stream = static_cast<cudaStream_t>(cuda_stream);
  ctx->alloc = alloc;
  ctx->release = release;
  ctx->user = user;
  qtt_stats_bind(&ctx->stats);
  if (workspace_bytes < ((size_t)1 << 20)) workspace_bytes = (size_t)1 << 20;
  ctx->arena.base = static_cast<char*>(alloc(workspace_bytes, user));
  if (!ctx->arena.base) {
    delete ctx;
    return QTT_CAPACITY;
  }
  ctx->arena.size = workspace_bytes & ~(size_t)255;
  try {
    // persistent constants at the bottom of the workspace
    if (ctx->arena.size >= ((size_t)256 << 20)) {
      const size_t side = (ctx->arena.size / 4) & ~(size_t)255;
      ctx->side_arena.base = ctx->arena.base + (ctx->arena.size - side);
      ctx->side_arena.size = side;
      ctx->side_arena.lo = 0;
      ctx->side_arena.hi = side;
      ctx->arena.size -= side;
      QTT_CU(cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking));
      QTT_CU(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
      QTT_CU(cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming));
    }
    ctx->arena.lo = 0;
    ctx->arena.hi = ctx->arena.size;
    ctx->ones = ctx->arena.keep(32);
    ctx->jac_status = reinterpret_cast<int*>(ctx->arena.keep(32));
    QTT_CU(qtt_launch_fill(ctx->ones, 32, 1.0, ctx->stream));
    QTT_CU(cudaMemsetAsync(ctx->jac_status, 0, 32 * sizeof(double), ctx->stream));
  } catch (const QttError& e) {
    if (ctx->side) cudaStreamDestroy(ctx->side);
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    release(ctx->arena.base, user);
    qtt_stats_destroy(&ctx->stats);
    delete ctx;
    return e.status;
  }
  *out = ctx;
  return QTT_OK;
}

void qtt_ctx_destroy(qtt_ctx* ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  for (Rk4Plan* p : ctx->plans) plan_free(ctx, p);
  if (ctx->side) {
    cudaStreamSynchronize(ctx->side);
    cudaStreamDestroy(ctx->side);
  }
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
  if (ctx->arena.base) ctx->release(ctx->arena.base, ctx->user);
  qtt_stats_destroy(&ctx->stats);
  delete ctx;
}

const char* qtt_last_error(const qtt_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

qtt_status qtt_ctx_set_chi_work(qtt_ctx* ctx, int chi_work) {
  if (!ctx || chi_work < 0) return QTT_INVALID_ARG;
  ctx->chi_work = chi_work;
  return QTT_OK;
}
qtt_status qtt_ctx_set_phys_dim(qtt_ctx* ctx, int d) {
  if (!ctx || (d != 4 && d != 8)) return QTT_INVALID_ARG;
  if (d != ctx->d && ctx->live != 0) {
    ctx->err = "qtt_ctx_set_phys_dim: free every MPS / MPO handle of the context before switching the encoding";
    return QTT_INVALID_ARG;
  }
  ctx->d = d;
  return QTT_OK;
}
int qtt_ctx_phys_dim(const qtt_ctx* ctx) { return ctx ? ctx->d : 0; }
qtt_status qtt_ctx_set_materialize_limit(qtt_ctx* ctx, size_t bytes) {
  if (!ctx) return QTT_INVALID_ARG;
  ctx->mat_limit = bytes;
  return QTT_OK;
}
qtt_status qtt_ctx_set_convection(qtt_ctx* ctx, int skew_symmetric) {
  if (!ctx || (skew_symmetric != 0 && skew_symmetric != 1)) return QTT_INVALID_ARG;
  ctx->skew = skew_symmetric;
  return QTT_OK;
}
qtt_status qtt_ctx_set_product_compression(qtt_ctx* ctx, int mode, unsigned long long seed) {
  if (!ctx || (mode != 0 && mode != 1)) return QTT_INVALID_ARG;
  ctx->sketch = mode;
  ctx->sketch_seed = seed;
  return QTT_OK;
}
qtt_status qtt_ctx_set_graphs(qtt_ctx* ctx, int enabled) {
  if (!ctx) return QTT_INVALID_ARG;
  ctx->graphs = enabled ? 1 : 0;
  return QTT_OK;
}
qtt_status qtt_ctx_jacobi_stats(qtt_ctx* ctx, int* max_sweeps, int* limit_hits) {
  if (!ctx) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  int h[2] = {0, 0};
  QTT_CU(cudaMemcpyAsync(h, ctx->jac_status, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
  QTT_CU(cudaMemsetAsync(ctx->jac_status, 0, sizeof(h), ctx->stream));
  QTT_CU(cudaStreamSynchronize(ctx->stream));
  if (max_sweeps) *max_sweeps = h[0];
  if (limit_hits) *limit_hits = h[1];
  ctx->numeric_seen = 0;
  if (h[1] > 0) QTT_THROW(QTT_NUMERIC, "Jacobi sweep limit hit");
  QTT_API_END(ctx)
}
qtt_status qtt_ctx_profile(qtt_ctx* ctx, int enabled) {
  if (!ctx) return QTT_INVALID_ARG;
  ctx->profiling = enabled ? 1 : 0;
  ctx->stats.prof_on = enabled != 0;
  return QTT_OK;
}
qtt_status qtt_ctx_profile_report(qtt_ctx* ctx, double* ms_host, double* work_host, long long* launches_host) {
  if (!ctx || !ms_host || !work_host || !launches_host) return QTT_INVALID_ARG;
  static_assert(QK_COUNT == QTT_PROF_FAMILIES, "family count");
  QTT_API_BEGIN
  set_device(ctx);
  QTT_CU(qtt_prof_collect(&ctx->stats, ms_host, work_host, launches_host));
  QTT_API_END(ctx)
}
long long qtt_ctx_launch_count(const qtt_ctx* ctx) { return ctx ? ctx->stats.launches + ctx->graph_launches : 0; }

// ------------------------------------------------------------------------------------------ MPS / MPO
qtt_status qtt_mps_from_cores(qtt_ctx* ctx, int n, const int* bonds, const double* const* cores_host, qtt_mps** out) {
  if (!ctx || !bonds || !cores_host || !out || n < 1) return QTT_INVALID_ARG;
  if (bonds[0] != 1 || bonds[n] != 1) return QTT_SHAPE_MISMATCH;
  QTT_API_BEGIN
  set_device(ctx);
  std::vector<int> r(bonds, bonds + n + 1);
  for (int v : r)
    if (v < 1) QTT_THROW(QTT_SHAPE_MISMATCH, "bond dimensions must be >= 1");
  Body* b = body_new_dense(ctx, r);
  for (int k = 0; k < n; ++k)
    QTT_CU(cudaMemcpyAsync(b->core[k], cores_host[k], sizeof(double) * (size_t)r[k] * ctx->d * r[k + 1],
                           cudaMemcpyHostToDevice, ctx->stream));
  QTT_CU(cudaStreamSynchronize(ctx->stream));  // host arrays may go away
  *out = new qtt_mps{ctx, b};
  QTT_API_END(ctx)
}

qtt_status qtt_mpo_create(qtt_ctx* ctx, int n, const int* bonds, const double* const* cores_host, qtt_mpo** out) {
  if (!ctx || !bonds || !cores_host || !out || n < 1) return QTT_INVALID_ARG;
  if (bonds[0] != 1 || bonds[n] != 1) return QTT_SHAPE_MISMATCH;
  QTT_API_BEGIN
  set_device(ctx);
  MpoData* w = new MpoData();
  w->ctx = ctx;
  w->n = n;
  w->D.assign(bonds, bonds + n + 1);
  size_t tot = 0;
  const size_t dd = (size_t)ctx->d * ctx->d;
  for (int k = 0; k < n; ++k) tot += (((size_t)w->D[k] * dd * w->D[k + 1]) + 31) & ~(size_t)31;
  w->storage = static_cast<double*>(ctx->alloc(tot * sizeof(double), ctx->user));
  if (!w->storage) {
    delete w;
    QTT_THROW(QTT_CAPACITY, "alloc callback returned NULL");
  }
  ++ctx->live;
  size_t off = 0;
  w->core.resize(n);
  for (int k = 0; k < n; ++k) {
    size_t sz = (size_t)w->D[k] * dd * w->D[k + 1];
    w->core[k] = w->storage + off;
    QTT_CU(cudaMemcpyAsync(w->storage + off, cores_host[k], sz * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    off += (sz + 31) & ~(size_t)31;
  }
  QTT_CU(cudaStreamSynchronize(ctx->stream));
  *out = new qtt_mpo{w};
  QTT_API_END(ctx)
}

void qtt_mpo_free(qtt_mpo* w) {
  if (!w) return;
  mpo_release(w->data);
  delete w;
}

void qtt_mps_free(qtt_mps* x) {
  if (!x) return;
  body_release(x->body);
  delete x;
}

int qtt_mps_num_sites(const qtt_mps* x) { return x ? x->body->n : 0; }

qtt_status qtt_mps_bonds(const qtt_mps* x, int* bonds_out) {
  if (!x || !bonds_out) return QTT_INVALID_ARG;
  for (int k = 0; k <= x->body->n; ++k) bonds_out[k] = x->body->r[k];
  return QTT_OK;
}

qtt_status qtt_mps_clone(qtt_ctx* ctx, const qtt_mps* x, qtt_mps** out) {
  if (!ctx || !x || !out) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  View v = materialize(ctx, x->body);
  Body* b = body_new_dense(ctx, v.r);
  for (int k = 0; k < v.n; ++k)
    QTT_CU(cudaMemcpyAsync(b->core[k], v.core[k], sizeof(double) * (size_t)v.r[k] * ctx->d * v.r[k + 1],
                           cudaMemcpyDeviceToDevice, ctx->stream));
  *out = new qtt_mps{ctx, b};
  QTT_API_END(ctx)
}

qtt_status qtt_mps_get_core(qtt_ctx* ctx, const qtt_mps* x, int k, double* host_out) {
  if (!ctx || !x || !host_out || k < 0 || k >= x->body->n) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  View v = materialize(ctx, x->body);
  QTT_CU(cudaMemcpyAsync(host_out, v.core[k], sizeof(double) * (size_t)v.r[k] * ctx->d * v.r[k + 1], cudaMemcpyDeviceToHost,
                         ctx->stream));
  check_numeric(ctx);
  QTT_API_END(ctx)
}

qtt_status qtt_mps_core_ptr(qtt_ctx* ctx, const qtt_mps* x, int k, const double** core_dev_out) {
  if (!ctx || !x || !core_dev_out || k < 0 || k >= x->body->n) return QTT_INVALID_ARG;
  if (x->body->kind != BODY_DENSE) {
    ctx->err = "qtt_mps_core_ptr needs explicit cores: round the lazy handle first (or use qtt_mps_get_core)";
    return QTT_INVALID_ARG;
  }
  *core_dev_out = x->body->core[k];
  return QTT_OK;
}

qtt_status qtt_mps_from_dense(qtt_ctx* ctx, const double* dense_dev, int n_bits, int chi_max, double eps,
                              qtt_mps** out) {
  if (!ctx || !dense_dev || !out || n_bits < 1 || n_bits > (ctx->d == 8 ? 9 : 13) || chi_max < 1 || eps < 0.0)
    return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  const int n = n_bits;
  std::vector<int> full(n + 1, 1);
  for (int k = 1; k < n; ++k) {
    int l = std::min(k, n - k);
    full[k] = l >= (ctx->d == 8 ? 10 : 15) ? (1 << 30) : (1 << ((ctx->d == 8 ? 3 : 2) * l));
  }
  std::vector<int> caps(n + 1, 1);
  for (int k = n - 1; k >= 1; --k)
    caps[k] = (int)std::min<long long>(std::min<long long>(chi_max, full[k]), (long long)ctx->d * caps[k + 1]);
  Body* b = body_new_dense(ctx, caps);
  try {
    OutMps o = out_of_body(b);
    qtt_from_dense(ctx, dense_dev, n, chi_max, eps, o);
    body_set_bonds(b, o.r);
  } catch (...) {
    body_release(b);
    throw;
  }
  *out = new qtt_mps{ctx, b};
  QTT_API_END(ctx)
}

qtt_status qtt_to_dense(qtt_ctx* ctx, const qtt_mps* x, double* dense_dev_out) {
  if (!ctx || !x || !dense_dev_out) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  View v = materialize(ctx, x->body);
  qtt_to_dense_view(ctx, v, dense_dev_out);
  QTT_API_END(ctx)
}

// ------------------------------------------------------------------------------------------ lazy algebra
qtt_status qtt_apply_mpo(qtt_ctx* ctx, const qtt_mpo* w, const qtt_mps* x, qtt_mps** y) {
  if (!ctx || !w || !x || !y) return QTT_INVALID_ARG;
  if (w->data->n != x->body->n) {
    ctx->err = "MPO and MPS differ in length";
    return QTT_SHAPE_MISMATCH;
  }
  QTT_API_BEGIN
  Body* b = new Body();
  b->ctx = ctx;
  b->kind = BODY_APPLIED;
  b->n = x->body->n;
  b->r.resize(b->n + 1);
  for (int k = 0; k <= b->n; ++k) b->r[k] = w->data->D[k] * x->body->r[k];
  b->mpo = w->data;
  ++w->data->refs;
  b->x = body_retain(x->body);
  *y = new qtt_mps{ctx, b};
  QTT_API_END(ctx)
}

qtt_status qtt_hadamard(qtt_ctx* ctx, const qtt_mps* a, const qtt_mps* b, qtt_mps** c) {
  if (!ctx || !a || !b || !c) return QTT_INVALID_ARG;
  if (a->body->n != b->body->n) {
    ctx->err = "product operands differ in length";
    return QTT_SHAPE_MISMATCH;
  }
  QTT_API_BEGIN
  Body* p = new Body();
  p->ctx = ctx;
  p->kind = BODY_PRODUCT;
  p->n = a->body->n;
  p->r.resize(p->n + 1);
  for (int k = 0; k <= p->n; ++k) {
    long long v = (long long)a->body->r[k] * b->body->r[k];
    if (v > (1ll << 30)) {
      delete p;
      QTT_THROW(QTT_CAPACITY, "product bond overflows");
    }
    p->r[k] = (int)v;
  }
  p->a = body_retain(a->body);
  p->b = body_retain(b->body);
  *c = new qtt_mps{ctx, p};
  QTT_API_END(ctx)
}

qtt_status qtt_axpy(qtt_ctx* ctx, double alpha, const qtt_mps* x, qtt_mps* y) {
  if (!ctx || !x || !y) return QTT_INVALID_ARG;
  if (x->body->n != y->body->n) {
    ctx->err = "summands differ in length";
    return QTT_SHAPE_MISMATCH;
  }
  if (x->body->n < 2) {
    ctx->err = "sums need at least two sites";
    return QTT_INVALID_ARG;
  }
  QTT_API_BEGIN
  Body* s = new Body();
  s->ctx = ctx;
  s->kind = BODY_SUM;
  s->n = y->body->n;
  // oracle O5 / axpy: alpha*X first, then Y; nested sums are flattened (a sum with unit weight)
  s->terms.push_back({alpha, body_retain(x->body)});
  Body* old = y->body;
  if (old->kind == BODY_SUM) {
    for (auto& t : old->terms) s->terms.push_back({t.first, body_retain(t.second)});
  } else {
    s->terms.push_back({1.0, body_retain(old)});
  }
  s->r.assign(s->n + 1, 0);
  for (auto& t : s->terms)
    for (int k = 0; k <= s->n; ++k) s->r[k] += t.second->r[k];
  s->r[0] = s->r[s->n] = 1;
  body_release(old);
  y->body = s;
  QTT_API_END(ctx)
}

// ------------------------------------------------------------------------------------------ rounding
static qtt_status round_batch_impl(qtt_ctx* ctx, int batch, qtt_mps* const* xs, int chi_max, double eps,
                                   int chi_work) {
  if (!ctx || !xs || batch < 1 || chi_max < 1 || eps < 0.0 || chi_work < 0) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  std::vector<int> prod_idx, dense_idx;
  for (int i = 0; i < batch; ++i) {
    if (!xs[i]) QTT_THROW(QTT_INVALID_ARG, "null operand");
    (xs[i]->body->kind == BODY_PRODUCT ? prod_idx : dense_idx).push_back(i);
  }
  std::vector<Body*> fresh(batch, nullptr);
  try {
    if (!dense_idx.empty()) {
      std::vector<View> in;
      std::vector<OutMps> out;
      for (int i : dense_idx) {
        in.push_back(materialize(ctx, xs[i]->body));
        fresh[i] = body_new_dense(ctx, qtt_round_caps(in.back().r, chi_max, ctx->d));
        out.push_back(out_of_body(fresh[i]));
      }
      qtt_round_dense_batch(ctx, in, chi_max, eps, out);
      for (size_t j = 0; j < dense_idx.size(); ++j) body_set_bonds(fresh[dense_idx[j]], out[j].r);
    }
    if (!prod_idx.empty()) {
      const int cw = chi_work > 0 ? chi_work : (ctx->chi_work > 0 ? ctx->chi_work : 2 * chi_max);
      std::vector<View> A, B;
      std::vector<OutMps> out;
      for (int i : prod_idx) {
        A.push_back(materialize(ctx, xs[i]->body->a));
        B.push_back(materialize(ctx, xs[i]->body->b));
        std::vector<int> rw, ro;
        qtt_zip_caps(A.back().r, B.back().r, chi_max, cw, rw, ro, ctx->d);
        fresh[i] = body_new_dense(ctx, ro);
        out.push_back(out_of_body(fresh[i]));
      }
      qtt_round_product_batch(ctx, A, B, chi_max, eps, cw, out);
      for (size_t j = 0; j < prod_idx.size(); ++j) body_set_bonds(fresh[prod_idx[j]], out[j].r);
    }
  } catch (...) {
    for (Body* b : fresh) body_release(b);
    throw;
  }
  for (int i = 0; i < batch; ++i) {
    body_release(xs[i]->body);
    xs[i]->body = fresh[i];
  }
  if (eps > 0.0) check_numeric(ctx);  // this path synchronised once per bond already
  QTT_API_END(ctx)
}

qtt_status qtt_round_batch(qtt_ctx* ctx, int batch, qtt_mps* const* xs, int chi_max, double eps) {
  return round_batch_impl(ctx, batch, xs, chi_max, eps, 0);
}

qtt_status qtt_round(qtt_ctx* ctx, qtt_mps* x, int chi_max, double eps) {
  qtt_mps* xs[1] = {x};
  return round_batch_impl(ctx, 1, xs, chi_max, eps, 0);
}

qtt_status qtt_round_ex(qtt_ctx* ctx, qtt_mps* x, int chi_max, double eps, int chi_work) {
  qtt_mps* xs[1] = {x};
  return round_batch_impl(ctx, 1, xs, chi_max, eps, chi_work);
}

// ------------------------------------------------------------------------------------------ RK4
qtt_status qtt_rk4_step3(qtt_ctx* ctx, qtt_mps* const u[3], const qtt_mpo* const D[3], const qtt_mpo* Lap, double Re, double dt,
                         int chi_max, double eps) {
  if (!ctx || !u || !D || !Lap || chi_max < 1 || eps < 0.0 || !(Re > 0.0)) return QTT_INVALID_ARG;
  for (int i = 0; i < 3; ++i)
    if (!u[i] || !D[i]) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  if (ctx->d != 8) QTT_THROW(QTT_INVALID_ARG, "qtt_rk4_step3 needs the 3D encoding (qtt_ctx_set_phys_dim(ctx, 8))");
  if (ctx->sketch) QTT_THROW(QTT_INVALID_ARG, "the sketched product compression is built for physical dimension 4 only");
  const int n = u[0]->body->n;
  for (int i = 0; i < 3; ++i)
    if (u[i]->body->n != n || D[i]->data->n != n) QTT_THROW(QTT_SHAPE_MISMATCH, "rk4_step3 operands differ in length");
  if (Lap->data->n != n || n < 2) QTT_THROW(QTT_SHAPE_MISMATCH, "rk4_step3 operands differ in length (or fewer than two sites)");
  const int cw = ctx->chi_work > 0 ? ctx->chi_work : 2 * chi_max;
  ArenaScope scope(ctx);
  View uv[3] = {materialize(ctx, u[0]->body), materialize(ctx, u[1]->body), materialize(ctx, u[2]->body)};
  const MpoData* Dj[3] = {D[0]->data, D[1]->data, D[2]->data};
  // capacity bonds of the result: min(chi, 8^k, 8^(n-k)) (the sweep fills in the actual ones)
  std::vector<int> caps(n + 1, 1);
  for (int k = 1; k < n; ++k) {
    const int l = std::min(k, n - k);
    caps[k] = (int)std::min<long long>(chi_max, l >= 10 ? (1ll << 30) : (1ll << (3 * l)));
  }
  Body* fresh[3] = {nullptr, nullptr, nullptr};
  try {
    for (int i = 0; i < 3; ++i) fresh[i] = body_new_dense(ctx, caps);
    OutMps out[3] = {out_of_body(fresh[0]), out_of_body(fresh[1]), out_of_body(fresh[2])};
    qtt_rk4_eager3(ctx, uv, Dj, Lap->data, Re, dt, chi_max, eps, cw, out);
    for (int i = 0; i < 3; ++i) body_set_bonds(fresh[i], out[i].r);
  } catch (...) {
    for (int i = 0; i < 3; ++i) body_release(fresh[i]);
    throw;
  }
  for (int i = 0; i < 3; ++i) {
    body_release(u[i]->body);
    u[i]->body = fresh[i];
  }
  if (eps > 0.0) check_numeric(ctx);
  QTT_API_END(ctx)
}

qtt_status qtt_rk4_step(qtt_ctx* ctx, qtt_mps* const u[2], const qtt_mpo* Dx, const qtt_mpo* Dy, const qtt_mpo* Lap,
                        double Re, double dt, int chi_max, double eps) {
  if (!ctx || !u || !u[0] || !u[1] || !Dx || !Dy || !Lap || chi_max < 1 || eps < 0.0 || !(Re > 0.0))
    return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  if (ctx->d != 4) QTT_THROW(QTT_INVALID_ARG, "qtt_rk4_step is built for the 2D encoding (physical dimension 4)");
  const int n = u[0]->body->n;
  if (u[1]->body->n != n || Dx->data->n != n || Dy->data->n != n || Lap->data->n != n || n < 2)
    QTT_THROW(QTT_SHAPE_MISMATCH, "rk4_step operands differ in length (or fewer than two sites)");
  const int cw = ctx->chi_work > 0 ? ctx->chi_work : 2 * chi_max;
  ArenaScope scope(ctx);

  if (eps > 0.0 || !ctx->graphs || ctx->profiling) {
    // eager path (eps > 0 synchronises once per bond)
    View uv[2] = {materialize(ctx, u[0]->body), materialize(ctx, u[1]->body)};
    std::vector<int> rin[2] = {uv[0].r, uv[1].r}, rout[2];
    rk4_out_bonds(rin, Dx->data, Dy->data, Lap->data, chi_max, cw, ctx->skew, rout);
    Body* fresh[2] = {body_new_dense(ctx, rout[0]), nullptr};
    try {
      fresh[1] = body_new_dense(ctx, rout[1]);
      OutMps out[2] = {out_of_body(fresh[0]), out_of_body(fresh[1])};
      qtt_rk4_eager(ctx, uv, Dx->data, Dy->data, Lap->data, Re, dt, chi_max, eps, cw, ctx->skew, out);
      body_set_bonds(fresh[0], out[0].r);
      body_set_bonds(fresh[1], out[1].r);
    } catch (...) {
      body_release(fresh[0]);
      body_release(fresh[1]);
      throw;
    }
    for (int i = 0; i < 2; ++i) {
      body_release(u[i]->body);
      u[i]->body = fresh[i];
    }
    if (eps > 0.0) check_numeric(ctx);
    return QTT_OK;
  }

  // ---- graph path: one captured graph per shape signature, fixed staging buffers
  View uv[2] = {materialize(ctx, u[0]->body), materialize(ctx, u[1]->body)};
  Rk4Plan* plan = nullptr;
  for (Rk4Plan* p : ctx->plans)
    if (p->rin[0] == uv[0].r && p->rin[1] == uv[1].r && p->Dx == Dx->data && p->Dy == Dy->data &&
        p->Lap == Lap->data && p->Re == Re && p->dt == dt && p->chi == chi_max && p->chi_work == cw && p->skew == ctx->skew && p->sketch == ctx->sketch && p->sketch_seed == ctx->sketch_seed &&
        p->lo0 == ctx->arena.lo && p->hi0 == ctx->arena.hi)
      plan = p;
  if (!plan) {
    if (ctx->plans.size() >= 8) {
      QTT_CU(cudaStreamSynchronize(ctx->stream));
      plan_free(ctx, ctx->plans.front());
      ctx->plans.erase(ctx->plans.begin());
    }
    plan = new Rk4Plan();
    plan->Dx = Dx->data; plan->Dy = Dy->data; plan->Lap = Lap->data;
    ++Dx->data->refs; ++Dy->data->refs; ++Lap->data->refs;
    plan->Re = Re; plan->dt = dt; plan->chi = chi_max; plan->chi_work = cw; plan->skew = ctx->skew;
    plan->sketch = ctx->sketch; plan->sketch_seed = ctx->sketch_seed;
    plan->lo0 = ctx->arena.lo; plan->hi0 = ctx->arena.hi;
    for (int i = 0; i < 2; ++i) plan->rin[i] = uv[i].r;
    rk4_out_bonds(plan->rin, Dx->data, Dy->data, Lap->data, chi_max, cw, ctx->skew, plan->rout);
    try {
      for (int i = 0; i < 2; ++i) {
        plan->in_buf[i] = static_cast<double*>(ctx->alloc(cores_doubles(plan->rin[i], 4) * sizeof(double), ctx->user));
        plan->out_buf[i] = static_cast<double*>(ctx->alloc(cores_doubles(plan->rout[i], 4) * sizeof(double), ctx->user));
        if (!plan->in_buf[i] || !plan->out_buf[i]) QTT_THROW(QTT_CAPACITY, "alloc callback returned NULL");
      }
      View pin[2] = {packed_view(plan->rin[0], plan->in_buf[0]), packed_view(plan->rin[1], plan->in_buf[1])};
      OutMps pout[2] = {packed_out(plan->rout[0], plan->out_buf[0]), packed_out(plan->rout[1], plan->out_buf[1])};
      const long long launches_before = ctx->stats.launches;  // captured launches run at replay, counted there
      QTT_CU(cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeRelaxed));
      try {
        qtt_rk4_eager(ctx, pin, Dx->data, Dy->data, Lap->data, Re, dt, chi_max, 0.0, cw, ctx->skew, pout);
      } catch (...) {
        cudaGraph_t junk = nullptr;
        ctx->stats.launches = launches_before;
        cudaStreamEndCapture(ctx->stream, &junk);
        if (junk) cudaGraphDestroy(junk);
        throw;
      }
      QTT_CU(cudaStreamEndCapture(ctx->stream, &plan->graph));
      plan->nodes = (size_t)(ctx->stats.launches - launches_before);  // kernel nodes only
      ctx->stats.launches = launches_before;
      QTT_CU(cudaGraphInstantiate(&plan->exec, plan->graph, 0));
    } catch (...) {
      plan_free(ctx, plan);
      throw;
    }
    ctx->plans.push_back(plan);
  }
  // stage in, replay, stage out
  for (int i = 0; i < 2; ++i) {
    size_t off = 0;
    if (u[i]->body->kind == BODY_DENSE && u[i]->body->tight) {
      QTT_CU(cudaMemcpyAsync(plan->in_buf[i], u[i]->body->storage, cores_doubles(uv[i].r, 4) * sizeof(double),
                             cudaMemcpyDeviceToDevice, ctx->stream));
    } else {
      for (int k = 0; k < n; ++k) {
        size_t sz = (size_t)uv[i].r[k] * 4 * uv[i].r[k + 1];
        QTT_CU(cudaMemcpyAsync(plan->in_buf[i] + off, uv[i].core[k], sz * sizeof(double), cudaMemcpyDeviceToDevice,
                               ctx->stream));
        off += sz;
      }
    }
  }
  QTT_CU(cudaGraphLaunch(plan->exec, ctx->stream));
  ctx->graph_launches += (long long)plan->nodes;
  for (int i = 0; i < 2; ++i) {
    Body* b = u[i]->body;
    if (!(b->kind == BODY_DENSE && b->tight && b->refs == 1 && b->r == plan->rout[i])) {
      Body* nb = body_new_dense(ctx, plan->rout[i]);
      body_release(b);
      u[i]->body = b = nb;
    }
    QTT_CU(cudaMemcpyAsync(b->storage, plan->out_buf[i], cores_doubles(plan->rout[i], 4) * sizeof(double),
                           cudaMemcpyDeviceToDevice, ctx->stream));
  }
  QTT_API_END(ctx)
}

// ------------------------------------------------------------------------------------------ inspection
qtt_status qtt_mps_dot(qtt_ctx* ctx, const qtt_mps* a, const qtt_mps* b, double* out_host) {
  if (!ctx || !a || !b || !out_host) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  View va = materialize(ctx, a->body), vb = materialize(ctx, b->body);
  double* d = qtt_dot_view(ctx, va, vb);
  QTT_CU(cudaMemcpyAsync(out_host, d, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  check_numeric(ctx);
  QTT_API_END(ctx)
}

qtt_status qtt_mps_schmidt(qtt_ctx* ctx, const qtt_mps* x, double* sigma_host, int cap, int* counts) {
  if (!ctx || !x || !sigma_host || !counts || cap < 1) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  View v = materialize(ctx, x->body);
  const int n = v.n;
  for (int k = 0; k <= n; ++k) counts[k] = 0;
  if (n < 2) return QTT_OK;
  const int big = 1 << 30;
  std::vector<int> caps = qtt_round_caps(v.r, big, ctx->d);
  OutMps o;
  o.n = n;
  o.rcap = caps;
  o.core.resize(n);
  for (int k = 0; k < n; ++k) o.core[k] = ctx->arena.keep((size_t)caps[k] * ctx->d * caps[k + 1]);
  std::vector<OutMps> outs{o};
  SigmaCapture sc;
  qtt_round_dense_batch(ctx, {v}, big, 0.0, outs, &sc);
  for (int k = 1; k < n; ++k) {
    int c = std::min(sc.count[0][k], cap);
    counts[k] = c;
    QTT_CU(cudaMemcpyAsync(sigma_host + (size_t)k * cap, sc.sigma[0][k], sizeof(double) * c, cudaMemcpyDeviceToHost,
                           ctx->stream));
  }
  check_numeric(ctx);
  QTT_API_END(ctx)
}

qtt_status qtt_mps_norm(qtt_ctx* ctx, const qtt_mps* x, double* out_host) {
  if (!ctx || !x || !out_host) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  ArenaScope scope(ctx);
  View v = materialize(ctx, x->body);
  const int n = v.n;
  if (n < 2) {
    double h[8] = {0, 0, 0, 0, 0, 0, 0, 0}, s2 = 0.0;
    QTT_CU(cudaMemcpyAsync(h, v.core[0], sizeof(double) * ctx->d, cudaMemcpyDeviceToHost, ctx->stream));
    QTT_CU(cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < ctx->d; ++i) s2 += h[i] * h[i];
    *out_host = std::sqrt(s2);
    return QTT_OK;
  }
  // the Schmidt values of the last bond carry the whole norm
  const int big = 1 << 30;
  std::vector<int> caps = qtt_round_caps(v.r, big, ctx->d);
  OutMps o;
  o.n = n;
  o.rcap = caps;
  o.core.resize(n);
  for (int k = 0; k < n; ++k) o.core[k] = ctx->arena.keep((size_t)caps[k] * ctx->d * caps[k + 1]);
  std::vector<OutMps> outs{o};
  SigmaCapture sc;
  qtt_round_dense_batch(ctx, {v}, big, 0.0, outs, &sc);
  const int c = sc.count[0][n - 1];
  std::vector<double> s(c);
  QTT_CU(cudaMemcpyAsync(s.data(), sc.sigma[0][n - 1], sizeof(double) * c, cudaMemcpyDeviceToHost, ctx->stream));
  check_numeric(ctx);
  double t = 0.0;
  for (int i = c - 1; i >= 0; --i) t += s[i] * s[i];
  *out_host = std::sqrt(t);
  QTT_API_END(ctx)
}

// PAPER.md:160 Eq. 12 and PAPER.md:238-244 Eq. 16-17: compositions of the calls above
qtt_status qtt_mps_fidelity(qtt_ctx* ctx, const qtt_mps* a, const qtt_mps* b, double* out_host) {
  if (!ctx || !a || !b || !out_host) return QTT_INVALID_ARG;
  double ab = 0.0, na = 0.0, nb = 0.0;
  qtt_status st = qtt_mps_dot(ctx, a, b, &ab);
  if (st == QTT_OK) st = qtt_mps_norm(ctx, a, &na);
  if (st == QTT_OK) st = qtt_mps_norm(ctx, b, &nb);
  if (st != QTT_OK) return st;
  const double d = na * na * nb * nb;
  *out_host = d > 0.0 ? ab * ab / d : 0.0;
  return QTT_OK;
}

qtt_status qtt_tke_spectrum(qtt_ctx* ctx, const qtt_mps* u1, const qtt_mps* u2, const qtt_mps* mean1, const qtt_mps* mean2,
                            int nbins, double* E_host) {
  if (!ctx || !u1 || !u2 || !E_host || nbins < 1) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  if (ctx->d != 4) QTT_THROW(QTT_INVALID_ARG, "qtt_tke_spectrum is built for the 2D encoding (physical dimension 4)");
  ArenaScope scope(ctx);
  const int n = u1->body->n;
  if (u2->body->n != n || (mean1 && mean1->body->n != n) || (mean2 && mean2->body->n != n))
    QTT_THROW(QTT_SHAPE_MISMATCH, "velocity components differ in length");
  if (n < 1 || n > 12) QTT_THROW(QTT_CAPACITY, "TKE spectrum: grids up to 2^12 x 2^12");
  const i64 N = 1ll << n;
  const int max_shell = (int)std::floor(std::sqrt(2.0) * (double)(N / 2) + 0.5);
  if (nbins < max_shell + 1) QTT_THROW(QTT_INVALID_ARG, "nbins must be at least floor(N / sqrt(2) + 1/2) + 1");
  double* spec[2];
  const qtt_mps* us[2] = {u1, u2};
  const qtt_mps* ms[2] = {mean1, mean2};
  for (int i = 0; i < 2; ++i) {
    spec[i] = ctx->arena.keep((size_t)2 * N * N);
    const size_t mark = ctx->arena.hi;
    View v = materialize(ctx, us[i]->body);
    if (ms[i]) {  // u' = u - u_mean (Eq. 14) as an exact direct sum
      if (n < 2) QTT_THROW(QTT_INVALID_ARG, "a mean field needs at least two sites");
      View m = materialize(ctx, ms[i]->body);
      std::vector<View> o;
      qtt_concat_batch(ctx, {{{1.0, v}, {-1.0, m}}}, o);
      v = o[0];
    }
    double* dense = ctx->arena.tmp((size_t)N * N);
    qtt_to_dense_view(ctx, v, dense);
    double* tmp = ctx->arena.tmp((size_t)2 * N * N);
    QTT_CU(qtt_launch_fft2_real(dense, spec[i], tmp, n, ctx->stream));
    ctx->arena.hi = mark;
  }
  double* partial = ctx->arena.tmp((size_t)N * nbins);
  double* E = ctx->arena.tmp((size_t)nbins);
  QTT_CU(qtt_launch_tke_shells(spec[0], spec[1], n, nbins, partial, E, ctx->stream));
  QTT_CU(cudaMemcpyAsync(E_host, E, sizeof(double) * nbins, cudaMemcpyDeviceToHost, ctx->stream));
  check_numeric(ctx);
  QTT_API_END(ctx)
}

qtt_status qtt_mps_chi_eps(qtt_ctx* ctx, const qtt_mps* x, double eps, int* chi_host, int* chi_max_host) {
  if (!ctx || !x || !chi_host || !(eps >= 0.0)) return QTT_INVALID_ARG;
  const int n = qtt_mps_num_sites(x);
  std::vector<int> r(n + 1), counts(n + 1, 0);
  qtt_status st = qtt_mps_bonds(x, r.data());
  if (st != QTT_OK) return st;
  int cap = 1;
  for (int k = 0; k <= n; ++k) cap = std::max(cap, r[k]);
  cap *= ctx->d;
  std::vector<double> sig((size_t)(n + 1) * cap, 0.0);
  st = qtt_mps_schmidt(ctx, x, sig.data(), cap, counts.data());
  if (st != QTT_OK) return st;
  int worst = 1;
  for (int k = 0; k <= n; ++k) chi_host[k] = 1;
  for (int k = 1; k < n; ++k) {
    const double* s = sig.data() + (size_t)k * cap;
    double tot = 0.0;
    for (int i = counts[k] - 1; i >= 0; --i) tot += s[i] * s[i];
    // smallest chi with sqrt(sum_{i >= chi} s_i^2) <= eps * ||x||   (||x||^2 = sum of all s_i^2 at any bond)
    double tail = 0.0;
    int chi = counts[k];
    for (int cand = counts[k]; cand >= 1; --cand) {
      if (std::sqrt(tail) <= eps * std::sqrt(tot)) chi = cand; else break;
      tail += s[cand - 1] * s[cand - 1];
    }
    chi_host[k] = std::max(1, chi);
    worst = std::max(worst, chi_host[k]);
  }
  if (chi_max_host) *chi_max_host = worst;
  return QTT_OK;
}

// ------------------------------------------------------------------------------------------ variational stage
qtt_status qtt_variational_cost(qtt_ctx* ctx, const qtt_mps* const v[2], const qtt_mps* const a[2], const qtt_mps* const B[2],
                                const qtt_mpo* D1, const qtt_mpo* D2, double h, double mu, double* theta_host) {
  if (!ctx || !v || !a || !B || !D1 || !D2 || !theta_host || !(h > 0.0) || mu < 0.0) return QTT_INVALID_ARG;
  for (int i = 0; i < 2; ++i)
    if (!v[i] || !a[i] || !B[i]) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  if (ctx->d != 4) QTT_THROW(QTT_INVALID_ARG, "qtt_variational_cost is built for the 2D encoding (physical dimension 4)");
  ArenaScope scope(ctx);
  View vv[2], va[2], vb[2];
  for (int i = 0; i < 2; ++i) {
    vv[i] = materialize(ctx, v[i]->body);
    va[i] = materialize(ctx, a[i]->body);
    vb[i] = materialize(ctx, B[i]->body);
    if (vv[i].n != D1->data->n || va[i].n != vv[i].n || vb[i].n != vv[i].n || D2->data->n != vv[i].n)
      QTT_THROW(QTT_SHAPE_MISMATCH, "operands differ in length");
  }
  *theta_host = qtt_variational_cost_impl(ctx, vv, va, vb, D1->data, D2->data, h, mu);
  QTT_API_END(ctx)
}

qtt_status qtt_variational_stage(qtt_ctx* ctx, qtt_mps* const v[2], const qtt_mps* const a[2], const qtt_mps* const B[2],
                                 const qtt_mpo* D1, const qtt_mpo* D2, double h, double mu, int max_sweeps, double sweep_tol,
                                 int cg_maxit, double cg_tol, int* sweeps_host, long long* cg_iterations_host,
                                 int* cg_max_host) {
  if (!ctx || !v || !a || !B || !D1 || !D2 || !(h > 0.0) || mu < 0.0 || max_sweeps < 1 || cg_maxit < 0 || sweep_tol < 0.0 ||
      cg_tol < 0.0)
    return QTT_INVALID_ARG;
  for (int i = 0; i < 2; ++i)
    if (!v[i] || !a[i] || !B[i]) return QTT_INVALID_ARG;
  QTT_API_BEGIN
  set_device(ctx);
  if (ctx->d != 4) QTT_THROW(QTT_INVALID_ARG, "qtt_variational_stage is built for the 2D encoding (physical dimension 4)");
  ArenaScope scope(ctx);
  View vv[2], va[2], vb[2];
  for (int i = 0; i < 2; ++i) {
    vv[i] = materialize(ctx, v[i]->body);
    va[i] = materialize(ctx, a[i]->body);
    vb[i] = materialize(ctx, B[i]->body);
  }
  Body* fresh[2] = {nullptr, nullptr};
  try {
    OutMps out[2];
    for (int i = 0; i < 2; ++i) {
      fresh[i] = body_new_dense(ctx, vv[i].r);
      out[i] = out_of_body(fresh[i]);
    }
    qtt_variational_stage_impl(ctx, vv, va, vb, D1->data, D2->data, h, mu, max_sweeps, sweep_tol, cg_maxit, cg_tol, out,
                               sweeps_host, cg_iterations_host, cg_max_host);
    for (int i = 0; i < 2; ++i) body_set_bonds(fresh[i], out[i].r);
  } catch (...) {
    for (Body* b : fresh) body_release(b);
    throw;
  }
  for (int i = 0; i < 2; ++i) {
    body_release(v[i]->body);
    v[i]->body = fresh[i];
  }
  check_numeric(ctx);
  QTT_API_END(ctx)
}

// ------------------------------------------------------------------------------------------ diagnostics
int qtt_diag_gemm(void* stream, const double* A, const double* B, double* C, int M, int N, int K, int transA,
                  int transB, long long lda, long long ldb, long long ldc, double alpha, double beta, int nbatch,
                  long long sa, long long sb, long long sc) {
  GemmProb p;
  std::memset(&p, 0, sizeof(p));
  p.A = A; p.B = B; p.C = C;
  p.M = M; p.N = N; p.K = K;
  p.nbatch = nbatch;
  if (transA) { p.a_lo = 1; p.a_k = lda; } else { p.a_lo = lda; p.a_k = 1; }
  if (transB) { p.b_k = 1; p.b_n = ldb; } else { p.b_k = ldb; p.b_n = 1; }
  p.c_lo = ldc; p.c_n = 1;
  p.a_bs = sa; p.b_bs = sb; p.c_bs = sc;
  p.alpha = alpha; p.beta = beta;
  return (int)qtt_launch_gemm(&p, 1, static_cast<cudaStream_t>(stream));
}

int qtt_diag_lq(void* stream, double* Y, int batch, int k, int m, int ld, double* R, double* scratch) {
  if (k <= m && qtt_qrcp_fits(m, k)) {  // the cluster-resident Householder kernel, as in the sweeps
    std::vector<QrcpProb> qp(batch);
    for (int i = 0; i < batch; ++i) qp[i] = QrcpProb{Y + (size_t)i * k * ld, m, k, ld, nullptr, 1, R + (size_t)i * k * k};
    return (int)qtt_launch_qrcp(qp.data(), batch, 0, static_cast<cudaStream_t>(stream));
  }
  std::vector<LqProb> probs(batch);
  std::vector<TriProb> tris(batch);
  const size_t s = qtt_lq_scratch_doubles(m);
  for (int i = 0; i < batch; ++i) {
    probs[i].Y = Y + (size_t)i * k * ld;
    probs[i].k = k; probs[i].m = m; probs[i].ld = ld;
    probs[i].V = scratch + (size_t)i * 3 * s;
    probs[i].TV = probs[i].V + s;
    probs[i].W = probs[i].TV + s;
    tris[i] = TriProb{probs[i].Y, k, ld, R + (size_t)i * k * k, k};
  }
  cudaError_t e = qtt_launch_lq(probs.data(), batch, static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return (int)e;
  return (int)qtt_launch_extract_tri(tris.data(), batch, 0, static_cast<cudaStream_t>(stream));
}

int qtt_diag_rowjacobi(void* stream, double* X, int batch, int p, int q, int ld, int* status) {
  std::vector<JacProb> probs(batch);
  for (int i = 0; i < batch; ++i) {
    probs[i].X = X + (size_t)i * p * ld;
    probs[i].p = p; probs[i].q = q; probs[i].ld = ld;
    probs[i].p_dev = nullptr;
    probs[i].work = nullptr;
    probs[i].sweep_cap = 0;
    probs[i].status = status;
  }
  return (int)qtt_launch_rowjacobi(probs.data(), batch, static_cast<cudaStream_t>(stream));
}

int qtt_diag_rowjacobi_streamed(void* stream, double* X, int batch, int p, int q, int ld, int* status, double* work) {
  if (!qtt_sbj_fits(p, q) || !work) return (int)cudaErrorInvalidConfiguration;
  std::vector<JacProb> probs(batch);
  for (int i = 0; i < batch; ++i) {
    probs[i].X = X + (size_t)i * p * ld;
    probs[i].p = p; probs[i].q = q; probs[i].ld = ld;
    probs[i].p_dev = nullptr;
    probs[i].work = work + 8 * (size_t)i;
    probs[i].sweep_cap = 0;
    probs[i].status = status;
  }
  return (int)qtt_launch_sbj(probs.data(), batch, static_cast<cudaStream_t>(stream));
}

int qtt_diag_svd_rows(void* stream, double* X, int batch, int p, int q, int ld, int* rank_dev, int* status) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (!qtt_qrcp_fits(p, q)) return (int)cudaErrorInvalidConfiguration;
  std::vector<QrcpProb> qp(batch);
  std::vector<JacProb> probs(batch);
  for (int i = 0; i < batch; ++i) {
    qp[i] = QrcpProb{X + (size_t)i * p * ld, p, q, ld, rank_dev + i, 0, nullptr};
    probs[i].X = qp[i].X;
    probs[i].p = p < q ? p : q; probs[i].q = q; probs[i].ld = ld;
    probs[i].p_dev = rank_dev + i;
    probs[i].work = nullptr;
    probs[i].sweep_cap = 0;
    probs[i].status = status;
  }
  cudaError_t e = qtt_launch_qrcp(qp.data(), batch, 1, st);
  if (e != cudaSuccess) return (int)e;
  if (!status) return 0;  // status == NULL: preconditioner only
  return (int)qtt_launch_rowjacobi(probs.data(), batch, st);
}

int qtt_diag_select(void* stream, const double* X, int p, int q, int ld, double* out, int r_cap, double* sigma,
                    int* rank, int chi_max, double delta) {
  // delta >= 0 is passed through a one-shot device scalar living at the end of `sigma` (p+1 doubles needed)
  SelProb s;
  std::memset(&s, 0, sizeof(s));
  s.X = X; s.p = p; s.q = q; s.ld = ld;
  s.out = out; s.out_ld = q; s.r_cap = r_cap;
  s.sigma = sigma; s.rank = rank;
  s.chi_max = chi_max;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (delta >= 0.0) {
    cudaError_t e = qtt_launch_fill(sigma + p, 1, delta, st);
    if (e != cudaSuccess) return (int)e;
    s.delta_ptr = sigma + p;
  }
  return (int)qtt_launch_select(&s, 1, st);
}

}  // extern "C"
