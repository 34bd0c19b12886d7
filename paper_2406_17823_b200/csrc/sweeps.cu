// Batched rounding sweeps of the QTT step, sequencing the kernels of
// common.cuh.  The rounding is "Q-less": the L->R sweep keeps only the triangular factors R_k of the left
// blocks, and the R->L sweep works in the original gauge with R_{k-1} as the metric,
//     M = R_{k-1} (A_k C_k),  rows of J M = Sigma V^T,  core'_k = V^T[:r'],  C_{k-1} = (A_k C_k) V[:, :r'],
// which is the same truncation as oracle O6 (QR sweep, then truncated SVDs) without ever forming a Q.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "engine.cuh"



// ------------------------------------------------------------------------------------------ arena
double* Arena::keep(size_t doubles) {
  size_t bytes = (doubles * sizeof(double) + 255) & ~(size_t)255;
  if (lo + bytes > hi) QTT_THROW(QTT_CAPACITY, "workspace exhausted (keep stack)");
  double* p = reinterpret_cast<double*>(base + lo);
  lo += bytes;
  return p;
}
double* Arena::tmp(size_t doubles) {
  size_t bytes = (doubles * sizeof(double) + 255) & ~(size_t)255;
  if (bytes > hi || hi - bytes < lo) QTT_THROW(QTT_CAPACITY, "workspace exhausted (tmp stack)");
  hi -= bytes;
  return reinterpret_cast<double*>(base + hi);
}

// ------------------------------------------------------------------------------------------ shapes
std::vector<int> qtt_round_caps(const std::vector<int>& r, int chi, int d) {
  const int n = (int)r.size() - 1;
  std::vector<int> p(n + 1), out(n + 1);
  p[0] = 1;
  for (int k = 1; k <= n; ++k) p[k] = (int)std::min<long long>((long long)d * p[k - 1], r[k]);
  out[n] = 1;
  for (int k = n - 1; k >= 1; --k) out[k] = std::max(1, (int)std::min<long long>(std::min(chi, p[k]), (long long)d * out[k + 1]));
  out[0] = 1;
  return out;
}

void qtt_zip_caps(const std::vector<int>& ra, const std::vector<int>& rb, int chi, int chi_work,
                  std::vector<int>& rwork, std::vector<int>& rout, int d) {
  const int n = (int)ra.size() - 1;
  rwork.assign(n + 1, 1);
  for (int k = 1; k < n; ++k) {
    long long kk = (long long)ra[k] * rb[k];
    long long m = (long long)d * rwork[k - 1];
    rwork[k] = (int)std::min<long long>(std::min(m, kk), chi_work);
  }
  rout.assign(n + 1, 1);
  for (int k = n - 1; k >= 1; --k) rout[k] = std::max(1, (int)std::min<long long>(std::min(chi, rwork[k]), (long long)d * rout[k + 1]));
}

// ------------------------------------------------------------------------------------------ helpers
namespace {

void run_gemms(qtt_ctx* ctx, std::vector<GemmProb>& v) {
  if (v.empty()) return;
  QTT_CU(qtt_launch_gemm(v.data(), (int)v.size(), ctx->stream));
  v.clear();
}

constexpr int LQ_MAX_M = 16384;
constexpr int LQ_CHUNK = 8192;

struct LqJob {
  double* Y;  // k x m, ld, destroyed
  int k, m, ld;
  double* R;  // k x k upper triangular out (ld = k)
};

// Q-less LQ of a batch; very wide matrices go through a TSQR tree over column chunks.
void run_lq(qtt_ctx* ctx, std::vector<LqJob>& jobs) {
  if (jobs.empty()) return;
  std::vector<LqProb> probs;
  std::vector<TriProb> tris;
  std::vector<LqJob> next;  // second-level jobs of the TSQR tree
  std::vector<QrcpProb> resident;  // small enough for the cluster-resident Householder kernel (qrcp.cu)
  for (const LqJob& j : jobs) {
    if (j.k > j.m) QTT_THROW(QTT_INVALID_ARG, "internal: LQ needs k <= m");
    if (qtt_qrcp_fits(j.m, j.k)) {
      resident.push_back(QrcpProb{j.Y, j.m, j.k, j.ld, nullptr, 1, j.R});
    } else if (j.m <= LQ_MAX_M) {
      LqProb p;
      p.Y = j.Y; p.k = j.k; p.m = j.m; p.ld = j.ld;
      p.V = p.TV = p.W = nullptr;
      probs.push_back(p);
      tris.push_back(TriProb{j.Y, j.k, j.ld, j.R, j.k});
    } else {
      const int chunk = std::max(LQ_CHUNK, j.k);
      const int nch = (j.m + chunk - 1) / chunk;
      // [L_1 | L_2 | ...] with the last chunk possibly narrower than k (then it is copied as it is)
      std::vector<int> widths;
      int total = 0;
      for (int c = 0; c < nch; ++c) {
        int mc = std::min(chunk, j.m - c * chunk);
        widths.push_back(mc);
        total += std::min(mc, j.k);
      }
      double* stack = ctx->arena.tmp((size_t)j.k * total);
      int off = 0;
      for (int c = 0; c < nch; ++c) {
        int mc = widths[c];
        double* Yc = j.Y + (size_t)c * chunk;
        if (mc >= j.k) {
          LqProb p;
          p.Y = Yc; p.k = j.k; p.m = mc; p.ld = j.ld;
          p.V = p.TV = p.W = nullptr;
          probs.push_back(p);
          tris.push_back(TriProb{Yc, j.k, j.ld, stack + off, total});  // mode 1 below
          off += j.k;
        } else {
          QTT_CU(qtt_launch_copy2d(Yc, j.k, mc, j.ld, stack + off, total, ctx->stream));
          off += mc;
        }
      }
      next.push_back(LqJob{stack, j.k, total, total, j.R});
    }
  }
  if (!resident.empty()) QTT_CU(qtt_launch_qrcp(resident.data(), (int)resident.size(), 0, ctx->stream));
  // reflector scratch: the launcher runs consecutive groups of QTT_LQ_MAX_BATCH problems one after the
  // other on the stream, so problem i can share the scratch slot i % QTT_LQ_MAX_BATCH
  {
    int mmax = 0;
    for (const LqProb& p : probs) mmax = std::max(mmax, p.m);
    const int nslot = std::min<int>((int)probs.size(), QTT_LQ_MAX_BATCH);
    std::vector<double*> slotV(nslot), slotTV(nslot), slotW(nslot);
    for (int s2 = 0; s2 < nslot; ++s2) {
      slotV[s2] = ctx->arena.tmp(qtt_lq_scratch_doubles(mmax));
      slotTV[s2] = ctx->arena.tmp(qtt_lq_scratch_doubles(mmax));
      slotW[s2] = ctx->arena.tmp(qtt_lq_scratch_doubles(mmax));
    }
    for (size_t i = 0; i < probs.size(); ++i) {
      probs[i].V = slotV[i % QTT_LQ_MAX_BATCH];
      probs[i].TV = slotTV[i % QTT_LQ_MAX_BATCH];
      probs[i].W = slotW[i % QTT_LQ_MAX_BATCH];
    }
  }
  // direct problems and chunk problems share the panel launches; their triangles are extracted separately
  if (!probs.empty()) QTT_CU(qtt_launch_lq(probs.data(), (int)probs.size(), ctx->stream));
  std::vector<TriProb> t0, t1;
  {
    size_t ti = 0;
    for (const LqJob& j : jobs) {
      if (qtt_qrcp_fits(j.m, j.k)) continue;
      if (j.m <= LQ_MAX_M) {
        t0.push_back(tris[ti++]);
      } else {
        const int chunk = std::max(LQ_CHUNK, j.k);
        const int nch = (j.m + chunk - 1) / chunk;
        for (int c = 0; c < nch; ++c)
          if (std::min(chunk, j.m - c * chunk) >= j.k) t1.push_back(tris[ti++]);
      }
    }
  }
  if (!t0.empty()) QTT_CU(qtt_launch_extract_tri(t0.data(), (int)t0.size(), 0, ctx->stream));
  if (!t1.empty()) QTT_CU(qtt_launch_extract_tri(t1.data(), (int)t1.size(), 1, ctx->stream));
  jobs.clear();
  if (!next.empty()) run_lq(ctx, next);
}

struct SvdJob {
  double* X;  // p x q (ld = q), destroyed: rows orthogonalised in place
  int p, q;
  double* out;  // r_cap x q
  int r_cap, chi_max;
  double* sigma;  // p doubles or nullptr
  int* rank;      // device int
  const double* delta_ptr;
  double* delta_out;
  double delta_scale;
  bool rank_deficient = false;  // expanded / direct-sum cores (rows a1, a3): rank-deficient by construction
};

// right singular vectors by row-Jacobi, preconditioned by a rank-revealing pivoted QR (qrcp.cu): X <- Q^T X has
// graded rows (7-9 Jacobi sweeps instead of 20-45) and only its first rank(X) rows are non-zero, so the Jacobi
// kernel rotates rank(X) rows.  Inputs too large for the cluster-resident QR are first reduced to their
// triangular factor by the blocked LQ.
void run_svd(qtt_ctx* ctx, std::vector<SvdJob>& jobs) {
  if (jobs.empty()) return;
  std::vector<LqJob> lq;
  for (SvdJob& j : jobs) {
    if (!qtt_qrcp_fits(j.p, j.q) && j.p > j.q && j.p >= 8) {
      // X = Q R_X, same right singular vectors: R_X (q x q) from the LQ of X^T (q x p)
      double* Xt = ctx->arena.tmp((size_t)j.q * j.p);
      QTT_CU(qtt_launch_transpose(j.X, j.p, j.q, j.q, Xt, j.p, ctx->stream));
      double* R = ctx->arena.tmp((size_t)j.q * j.q);
      lq.push_back(LqJob{Xt, j.q, j.p, j.p, R});
      j.X = R;
      j.p = j.q;
    }
  }
  run_lq(ctx, lq);
  std::vector<QrcpProb> qp;
  std::vector<JacProb> jp;
  std::vector<SelProb> sp;
  for (const SvdJob& j : jobs) {
    if (j.p > qtt_select_max_rows())
      QTT_THROW(QTT_CAPACITY, "SVD with " + std::to_string(j.p) + " rows: the rank selection sorts at most " +
                                  std::to_string(qtt_select_max_rows()) + " rows");
    int prow = j.p;
    const int* rank_dev = nullptr;
    // (the zip-up's triangular factors are preconditioned too: measured on the config-3 step, skipping the pivoted QR
    // for them raises the Jacobi sweep count from 11 to 20)
    if (j.p >= 2 && qtt_qrcp_fits(j.p, j.q)) {
      int* rk = reinterpret_cast<int*>(ctx->arena.tmp(1));
      qp.push_back(QrcpProb{j.X, j.p, j.q, j.q, rk, 0, nullptr});
      rank_dev = rk;
      prow = std::min(j.p, j.q);  // the rows below are exact zeros after the QR
    }
    JacProb a;
    a.X = j.X; a.p = prow; a.q = j.q; a.ld = j.q; a.p_dev = rank_dev; a.status = ctx->jac_status;
    a.work = ctx->arena.tmp(8);
    // without the pivoted-QR preconditioner (matrix too large for a cluster's shared memory) a rank-deficient input
    // needs 20-45 sweeps; the zip-up's full-rank triangular factors need < 20
    a.sweep_cap = (rank_dev == nullptr && j.rank_deficient) ? 60 : 0;
    jp.push_back(a);
    SelProb s;
    s.X = j.X; s.p = prow; s.q = j.q; s.ld = j.q;
    s.out = j.out; s.out_ld = j.q; s.r_cap = j.r_cap;
    s.sigma = j.sigma; s.rank = j.rank;
    s.delta_ptr = j.delta_ptr; s.delta_out = j.delta_out; s.delta_scale = j.delta_scale;
    s.chi_max = j.chi_max;
    sp.push_back(s);
  }
  if (!qp.empty()) QTT_CU(qtt_launch_qrcp(qp.data(), (int)qp.size(), 1, ctx->stream));
  QTT_CU(qtt_launch_rowjacobi(jp.data(), (int)jp.size(), ctx->stream));
  QTT_CU(qtt_launch_select(sp.data(), (int)sp.size(), ctx->stream));
  jobs.clear();
}

// one site tensor seen from the R->L sweep
struct LeftCore {
  const double* ptr;
  int rl, rr;
  int form;  // 0: dense [rl][4][rr]; 1: transposed isometry Qt [rr][4*rl]; 2: identity (rr == 4*rl)
};
struct SweepItem {
  int n;
  std::vector<LeftCore> core;
  std::vector<const double*> Rf;  // bond k = 1..n-1: metric factor (pk[k] x core[k].rl), nullptr = identity
  std::vector<int> pk;
};

// R->L truncated-SVD sweep (oracle O6 step ii) for a batch.
void sweep_rl(qtt_ctx* ctx, std::vector<SweepItem>& items, int chi, double eps, std::vector<OutMps>& out,
              SigmaCapture* cap) {
  const int d = ctx->d;
  const int nb = (int)items.size();
  const int n = items[0].n;
  std::vector<const double*> C(nb, ctx->ones);
  std::vector<int> rc(nb, 1);
  std::vector<double*> delta(nb, nullptr);
  std::vector<int*> rank_dev(nb, nullptr);
  std::vector<int> rank_host(nb, 0);
  std::vector<double*> Cbuf[2];
  Cbuf[0].assign(nb, nullptr);
  Cbuf[1].assign(nb, nullptr);
  for (int i = 0; i < nb; ++i) {
    out[i].r.assign(n + 1, 1);
    if (eps > 0.0) delta[i] = ctx->arena.tmp(1);
    rank_dev[i] = reinterpret_cast<int*>(ctx->arena.tmp(1));
    size_t mx = 1;
    for (int k = 1; k < n; ++k) mx = std::max(mx, (size_t)items[i].core[k].rl * out[i].rcap[k]);
    Cbuf[0][i] = ctx->arena.tmp(mx);
    Cbuf[1][i] = ctx->arena.tmp(mx);
  }
  std::vector<GemmProb> g;
  for (int k = n - 1; k >= 1; --k) {
    const size_t site_mark = ctx->arena.hi;
    std::vector<const double*> B(nb);
    std::vector<SvdJob> svd;
    std::vector<GemmProb> g2;
    // B = core_k * C   (r_k x 4 rc)
    for (int i = 0; i < nb; ++i) {
      const LeftCore& c = items[i].core[k];
      const int q = d * rc[i];
      if (c.form == 2) {
        B[i] = C[i];
      } else if (c.rr == 1 && rc[i] == 1 && C[i] == ctx->ones) {
        B[i] = c.ptr;
      } else {
        double* Bb = ctx->arena.tmp((size_t)c.rl * q);
        if (c.form == 0)
          g.push_back(gemm_nn(c.ptr, c.rr, C[i], rc[i], Bb, rc[i], d * c.rl, rc[i], c.rr));
        else
          g.push_back(gemm_tn(c.ptr, d * c.rl, C[i], rc[i], Bb, rc[i], d * c.rl, rc[i], c.rr));
        B[i] = Bb;
      }
    }
    run_gemms(ctx, g);
    // M = R_{k} * B  (pk x 4 rc), or a copy of B when the left block is an isometry
    for (int i = 0; i < nb; ++i) {
      const LeftCore& c = items[i].core[k];
      const int q = d * rc[i];
      const int p = items[i].Rf[k] ? items[i].pk[k] : c.rl;
      double* Mb = ctx->arena.tmp((size_t)p * q);
      if (items[i].Rf[k])
        g.push_back(gemm_nn(items[i].Rf[k], c.rl, B[i], q, Mb, q, p, q, c.rl));
      else
        QTT_CU(qtt_launch_copy2d(B[i], p, q, q, Mb, q, ctx->stream));
      SvdJob j;
      j.X = Mb; j.p = p; j.q = q;
      j.out = out[i].core[k];
      j.r_cap = out[i].rcap[k];
      j.chi_max = std::min(chi, out[i].rcap[k]);
      j.sigma = nullptr;
      if (cap) {
        j.sigma = ctx->arena.keep((size_t)p);
        cap->sigma[i][k] = j.sigma;
        cap->count[i][k] = std::min(p, q);
      }
      j.rank = rank_dev[i];
      j.rank_deficient = true;
      j.delta_ptr = nullptr; j.delta_out = nullptr; j.delta_scale = 0.0;
      if (eps > 0.0) {
        if (k == n - 1) {
          j.delta_out = delta[i];
          j.delta_scale = eps / std::sqrt((double)std::max(n - 1, 1));
        } else {
          j.delta_ptr = delta[i];
        }
      }
      svd.push_back(j);
    }
    run_gemms(ctx, g);
    run_svd(ctx, svd);
    // ranks
    for (int i = 0; i < nb; ++i) {
      const LeftCore& c = items[i].core[k];
      const int p = items[i].Rf[k] ? items[i].pk[k] : c.rl;
      rank_host[i] = std::max(1, std::min(std::min(chi, out[i].rcap[k]), std::min(p, d * rc[i])));
    }
    if (eps > 0.0) {
      for (int i = 0; i < nb; ++i)
        QTT_CU(cudaMemcpyAsync(&rank_host[i], rank_dev[i], sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
      QTT_CU(cudaStreamSynchronize(ctx->stream));
    }
    // C_{k} <- B * core'^T   (r_k x r')
    for (int i = 0; i < nb; ++i) {
      const LeftCore& c = items[i].core[k];
      const int q = d * rc[i];
      const int rn = rank_host[i];
      double* Cn = Cbuf[k & 1][i];
      g2.push_back(gemm_nt(B[i], q, out[i].core[k], q, Cn, rn, c.rl, rn, q));
      out[i].r[k] = rn;
      C[i] = Cn;
      rc[i] = rn;
    }
    run_gemms(ctx, g2);
    ctx->arena.hi = site_mark;
  }
  // first site: core'_0 = core_0 * C  (4 x rc)
  for (int i = 0; i < nb; ++i) {
    const LeftCore& c = items[i].core[0];
    if (c.form == 2)
      QTT_CU(qtt_launch_copy2d(C[i], d, rc[i], rc[i], out[i].core[0], rc[i], ctx->stream));
    else if (c.form == 0)
      g.push_back(gemm_nn(c.ptr, c.rr, C[i], rc[i], out[i].core[0], rc[i], d * c.rl, rc[i], c.rr));
    else
      g.push_back(gemm_tn(c.ptr, d * c.rl, C[i], rc[i], out[i].core[0], rc[i], d * c.rl, rc[i], c.rr));
  }
  run_gemms(ctx, g);
}

}  // namespace

// Orthonormal basis of the row space of X (p x q, ld = q, destroyed): out (min(p, q) x q, ld = q) <- the right singular
// vectors of X as rows, in the order of decreasing singular value (rows belonging to singular values in the noise floor
// are zeros).  The SVD step of the sweeps on its own, for callers that move a canonical centre (variational.cu).
void qtt_row_space_basis(qtt_ctx* ctx, double* X, int p, int q, double* out) {
  std::vector<SvdJob> svd(1);
  SvdJob& j = svd[0];
  j.X = X; j.p = p; j.q = q;
  j.out = out;
  j.r_cap = std::min(p, q);
  j.chi_max = j.r_cap;
  j.sigma = nullptr;
  j.rank = reinterpret_cast<int*>(ctx->arena.tmp(1));
  j.delta_ptr = nullptr; j.delta_out = nullptr; j.delta_scale = 0.0;
  j.rank_deficient = true;
  run_svd(ctx, svd);
}

// ------------------------------------------------------------------------------------------ O6
void qtt_round_dense_batch(qtt_ctx* ctx, const std::vector<View>& in, int chi, double eps, std::vector<OutMps>& out,
                           SigmaCapture* cap) {
  const int d = ctx->d;
  const int nb = (int)in.size();
  if (nb == 0) return;
  const int n = in[0].n;
  for (const View& v : in)
    if (v.n != n) QTT_THROW(QTT_SHAPE_MISMATCH, "batched rounding needs operands with the same number of sites");
  if (cap) {
    cap->sigma.assign(nb, std::vector<double*>(n + 1, nullptr));
    cap->count.assign(nb, std::vector<int>(n + 1, 0));
  }
  if (n == 1) {
    for (int i = 0; i < nb; ++i) {
      QTT_CU(qtt_launch_copy2d(in[i].core[0], 1, d, d, out[i].core[0], d, ctx->stream));
      out[i].r.assign(2, 1);
    }
    return;
  }
  std::vector<SweepItem> items(nb);
  for (int i = 0; i < nb; ++i) {
    SweepItem& it = items[i];
    it.n = n;
    it.core.resize(n);
    for (int k = 0; k < n; ++k) it.core[k] = LeftCore{in[i].core[k], in[i].r[k], in[i].r[k + 1], 0};
    it.Rf.assign(n + 1, nullptr);
    it.pk.assign(n + 1, 1);
    it.Rf[0] = ctx->ones;
  }
  // ---- L->R: metric factors R_k of the left blocks (oracle O6 step i, without forming Q)
  std::vector<GemmProb> g;
  for (int k = 0; k < n - 1; ++k) {
    std::vector<LqJob> lq;
    // persistent factors first, scratch after the mark
    std::vector<double*> Rnew(nb, nullptr);
    for (int i = 0; i < nb; ++i) {
      SweepItem& it = items[i];
      const int r1 = in[i].r[k + 1];
      const int rows = d * it.pk[k], cols = r1;
      if (rows <= cols) {
        if (k > 0) Rnew[i] = ctx->arena.tmp((size_t)rows * cols);
      } else {
        Rnew[i] = ctx->arena.tmp((size_t)cols * cols);
      }
    }
    const size_t site_mark = ctx->arena.hi;
    for (int i = 0; i < nb; ++i) {
      SweepItem& it = items[i];
      const int rk = in[i].r[k], r1 = in[i].r[k + 1];
      const int pk = it.pk[k];
      const int rows = d * pk, cols = r1;
      if (rows <= cols) {
        if (k == 0) {
          it.Rf[1] = in[i].core[0];
        } else {
          g.push_back(gemm_nn(it.Rf[k], rk, in[i].core[k], d * (i64)r1, Rnew[i], d * (i64)r1, pk, d * r1, rk));
          it.Rf[k + 1] = Rnew[i];
        }
        it.pk[k + 1] = rows;
      } else {
        // Y = X^T (cols x rows), written transposed by the GEMM:  Y[b][(i,w)] = sum_a core[a,w,b] R[i,a]
        double* Y = ctx->arena.tmp((size_t)cols * rows);
        GemmProb p = gemm_base(in[i].core[k], it.Rf[k], Y, r1, pk, rk);
        p.nbatch = d;
        p.a_lo = 1; p.a_k = d * (i64)r1; p.a_bs = r1;
        p.b_k = 1; p.b_n = rk; p.b_bs = 0;
        p.c_lo = d * (i64)pk; p.c_n = d; p.c_bs = 1;
        g.push_back(p);
        lq.push_back(LqJob{Y, cols, rows, rows, Rnew[i]});
        it.Rf[k + 1] = Rnew[i];
        it.pk[k + 1] = cols;
      }
    }
    run_gemms(ctx, g);
    run_lq(ctx, lq);
    ctx->arena.hi = site_mark;
  }
  sweep_rl(ctx, items, chi, eps, out, cap);
}

// ------------------------------------------------------------------------------------------ O7
void qtt_round_product_batch(qtt_ctx* ctx, const std::vector<View>& A, const std::vector<View>& B, int chi, double eps,
                             int chi_work, std::vector<OutMps>& out) {
  const int d = ctx->d;
  const int nb = (int)A.size();
  if (nb == 0) return;
  const int n = A[0].n;
  for (int i = 0; i < nb; ++i)
    if (A[i].n != n || B[i].n != n) QTT_THROW(QTT_SHAPE_MISMATCH, "product operands differ in length");
  std::vector<SweepItem> items(nb);
  std::vector<const double*> R(nb, ctx->ones);
  std::vector<int> r(nb, 1);
  std::vector<double*> Rbuf[2];
  Rbuf[0].assign(nb, nullptr);
  Rbuf[1].assign(nb, nullptr);
  for (int i = 0; i < nb; ++i) {
    items[i].n = n;
    items[i].core.resize(n);
    items[i].Rf.assign(n + 1, nullptr);
    items[i].pk.assign(n + 1, 1);
    // carry R_l (rwork[l] x a_l b_l) ping-pongs between two buffers of the largest size
    std::vector<int> rw, ro;
    qtt_zip_caps(A[i].r, B[i].r, chi, chi_work, rw, ro, d);
    size_t mx = 1;
    for (int l = 1; l < n; ++l) mx = std::max(mx, (size_t)rw[l] * A[i].r[l] * B[i].r[l]);
    Rbuf[0][i] = ctx->arena.tmp(mx);
    Rbuf[1][i] = ctx->arena.tmp(mx);
  }
  std::vector<GemmProb> g;
  // ---- sketched zip-up (reading 25): where does each operand take the sketch, and the probes (a random sign tensor train of
  //      bond P = chi_work over the physical indices) seen from every bond, right to left:
  //      S_l[(a,b),t] = sum_{w,u} G_l[w][u,t] sum_{a',b'} A_l[a,w,a'] B_l[b,w,b'] S_{l+1}[(a',b'),u],   S_n = 1
  std::vector<std::vector<char>> sk(nb, std::vector<char>(n, 0));
  std::vector<std::vector<double*>> S(nb, std::vector<double*>(n + 1, nullptr));
  if (ctx->sketch && d != 4)
    QTT_THROW(QTT_INVALID_ARG, "the sketched product compression is built for physical dimension 4 only");
  if (ctx->sketch) {
    const int P = chi_work;
    int lmin_all = n;
    for (int i = 0; i < nb; ++i) {
      std::vector<int> rw, ro;
      qtt_zip_caps(A[i].r, B[i].r, chi, chi_work, rw, ro);
      int lmin = n;
      for (int l = 0; l + 1 < n; ++l) {
        const i64 m = 4ll * rw[l], kk = (i64)A[i].r[l + 1] * B[i].r[l + 1];
        const int rem = n - 1 - l;
        // configurations to the right: many (oversampled random range finder) or few (the probes span the whole range)
        const bool enough = rem >= 16 || (1ll << (2 * rem)) >= 2ll * chi_work || (1ll << (2 * rem)) <= (i64)chi_work;
        if (chi_work < std::min(m, kk) && enough) {
          sk[i][l] = 1;
          lmin = std::min(lmin, l);
        }
      }
      if (lmin == n) continue;
      lmin_all = std::min(lmin_all, lmin);
      S[i][n] = ctx->arena.tmp((size_t)P);
      QTT_CU(qtt_launch_fill(S[i][n], P, 1.0, ctx->stream));
      for (int l = n - 1; l > lmin; --l) S[i][l] = ctx->arena.tmp((size_t)A[i].r[l] * B[i].r[l] * P);
    }
    for (int l = n - 1; l > lmin_all; --l) {
      const size_t mark = ctx->arena.hi;
      double* G = ctx->arena.tmp((size_t)4 * P * P);
      QTT_CU(qtt_launch_sketch_mixers(ctx->sketch_seed, l, G, P, ctx->stream));
      std::vector<double*> X(nb, nullptr), Z(nb, nullptr);
      for (int i = 0; i < nb; ++i) {
        if (!S[i][l]) continue;
        const int a = A[i].r[l], a2 = A[i].r[l + 1], b2 = B[i].r[l + 1];
        X[i] = ctx->arena.tmp((size_t)4 * a * b2 * P);
        Z[i] = ctx->arena.tmp((size_t)4 * a * b2 * P);
        // X[a][w][(b',u)] = sum_a' A[a,w,a'] S_{l+1}[a'][(b',u)]
        g.push_back(gemm_nn(A[i].core[l], a2, S[i][l + 1], (i64)b2 * P, X[i], (i64)b2 * P, 4 * a, b2 * P, a2));
      }
      run_gemms(ctx, g);
      for (int i = 0; i < nb; ++i) {
        if (!S[i][l]) continue;
        const int a = A[i].r[l], b2 = B[i].r[l + 1];
        // Z[a][w][b'][t] = sum_u X[a][w][b'][u] G[w][u][t]      (rows (a,b') of the w-th slab; batched over w)
        GemmProb p = gemm_base(X[i], G, Z[i], a * b2, P, P);
        p.nbatch = 4;
        p.a_div = b2; p.a_hi = 4 * (i64)b2 * P; p.a_lo = P; p.a_k = 1; p.a_bs = (i64)b2 * P;
        p.b_k = P; p.b_n = 1; p.b_bs = (i64)P * P;
        p.c_div = b2; p.c_hi = 4 * (i64)b2 * P; p.c_lo = P; p.c_n = 1; p.c_bs = (i64)b2 * P;
        g.push_back(p);
      }
      run_gemms(ctx, g);
      for (int i = 0; i < nb; ++i) {
        if (!S[i][l]) continue;
        const int a = A[i].r[l], b = B[i].r[l], b2 = B[i].r[l + 1];
        // S_l[(a,b)][t] = sum_{(w,b')} B[b,(w,b')] Z[a][(w,b')][t]      (batched over a)
        GemmProb p = gemm_nn(B[i].core[l], 4 * (i64)b2, Z[i], P, S[i][l], P, b, P, 4 * b2);
        p.nbatch = a;
        p.a_bs = 0; p.b_bs = 4 * (i64)b2 * P; p.c_bs = (i64)b * P;
        g.push_back(p);
      }
      run_gemms(ctx, g);
      ctx->arena.hi = mark;
    }
  }
  for (int l = 0; l < n; ++l) {
    const size_t site_mark = ctx->arena.hi;
    std::vector<double*> T(nb);
    // X[i,(w,a'),b] = sum_a A[a,(w,a')] R[i,a,b]      (first half of the site contraction, row a2)
    std::vector<double*> X(nb);
    for (int i = 0; i < nb; ++i) {
      const int a = A[i].r[l], a2 = A[i].r[l + 1], b = B[i].r[l];
      X[i] = ctx->arena.tmp((size_t)r[i] * d * a2 * b);
      GemmProb p = gemm_base(A[i].core[l], R[i], X[i], d * a2, b, a);
      p.nbatch = r[i];
      p.a_lo = 1; p.a_k = d * (i64)a2; p.a_bs = 0;
      p.b_k = b; p.b_n = 1; p.b_bs = (i64)a * b;
      p.c_lo = b; p.c_n = 1; p.c_bs = d * (i64)a2 * b;
      g.push_back(p);
    }
    run_gemms(ctx, g);
    // T[(i,w),(a',b')] = sum_b X[i,w,a',b] B[b,w,b']   (second half)
    for (int i = 0; i < nb; ++i) {
      const int a2 = A[i].r[l + 1], b = B[i].r[l], b2 = B[i].r[l + 1];
      const size_t tsz = (size_t)d * r[i] * a2 * b2;
      T[i] = (l == n - 1) ? ctx->arena.keep(tsz) : ctx->arena.tmp(tsz);
      GemmProb p = gemm_base(X[i], B[i].core[l], T[i], r[i] * a2, b2, b);
      p.nbatch = d;
      p.a_div = a2; p.a_hi = d * (i64)a2 * b; p.a_lo = b; p.a_k = 1; p.a_bs = (i64)a2 * b;
      p.b_k = d * (i64)b2; p.b_n = 1; p.b_bs = b2;
      p.c_div = a2; p.c_hi = d * (i64)a2 * b2; p.c_lo = b2; p.c_n = 1; p.c_bs = (i64)a2 * b2;
      g.push_back(p);
    }
    run_gemms(ctx, g);
    if (l == n - 1) {
      for (int i = 0; i < nb; ++i) items[i].core[l] = LeftCore{T[i], r[i], 1, 0};
      ctx->arena.hi = site_mark;
      break;
    }
    // factorise T (m x kk): identity / truncated SVD keeping min(chi_work, m, kk) left singular vectors
    std::vector<LqJob> lq;
    std::vector<SvdJob> svd;
    std::vector<int> keep(nb, 0);
    std::vector<double*> Qt(nb, nullptr);
    for (int i = 0; i < nb; ++i) {
      const int m = d * r[i];
      const i64 kk = (i64)A[i].r[l + 1] * B[i].r[l + 1];
      if (m <= std::min<i64>(kk, chi_work)) {
        items[i].core[l] = LeftCore{nullptr, r[i], m, 2};
        keep[i] = 0;
        continue;
      }
      keep[i] = (int)std::min<i64>(std::min<i64>(m, kk), chi_work);
      Qt[i] = ctx->arena.keep((size_t)keep[i] * m);
      SvdJob j;
      if (sk[i][l]) {
        // cheaper compression (reading 25): Q = a basis of range(T S_{l+1}) with chi_work structured sign probes instead of the
        // top-chi_work left singular vectors: one GEMM and the SVD step of a chi_work x m matrix instead of the LQ of T and the
        // SVD of its m x m factor.   Yt[t][i] = sum_c S[c][t] T[i][c]
        double* Yt = ctx->arena.tmp((size_t)keep[i] * m);
        GemmProb p = gemm_base(S[i][l + 1], T[i], Yt, keep[i], m, (int)kk);
        p.a_lo = 1; p.a_k = keep[i];
        p.b_k = 1; p.b_n = kk;
        p.c_lo = m; p.c_n = 1;
        g.push_back(p);
        j.X = Yt; j.p = keep[i]; j.q = m;
        j.out = Qt[i]; j.r_cap = keep[i]; j.chi_max = keep[i];
        j.sigma = nullptr;
        j.rank = reinterpret_cast<int*>(ctx->arena.tmp(1));
        j.delta_ptr = nullptr; j.delta_out = nullptr; j.delta_scale = 0.0;
        j.rank_deficient = true;
        svd.push_back(j);
        continue;
      }
      if (m <= kk) {
        double* Tc = ctx->arena.tmp((size_t)m * kk);
        QTT_CU(cudaMemcpyAsync(Tc, T[i], sizeof(double) * (size_t)m * kk, cudaMemcpyDeviceToDevice, ctx->stream));
        double* R1 = ctx->arena.tmp((size_t)m * m);
        lq.push_back(LqJob{Tc, m, (int)kk, (int)kk, R1});
        j.X = R1; j.p = m; j.q = m;
      } else {
        double* Y = ctx->arena.tmp((size_t)kk * m);
        QTT_CU(qtt_launch_transpose(T[i], m, (int)kk, (int)kk, Y, m, ctx->stream));
        j.X = Y; j.p = (int)kk; j.q = m;
      }
      j.out = Qt[i]; j.r_cap = keep[i]; j.chi_max = keep[i];
      j.sigma = nullptr;
      j.rank = reinterpret_cast<int*>(ctx->arena.tmp(1));
      j.delta_ptr = nullptr; j.delta_out = nullptr; j.delta_scale = 0.0;
      svd.push_back(j);
    }
    run_gemms(ctx, g);  // (the sketches Y^T = Omega^T T^T, if any)
    run_lq(ctx, lq);
    run_svd(ctx, svd);
    // R' = Q^T T  (keep x kk), into the other carry buffer
    for (int i = 0; i < nb; ++i) {
      const int m = d * r[i];
      const i64 kk = (i64)A[i].r[l + 1] * B[i].r[l + 1];
      double* Rn = Rbuf[l & 1][i];
      if (keep[i] == 0) {
        QTT_CU(cudaMemcpyAsync(Rn, T[i], sizeof(double) * (size_t)m * kk, cudaMemcpyDeviceToDevice, ctx->stream));
        r[i] = m;
      } else {
        g.push_back(gemm_nn(Qt[i], m, T[i], kk, Rn, kk, keep[i], (int)kk, m));
        items[i].core[l] = LeftCore{Qt[i], r[i], keep[i], 1};
        r[i] = keep[i];
      }
      R[i] = Rn;
    }
    run_gemms(ctx, g);
    ctx->arena.hi = site_mark;
  }
  if (n == 1) {
    for (int i = 0; i < nb; ++i) {
      QTT_CU(qtt_launch_copy2d(items[i].core[0].ptr, 1, d, d, out[i].core[0], d, ctx->stream));
      out[i].r.assign(2, 1);
    }
    return;
  }
  sweep_rl(ctx, items, chi, eps, out, nullptr);
}

// ------------------------------------------------------------------------------------------ lazy kinds
void qtt_expand_apply_batch(qtt_ctx* ctx, const std::vector<const MpoData*>& W, const std::vector<View>& x,
                            std::vector<View>& out) {
  const int d = ctx->d;
  const int nb = (int)x.size();
  out.assign(nb, View());
  if (nb == 0) return;
  const int n = x[0].n;
  for (int i = 0; i < nb; ++i) {
    if (W[i]->n != x[i].n || x[i].n != n) QTT_THROW(QTT_SHAPE_MISMATCH, "MPO and MPS differ in length");
    out[i].n = n;
    out[i].r.resize(n + 1);
    out[i].core.resize(n);
    for (int k = 0; k <= n; ++k) out[i].r[k] = W[i]->D[k] * x[i].r[k];
  }
  for (int k = 0; k < n; ++k) {
    std::vector<ExpandProb> e;
    for (int i = 0; i < nb; ++i) {
      double* o = ctx->arena.tmp((size_t)out[i].r[k] * d * out[i].r[k + 1]);
      out[i].core[k] = o;
      e.push_back(ExpandProb{W[i]->core[k], x[i].core[k], o, W[i]->D[k], W[i]->D[k + 1], x[i].r[k], x[i].r[k + 1], d});
    }
    QTT_CU(qtt_launch_expand(e.data(), (int)e.size(), ctx->stream));
  }
}

View qtt_expand_apply(qtt_ctx* ctx, const MpoData* W, const View& x) {
  std::vector<View> out;
  qtt_expand_apply_batch(ctx, {W}, {x}, out);
  return out[0];
}

void qtt_concat_batch(qtt_ctx* ctx, const std::vector<std::vector<std::pair<double, View>>>& terms,
                      std::vector<View>& out) {
  const int d = ctx->d;
  const int nb = (int)terms.size();
  out.assign(nb, View());
  if (nb == 0) return;
  const int n = terms[0][0].second.n;
  for (int i = 0; i < nb; ++i) {
    if (terms[i].empty() || terms[i].size() > 5) QTT_THROW(QTT_INVALID_ARG, "a sum has 1..5 terms");
    out[i].n = n;
    out[i].r.assign(n + 1, 0);
    out[i].core.resize(n);
    for (auto& t : terms[i]) {
      if (t.second.n != n) QTT_THROW(QTT_SHAPE_MISMATCH, "summands differ in length");
      for (int k = 0; k <= n; ++k) out[i].r[k] += t.second.r[k];
    }
    out[i].r[0] = out[i].r[n] = 1;
  }
  for (int k = 0; k < n; ++k) {
    std::vector<ConcatProb> c;
    for (int i = 0; i < nb; ++i) {
      ConcatProb p;
      std::memset(&p, 0, sizeof(p));
      p.nterm = (int)terms[i].size();
      p.d = d;
      for (int t = 0; t < p.nterm; ++t) {
        p.src[t] = terms[i][t].second.core[k];
        p.alpha[t] = terms[i][t].first;
        p.rl[t] = terms[i][t].second.r[k];
        p.rr[t] = terms[i][t].second.r[k + 1];
      }
      p.mode = (n == 1) ? 3 : (k == 0 ? 0 : (k == n - 1 ? 2 : 1));
      double* o = ctx->arena.tmp((size_t)out[i].r[k] * d * out[i].r[k + 1]);
      out[i].core[k] = o;
      p.out = o;
      c.push_back(p);
    }
    if (n == 1) QTT_THROW(QTT_INVALID_ARG, "sums of one-site MPS are not supported");
    QTT_CU(qtt_launch_concat(c.data(), (int)c.size(), ctx->stream));
  }
}

View qtt_kron(qtt_ctx* ctx, const View& a, const View& b) {
  if (a.n != b.n) QTT_THROW(QTT_SHAPE_MISMATCH, "product operands differ in length");
  const int d = ctx->d;
  View o;
  o.n = a.n;
  o.r.resize(a.n + 1);
  o.core.resize(a.n);
  for (int k = 0; k <= a.n; ++k) o.r[k] = a.r[k] * b.r[k];
  for (int k = 0; k < a.n; ++k) {
    double* out = ctx->arena.tmp((size_t)o.r[k] * d * o.r[k + 1]);
    KronProb p{a.core[k], b.core[k], out, a.r[k], a.r[k + 1], b.r[k], b.r[k + 1], d};
    QTT_CU(qtt_launch_kron(&p, 1, ctx->stream));
    o.core[k] = out;
  }
  return o;
}

// ------------------------------------------------------------------------------------------ boundary
void qtt_to_dense_view(qtt_ctx* ctx, const View& v, double* dense_dev_out) {
  const int d = ctx->d, ndim = d == 8 ? 3 : 2;
  const int n = v.n;
  if (ndim * n > 30) QTT_THROW(QTT_CAPACITY, "grid too large for a dense array");
  const double* T = v.core[0];  // 4 x r_1
  i64 rows = d;
  std::vector<GemmProb> g;
  for (int k = 1; k < n; ++k) {
    double* Tn = ctx->arena.tmp((size_t)rows * d * v.r[k + 1]);
    g.push_back(gemm_nn(T, v.r[k], v.core[k], d * (i64)v.r[k + 1], Tn, d * (i64)v.r[k + 1], (int)rows, d * v.r[k + 1],
                        v.r[k]));
    run_gemms(ctx, g);
    T = Tn;
    rows *= d;
  }
  QTT_CU(qtt_launch_interleave(T, dense_dev_out, n, ndim, 1, ctx->stream));
}

void qtt_from_dense(qtt_ctx* ctx, const double* dense_dev, int nbits, int chi, double eps, OutMps& out) {
  const int d = ctx->d, ndim = d == 8 ? 3 : 2;
  const int n = nbits;
  if (ndim * n > 30) QTT_THROW(QTT_CAPACITY, "grid too large for a dense array");
  const i64 total = 1ll << (ndim * n);
  double* carry = ctx->arena.tmp((size_t)total);
  QTT_CU(qtt_launch_interleave(dense_dev, carry, n, ndim, 0, ctx->stream));
  out.r.assign(n + 1, 1);
  if (n == 1) {
    QTT_CU(qtt_launch_copy2d(carry, 1, d, d, out.core[0], d, ctx->stream));
    return;
  }
  int rc = 1;
  double* delta = eps > 0.0 ? ctx->arena.tmp(1) : nullptr;
  int* rank_dev = reinterpret_cast<int*>(ctx->arena.tmp(1));
  std::vector<GemmProb> g;
  for (int k = n - 1; k >= 1; --k) {
    // unfolding M: d^k x (d rc)
    const i64 rows = 1ll << (ndim * k);
    const int q = d * rc;
    if (rows > 2147483647ll / std::max(q, 1)) QTT_THROW(QTT_CAPACITY, "grid too large");
    std::vector<SvdJob> svd;
    SvdJob j;
    if (rows <= q || rows < 8) {
      double* Mc = ctx->arena.tmp((size_t)rows * q);
      QTT_CU(qtt_launch_copy2d(carry, (int)rows, q, q, Mc, q, ctx->stream));
      j.X = Mc; j.p = (int)rows; j.q = q;
    } else {
      // same right singular vectors as its triangular factor: LQ of M^T (q x rows)
      double* Mt = ctx->arena.tmp((size_t)rows * q);
      QTT_CU(qtt_launch_transpose(carry, (int)rows, q, q, Mt, (int)rows, ctx->stream));
      double* R = ctx->arena.tmp((size_t)q * q);
      std::vector<LqJob> lq{LqJob{Mt, q, (int)rows, (int)rows, R}};
      run_lq(ctx, lq);
      j.X = R; j.p = q; j.q = q;
    }
    j.out = out.core[k];
    j.r_cap = out.rcap[k];
    j.chi_max = std::min(chi, out.rcap[k]);
    j.sigma = nullptr;
    j.rank = rank_dev;
    j.delta_ptr = nullptr; j.delta_out = nullptr; j.delta_scale = 0.0;
    if (eps > 0.0) {
      if (k == n - 1) {
        j.delta_out = delta;
        j.delta_scale = eps / std::sqrt((double)std::max(n - 1, 1));
      } else {
        j.delta_ptr = delta;
      }
    }
    svd.push_back(j);
    run_svd(ctx, svd);
    int rn = (int)std::max<i64>(1, std::min<i64>(std::min(chi, out.rcap[k]), std::min<i64>(rows, q)));
    if (eps > 0.0) {
      QTT_CU(cudaMemcpyAsync(&rn, rank_dev, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
      QTT_CU(cudaStreamSynchronize(ctx->stream));
    }
    // carry <- M * core'^T  (4^k x r')
    double* Cn = ctx->arena.tmp((size_t)rows * rn);
    g.push_back(gemm_nt(carry, q, out.core[k], q, Cn, rn, (int)rows, rn, q));
    run_gemms(ctx, g);
    carry = Cn;
    rc = rn;
    out.r[k] = rn;
  }
  QTT_CU(qtt_launch_copy2d(carry, d, rc, rc, out.core[0], rc, ctx->stream));
}

double* qtt_dot_view(qtt_ctx* ctx, const View& a, const View& b) {
  const int d = ctx->d;
  if (a.n != b.n) QTT_THROW(QTT_SHAPE_MISMATCH, "operands differ in length");
  const double* E = ctx->ones;  // ra x rb
  std::vector<GemmProb> g;
  for (int k = 0; k < a.n; ++k) {
    const int ra = a.r[k], rb = b.r[k], a2 = a.r[k + 1], b2 = b.r[k + 1];
    // G[b,(w,a')] = sum_a E[a,b] A[a,(w,a')]
    double* G = ctx->arena.tmp((size_t)rb * d * a2);
    g.push_back(gemm_tn(E, rb, a.core[k], d * (i64)a2, G, d * (i64)a2, rb, d * a2, ra));
    run_gemms(ctx, g);
    // E'[a',b'] = sum_{(b,w)} G[(b,w),a'] B[(b,w),b']
    double* En = ctx->arena.tmp((size_t)a2 * b2);
    g.push_back(gemm_tn(G, a2, b.core[k], b2, En, b2, a2, b2, d * rb));
    run_gemms(ctx, g);
    E = En;
  }
  return const_cast<double*>(E);
}

// ------------------------------------------------------------------------------------------ O8 / O9
namespace {

std::vector<OutMps> alloc_outs_keep(qtt_ctx* ctx, const std::vector<std::vector<int>>& caps) {
  std::vector<OutMps> out(caps.size());
  for (size_t i = 0; i < caps.size(); ++i) {
    const int n = (int)caps[i].size() - 1;
    out[i].n = n;
    out[i].rcap = caps[i];
    out[i].core.resize(n);
    for (int k = 0; k < n; ++k) out[i].core[k] = ctx->arena.keep((size_t)caps[i][k] * ctx->d * caps[i][k + 1]);
  }
  return out;
}
// Enqueue on the side stream with the side scratch region: swaps them into the context for the scope.
struct SideScope {
  qtt_ctx* ctx;
  size_t lo, hi;  // marks of the side scratch region, restored on exit (also when an exception unwinds the scope)
  explicit SideScope(qtt_ctx* c) : ctx(c) {
    std::swap(ctx->stream, ctx->side);
    std::swap(ctx->arena, ctx->side_arena);
    lo = ctx->arena.lo;
    hi = ctx->arena.hi;
  }
  ~SideScope() {
    ctx->arena.lo = lo;
    ctx->arena.hi = hi;
    std::swap(ctx->stream, ctx->side);
    std::swap(ctx->arena, ctx->side_arena);
  }
};
View view_of(const OutMps& o) {
  View v;
  v.n = o.n;
  v.r = o.r;
  v.core.assign(o.core.begin(), o.core.end());
  return v;
}

// f_i = -(u_1 (.) D_1 u_i + u_2 (.) D_2 u_i) + (1/Re) Lap u_i   (oracle O8)
void rhs(qtt_ctx* ctx, const View u[2], const MpoData* Dj[2], const MpoData* Lap, double Re, int chi, double eps,
         int chi_work, int skew, View f[2]) {
  // level 1: six applies + roundings: (D1 u_i, D2 u_i, Lap u_i) for i = 0, 1.  The two Laplacians are only needed by
  // level 3, so -- when the context has a side stream whose scratch region is large enough -- they are rounded
  // there, concurrently with the four D_j u_i on the main stream and with the products of level 2.
  std::vector<View> g(6);
  bool forked = false;
  {
    size_t need = (size_t)64 << 20;
    for (int i = 0; i < 2; ++i)
      for (int k = 0; k < u[i].n; ++k)
        need += (size_t)6 * 8 * 4 * (size_t)Lap->D[k] * u[i].r[k] * (size_t)Lap->D[k + 1] * u[i].r[k + 1];
    forked = ctx->side != nullptr && ctx->side_arena.size >= need;
  }
  if (forked) {
    std::vector<std::vector<int>> capsL;
    for (int i = 0; i < 2; ++i) {
      std::vector<int> re(u[i].n + 1);
      for (int k = 0; k <= u[i].n; ++k) re[k] = Lap->D[k] * u[i].r[k];
      capsL.push_back(qtt_round_caps(re, chi));
    }
    std::vector<OutMps> lout = alloc_outs_keep(ctx, capsL);  // results live in the main keep stack
    QTT_CU(cudaEventRecord(ctx->ev_fork, ctx->stream));
    QTT_CU(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
    {
      SideScope sc(ctx);  // ctx->stream / ctx->arena are the side stream and its scratch region in this scope
      const size_t mark = ctx->arena.hi;
      std::vector<const MpoData*> W{Lap, Lap};
      std::vector<View> X{u[0], u[1]};
      std::vector<View> ex;
      qtt_expand_apply_batch(ctx, W, X, ex);
      qtt_round_dense_batch(ctx, ex, chi, eps, lout);
      ctx->arena.hi = mark;
      QTT_CU(cudaEventRecord(ctx->ev_join, ctx->stream));
    }
    g[2] = view_of(lout[0]);
    g[5] = view_of(lout[1]);
    const size_t mark = ctx->arena.hi;
    std::vector<const MpoData*> W{Dj[0], Dj[1], Dj[0], Dj[1]};
    std::vector<View> X{u[0], u[0], u[1], u[1]};
    std::vector<View> ex;
    qtt_expand_apply_batch(ctx, W, X, ex);
    std::vector<std::vector<int>> caps;
    for (auto& e : ex) caps.push_back(qtt_round_caps(e.r, chi));
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_dense_batch(ctx, ex, chi, eps, out);
    g[0] = view_of(out[0]);
    g[1] = view_of(out[1]);
    g[3] = view_of(out[2]);
    g[4] = view_of(out[3]);
    ctx->arena.hi = mark;
  } else {
    const size_t mark = ctx->arena.hi;
    std::vector<const MpoData*> W{Dj[0], Dj[1], Lap, Dj[0], Dj[1], Lap};
    std::vector<View> X{u[0], u[0], u[0], u[1], u[1], u[1]};
    std::vector<View> ex;
    qtt_expand_apply_batch(ctx, W, X, ex);
    std::vector<std::vector<int>> caps;
    for (auto& e : ex) caps.push_back(qtt_round_caps(e.r, chi));
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_dense_batch(ctx, ex, chi, eps, out);
    for (int i = 0; i < 6; ++i) g[i] = view_of(out[i]);
    ctx->arena.hi = mark;
  }
  // level 2: four products c_ij = u_j (.) g_ij; with the skew-symmetric convection (PAPER.md:432-435 Eq. B2) also
  // p_11 = u_1 (.) u_1, p_12 = u_1 (.) u_2 (= p_21), p_22 = u_2 (.) u_2 in the same batch
  std::vector<View> c(4), pq(3);
  {
    const size_t mark = ctx->arena.hi;
    std::vector<View> A{u[0], u[1], u[0], u[1]};
    std::vector<View> B{g[0], g[1], g[3], g[4]};
    if (skew) {
      A.push_back(u[0]); B.push_back(u[0]);
      A.push_back(u[0]); B.push_back(u[1]);
      A.push_back(u[1]); B.push_back(u[1]);
    }
    std::vector<std::vector<int>> caps;
    for (size_t i = 0; i < A.size(); ++i) {
      std::vector<int> rw, ro;
      qtt_zip_caps(A[i].r, B[i].r, chi, chi_work, rw, ro);
      caps.push_back(ro);
    }
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_product_batch(ctx, A, B, chi, eps, chi_work, out);
    for (int i = 0; i < 4; ++i) c[i] = view_of(out[i]);
    if (skew)
      for (int i = 0; i < 3; ++i) pq[i] = view_of(out[4 + i]);
    ctx->arena.hi = mark;
  }
  // level 2b (skew only): d_ij = round(D_j p_ij) for (i,j) = (1,1), (1,2), (2,1), (2,2)
  std::vector<View> d(4);
  if (skew) {
    const size_t mark = ctx->arena.hi;
    std::vector<const MpoData*> W{Dj[0], Dj[1], Dj[0], Dj[1]};
    std::vector<View> X{pq[0], pq[1], pq[1], pq[2]};
    std::vector<View> ex;
    qtt_expand_apply_batch(ctx, W, X, ex);
    std::vector<std::vector<int>> caps;
    for (auto& e : ex) caps.push_back(qtt_round_caps(e.r, chi));
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_dense_batch(ctx, ex, chi, eps, out);
    for (int i = 0; i < 4; ++i) d[i] = view_of(out[i]);
    ctx->arena.hi = mark;
  }
  // level 3: f_i = -c_i1 - c_i2 + lap_i / Re, one rounding each
  if (forked) QTT_CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
  {
    const size_t mark = ctx->arena.hi;
    std::vector<std::vector<std::pair<double, View>>> terms(2);
    for (int i = 0; i < 2; ++i) {
      if (skew)
        terms[i] = {{-0.5, c[2 * i]}, {-0.5, c[2 * i + 1]}, {-0.5, d[2 * i]}, {-0.5, d[2 * i + 1]}, {1.0 / Re, g[3 * i + 2]}};
      else
        terms[i] = {{-1.0, c[2 * i]}, {-1.0, c[2 * i + 1]}, {1.0 / Re, g[3 * i + 2]}};
    }
    std::vector<View> s;
    qtt_concat_batch(ctx, terms, s);
    std::vector<std::vector<int>> caps;
    for (auto& e : s) caps.push_back(qtt_round_caps(e.r, chi));
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_dense_batch(ctx, s, chi, eps, out);
    for (int i = 0; i < 2; ++i) f[i] = view_of(out[i]);
    ctx->arena.hi = mark;
  }
}

void lincomb_round(qtt_ctx* ctx, const std::vector<std::vector<std::pair<double, View>>>& terms, int chi, double eps,
                   std::vector<OutMps>& out) {
  const size_t mark = ctx->arena.hi;
  std::vector<View> s;
  qtt_concat_batch(ctx, terms, s);
  qtt_round_dense_batch(ctx, s, chi, eps, out);
  ctx->arena.hi = mark;
}

// Three components on a 3D grid (d = 8; reading 26): f_i = -sum_j u_j (.) D_j u_i + (1/Re) Lap u_i (oracle rhs3),
// three batched levels: 12 applies + roundings, 9 zip-ups, 3 four-term sums.
void rhs3(qtt_ctx* ctx, const View u[3], const MpoData* const Dj[3], const MpoData* Lap, double Re, int chi, double eps,
          int chi_work, View f[3]) {
  const int d = ctx->d;
  std::vector<View> g(12);  // g[4 i + j] = round(D_j u_i), j < 3;  g[4 i + 3] = round(Lap u_i)
  {
    const size_t mark = ctx->arena.hi;
    std::vector<const MpoData*> W;
    std::vector<View> X;
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 4; ++j) {
        W.push_back(j < 3 ? Dj[j] : Lap);
        X.push_back(u[i]);
      }
    std::vector<View> ex;
    qtt_expand_apply_batch(ctx, W, X, ex);
    std::vector<std::vector<int>> caps;
    for (auto& e : ex) caps.push_back(qtt_round_caps(e.r, chi, d));
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_dense_batch(ctx, ex, chi, eps, out);
    for (int i = 0; i < 12; ++i) g[i] = view_of(out[i]);
    ctx->arena.hi = mark;
  }
  std::vector<View> c(9);  // c[3 i + j] = round(u_j (.) g_ij)
  {
    std::vector<View> A, B;
    std::vector<std::vector<int>> caps;
    size_t side_need = (size_t)64 << 20;
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        A.push_back(u[j]);
        B.push_back(g[4 * i + j]);
        std::vector<int> rw, ro;
        qtt_zip_caps(A.back().r, B.back().r, chi, chi_work, rw, ro, d);
        caps.push_back(ro);
        if (A.size() > 5) {  // scratch of one zip-up: carries, X, T, its copy, the LQ reflectors, factors
          size_t mx = 1;
          for (int l = 0; l + 1 < (int)rw.size() - 1; ++l)
            mx = std::max(mx, (size_t)d * rw[l] * A.back().r[l + 1] * B.back().r[l + 1]);
          side_need += 8 * sizeof(double) * mx;
        }
      }
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    // Only seven 16-CTA clusters are co-resident on the GPU (profiles/r2_three_d.md): nine factors in one launch run as
    // 7 + 2.  Two independent chains (five operands here, four on the side stream with its own scratch) share the seven
    // slots instead, each starting a kernel as soon as the other one leaves room.  Measured (bench.py --three-d): 64^3, chi = 32:
    // 240.0 -> 203.2 ms per step; 128^3, chi = 64, whose 1024-row factors take the L2-streamed Jacobi (one launch per tournament
    // round, no clusters): 1168 -> 1502 ms -- so only where the factors are cluster-resident (d chi_work <= 512 rows).
    const bool forked = ctx->side != nullptr && ctx->side_arena.size >= side_need && (long long)d * chi_work <= 512;
    if (forked) {
      std::vector<View> A1(A.begin(), A.begin() + 5), B1(B.begin(), B.begin() + 5), A2(A.begin() + 5, A.end()),
          B2(B.begin() + 5, B.end());
      std::vector<OutMps> o1(out.begin(), out.begin() + 5), o2(out.begin() + 5, out.end());
      QTT_CU(cudaEventRecord(ctx->ev_fork, ctx->stream));
      QTT_CU(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
      {
        SideScope sc(ctx);
        qtt_round_product_batch(ctx, A2, B2, chi, eps, chi_work, o2);
        QTT_CU(cudaEventRecord(ctx->ev_join, ctx->stream));
      }
      const size_t mark = ctx->arena.hi;
      qtt_round_product_batch(ctx, A1, B1, chi, eps, chi_work, o1);
      ctx->arena.hi = mark;
      QTT_CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
      for (int i = 0; i < 5; ++i) c[i] = view_of(o1[i]);
      for (int i = 0; i < 4; ++i) c[5 + i] = view_of(o2[i]);
    } else {
      const size_t mark = ctx->arena.hi;
      qtt_round_product_batch(ctx, A, B, chi, eps, chi_work, out);
      for (int i = 0; i < 9; ++i) c[i] = view_of(out[i]);
      ctx->arena.hi = mark;
    }
  }
  {
    const size_t mark = ctx->arena.hi;
    std::vector<std::vector<std::pair<double, View>>> terms(3);
    for (int i = 0; i < 3; ++i)
      terms[i] = {{-1.0, c[3 * i]}, {-1.0, c[3 * i + 1]}, {-1.0, c[3 * i + 2]}, {1.0 / Re, g[4 * i + 3]}};
    std::vector<View> s;
    qtt_concat_batch(ctx, terms, s);
    std::vector<std::vector<int>> caps;
    for (auto& e : s) caps.push_back(qtt_round_caps(e.r, chi, d));
    std::vector<OutMps> out = alloc_outs_keep(ctx, caps);
    qtt_round_dense_batch(ctx, s, chi, eps, out);
    for (int i = 0; i < 3; ++i) f[i] = view_of(out[i]);
    ctx->arena.hi = mark;
  }
}

}  // namespace

// Classical RK4 (Eq. 11) on three components in the d = 8 encoding (oracle rk4_step3); eager launches.
void qtt_rk4_eager3(qtt_ctx* ctx, const View u[3], const MpoData* const Dj[3], const MpoData* Lap, double Re, double dt,
                    int chi, double eps, int chi_work, OutMps out[3]) {
  const int d = ctx->d;
  View k1[3], k2[3], k3[3], k4[3], us[3];
  auto stage = [&](const View kk[3], double h, View dst[3]) {
    std::vector<std::vector<std::pair<double, View>>> terms(3);
    std::vector<std::vector<int>> caps;
    for (int i = 0; i < 3; ++i) {
      terms[i] = {{1.0, u[i]}, {h, kk[i]}};
      std::vector<int> rs(u[i].r.size());
      for (size_t b = 0; b < rs.size(); ++b) rs[b] = u[i].r[b] + kk[i].r[b];
      rs.front() = rs.back() = 1;
      caps.push_back(qtt_round_caps(rs, chi, d));
    }
    std::vector<OutMps> o = alloc_outs_keep(ctx, caps);
    lincomb_round(ctx, terms, chi, eps, o);
    for (int i = 0; i < 3; ++i) dst[i] = view_of(o[i]);
  };
  rhs3(ctx, u, Dj, Lap, Re, chi, eps, chi_work, k1);
  stage(k1, dt / 2, us);
  rhs3(ctx, us, Dj, Lap, Re, chi, eps, chi_work, k2);
  stage(k2, dt / 2, us);
  rhs3(ctx, us, Dj, Lap, Re, chi, eps, chi_work, k3);
  stage(k3, dt, us);
  rhs3(ctx, us, Dj, Lap, Re, chi, eps, chi_work, k4);
  std::vector<std::vector<std::pair<double, View>>> terms(3);
  for (int i = 0; i < 3; ++i)
    terms[i] = {{1.0, u[i]}, {dt / 6, k1[i]}, {dt / 3, k2[i]}, {dt / 3, k3[i]}, {dt / 6, k4[i]}};
  std::vector<OutMps> o{out[0], out[1], out[2]};
  lincomb_round(ctx, terms, chi, eps, o);
  for (int i = 0; i < 3; ++i) out[i] = o[i];
}

void qtt_rk4_eager(qtt_ctx* ctx, const View u[2], const MpoData* Dx, const MpoData* Dy, const MpoData* Lap, double Re,
                   double dt, int chi, double eps, int chi_work, int skew, OutMps out[2]) {
  const MpoData* Dj[2] = {Dx, Dy};
  View k1[2], k2[2], k3[2], k4[2], us[2];
  auto stage = [&](const View kk[2], double h, View dst[2]) {
    std::vector<std::vector<std::pair<double, View>>> terms(2);
    std::vector<std::vector<int>> caps;
    for (int i = 0; i < 2; ++i) {
      terms[i] = {{1.0, u[i]}, {h, kk[i]}};
      std::vector<int> rs(u[i].r.size());
      for (size_t b = 0; b < rs.size(); ++b) rs[b] = u[i].r[b] + kk[i].r[b];
      rs.front() = rs.back() = 1;
      caps.push_back(qtt_round_caps(rs, chi));
    }
    std::vector<OutMps> o = alloc_outs_keep(ctx, caps);
    lincomb_round(ctx, terms, chi, eps, o);
    for (int i = 0; i < 2; ++i) dst[i] = view_of(o[i]);
  };
  rhs(ctx, u, Dj, Lap, Re, chi, eps, chi_work, skew, k1);
  stage(k1, dt / 2, us);
  rhs(ctx, us, Dj, Lap, Re, chi, eps, chi_work, skew, k2);
  stage(k2, dt / 2, us);
  rhs(ctx, us, Dj, Lap, Re, chi, eps, chi_work, skew, k3);
  stage(k3, dt, us);
  rhs(ctx, us, Dj, Lap, Re, chi, eps, chi_work, skew, k4);
  std::vector<std::vector<std::pair<double, View>>> terms(2);
  for (int i = 0; i < 2; ++i)
    terms[i] = {{1.0, u[i]}, {dt / 6, k1[i]}, {dt / 3, k2[i]}, {dt / 3, k3[i]}, {dt / 6, k4[i]}};
  std::vector<OutMps> o{out[0], out[1]};
  lincomb_round(ctx, terms, chi, eps, o);
  out[0] = o[0];
  out[1] = o[1];
}
