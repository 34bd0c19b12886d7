// Finite-difference MPO builders of the C ABI (include/qtt.h: qtt_mpo_central_difference,
// qtt_mpo_laplacian).  Host code: the cores are tiny 0/1 tensors, built once and uploaded through
// qtt_mpo_create.
//
// Construction (App. A): a periodic shift x -> x + s, s = +-1, is a ripple-carry adder
// running from the least-significant site to the most-significant one.  The MPO bond carries the
// "request" still to be served: channel 0 = nothing to add (identity on the site), channel c > 0 = add
// s_c to the bit b_c of this site.  out[w] takes in[w'] with  bit(w') = bit(w) + s (mod 2)  and the
// request travels on to the more significant neighbour iff that addition wrapped.  The periodic
// boundary drops the request that leaves the most-significant site (L = all ones); the stencil
// weights sit on the least-significant end (R).  Index convention W[alpha_m][w (out)][w' (in)][alpha_{m+1}].
#include <vector>

#include "../../include/qtt.h"

namespace {

struct Channel {
  int bit;    // which bit of w is shifted (w = 2 x_bit + y_bit: 1 = x, 0 = y;  w = 4 x_bit + 2 y_bit + z_bit: 2, 1, 0); -1 = identity
  int shift;  // +1: out[i] = in[i+1];  -1: out[i] = in[i-1]
};

// bit of w that belongs to `direction` (1 = x, 2 = y, 3 = z) in a context of physical dimension d; -1 = no such direction
int bit_of(int d, int direction) {
  const int ndim = d == 8 ? 3 : 2;
  return (direction >= 1 && direction <= ndim) ? ndim - direction : -1;
}

// Bulk core for a list of channels (channel 0 must be the identity), D = channels.size(), physical dimension d.
std::vector<double> bulk_core(const std::vector<Channel>& ch, int d) {
  const int D = (int)ch.size();
  std::vector<double> C((size_t)D * d * d * D, 0.0);
  auto at = [&](int am, int w, int wp, int am1) -> double& { return C[(((size_t)am * d + w) * d + wp) * D + am1]; };
  for (int w = 0; w < d; ++w) at(0, w, w, 0) = 1.0;
  for (int c = 1; c < D; ++c) {
    const int mask = 1 << ch[c].bit;
    for (int w = 0; w < d; ++w) {
      const int out_bit = (w & mask) ? 1 : 0;
      const int wp = w ^ mask;  // the shifted bit always flips
      // in = out + 1: wraps when out_bit == 1;  in = out - 1: borrows when out_bit == 0
      const bool onward = (ch[c].shift > 0) ? (out_bit == 1) : (out_bit == 0);
      at(onward ? c : 0, w, wp, c) = 1.0;
    }
  }
  return C;
}

// Folds L = ones into the first core and R = Rvec into the last one, uploads.
qtt_status upload(qtt_ctx* ctx, int n, int D, int d, const std::vector<double>& C, const double* Rvec, qtt_mpo** out) {
  const int dd = d * d;
  // first core: L = ones contracted into alpha_m  -> [1][d][d][D]
  std::vector<double> first((size_t)dd * D, 0.0);
  // last core: R contracted into alpha_{m+1} -> [D][d][d][1]
  std::vector<double> last((size_t)D * dd, 0.0);
  for (int am = 0; am < D; ++am)
    for (int e = 0; e < dd; ++e)
      for (int a1 = 0; a1 < D; ++a1) {
        const double v = C[((size_t)am * dd + e) * D + a1];
        first[(size_t)e * D + a1] += v;
        last[(size_t)am * dd + e] += v * Rvec[a1];
      }
  std::vector<int> bonds(n + 1, D);
  bonds[0] = bonds[n] = 1;
  std::vector<const double*> cores(n, C.data());
  cores[0] = first.data();
  cores[n - 1] = last.data();
  return qtt_mpo_create(ctx, n, bonds.data(), cores.data(), out);
}

qtt_status build(qtt_ctx* ctx, int n, const std::vector<Channel>& ch, const std::vector<double>& Rvec, qtt_mpo** out) {
  if (!ctx || !out || n < 2) return QTT_INVALID_ARG;
  const int d = qtt_ctx_phys_dim(ctx);
  return upload(ctx, n, (int)ch.size(), d, bulk_core(ch, d), Rvec.data(), out);
}

}  // namespace

extern "C" {

qtt_status qtt_mpo_central_difference(qtt_ctx* ctx, int n_sites, int direction, double dx, qtt_mpo** out) {
  if (!ctx) return QTT_INVALID_ARG;
  const int bit = bit_of(qtt_ctx_phys_dim(ctx), direction);
  if (bit < 0) return QTT_INVALID_ARG;
  if (!(dx > 0.0)) return QTT_INVALID_ARG;
  std::vector<Channel> ch{{-1, 0}, {bit, +1}, {bit, -1}};
  std::vector<double> R{0.0, 1.0 / (2.0 * dx), -1.0 / (2.0 * dx)};
  return build(ctx, n_sites, ch, R, out);
}

qtt_status qtt_mpo_stencil(qtt_ctx* ctx, int n_sites, int direction, int half_width, const double* coeffs_host,
                           qtt_mpo** out) {
  if (!ctx || !out || !coeffs_host || n_sites < 2 || half_width < 1 || half_width > 16) return QTT_INVALID_ARG;
  const int d = qtt_ctx_phys_dim(ctx);
  const int pos = bit_of(d, direction);
  if (pos < 0) return QTT_INVALID_ARG;
  // carry automaton of x + k (App. A generalised to |k| <= K): bond index = carry + K
  const int K = half_width, D = 2 * K + 1;
  std::vector<double> C((size_t)D * d * d * D, 0.0);
  for (int cin = -K; cin <= K; ++cin)
    for (int w = 0; w < d; ++w) {
      const int b = (w >> pos) & 1;
      const int s = b + cin;
      const int bin = ((s % 2) + 2) % 2;
      const int cout = (s - bin) / 2;  // exact: s - bin is even
      const int wp = (w & ~(1 << pos)) | (bin << pos);
      C[(((size_t)(cout + K) * d + w) * d + wp) * D + (cin + K)] = 1.0;
    }
  // L = ones on the most-significant end, R = coefficients on the least-significant end
  return upload(ctx, n_sites, D, d, C, coeffs_host, out);
}

qtt_status qtt_mpo_laplacian(qtt_ctx* ctx, int n_sites, double dx, qtt_mpo** out) {
  if (!ctx) return QTT_INVALID_ARG;
  if (!(dx > 0.0)) return QTT_INVALID_ARG;
  const int d = qtt_ctx_phys_dim(ctx);
  const int ndim = d == 8 ? 3 : 2;
  // 2D: channels (x,+1), (x,-1), (y,+1), (y,-1), R = (-4, 1, 1, 1, 1) / dx^2;  3D: two more for z, R = (-6, 1, ...) / dx^2
  std::vector<Channel> ch{{-1, 0}};
  const double h = 1.0 / (dx * dx);
  std::vector<double> R{-2.0 * ndim * h};
  for (int dir = 1; dir <= ndim; ++dir) {
    ch.push_back({ndim - dir, +1});
    ch.push_back({ndim - dir, -1});
    R.push_back(h);
    R.push_back(h);
  }
  return build(ctx, n_sites, ch, R, out);
}

}  // extern "C"
