// Device helpers shared by the cluster-resident block Jacobi (jacobi.cu, bj2.cu) and the L2-streamed one (sbj.cu).
#pragma once
#include <cuda_runtime.h>

struct Rot {
  double c, s, t;
  bool apply, big;
};

// 1 / sqrt(x) for a normal, positive x: the hardware seed (MUFU.RSQ64H, ~2^-22) and two Newton steps, without the
// special-case handling of rsqrt() -- the library sqrt / divide / rsqrt sequences were ~150 of the ~470 instructions
// a warp issued per row-pair meeting (profiles/r2_bj2_full.md).
__device__ __forceinline__ double rsqrt_pos(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  y = y * fma(-(h * y), y, 1.5);
  y = y * fma(-(h * y), y, 1.5);
  return y;
}

// Rotation that orthogonalises two rows with Gram entries (aa, bb, ab):  a' = c a - s b,  b' = s a + c b, the small
// angle (|tan| <= 1).  With D = bb - aa and H = sqrt(D^2 + 4 ab^2):  cos 2theta = |D| / H, sin 2theta = 2 |ab| / H,
// c^2 = (1 + cos 2theta) / 2, s = sign(D ab) sin 2theta / (2 c), t = s / c.  Only two reciprocal square roots, no
// divide; the operands are first scaled by a power of two so that the fourth powers of the row norms neither
// overflow nor underflow.  c^2 + s^2 = 1 to rounding (what backward stability needs); the angle itself is accurate
// to a few ulps.
__device__ __forceinline__ Rot jacobi_rotation(double aa, double bb, double ab, double tol2, double floor2) {
  // straight-line code (no early exit): two rotations computed back to back interleave in the instruction stream
  Rot r;
  const double ab2 = ab * ab, nn = aa * bb;
  // power-of-two scale 2^-e, e = exponent of max(aa, bb): exact, keeps D^2 + 4 ab^2 in range
  const double m = fmax(aa, bb);
  const int hi = __double2hiint(m) & 0x7ff00000;
  // pairs already orthogonal to working accuracy, rows in the noise floor, subnormal / huge / inf / nan norms: skip
  const bool ok = (ab2 > tol2 * nn) && (aa > floor2) && (bb > floor2) && hi != 0 && hi < 0x7fe00000;
  const double sc = __hiloint2double(0x7fe00000 - hi, 0);
  const double a1 = aa * sc, b1 = bb * sc, x1 = ab * sc;
  const double d = b1 - a1;
  const double h2 = fma(d, d, 4.0 * x1 * x1);
  const double rh = rsqrt_pos(h2);
  const double cos2 = fabs(d) * rh, sin2 = 2.0 * fabs(x1) * rh;
  const double c2 = fma(0.5, cos2, 0.5);  // in [1/2, 1]
  const double rc = rsqrt_pos(c2);
  const double sg = copysign(0.5, d) * copysign(1.0, ab);
  const double hs = sg * sin2 * rc;  // s = sin 2theta / (2 c)
  const double c = c2 * rc;
  const bool fin = ok && (c == c) && (hs == hs) && hs != 0.0;
  r.c = fin ? c : 1.0;
  r.s = fin ? hs : 0.0;
  r.t = fin ? hs * rc : 0.0;
  r.apply = fin;
  r.big = fin && ab2 > 1e-15 * nn;
  return r;
}
__device__ __forceinline__ double warp_sum1(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
