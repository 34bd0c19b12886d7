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
// angle (|t| <= 1, t = tan theta).  With D = bb - aa, X = 2 ab and H = sqrt(D^2 + X^2):
//     t = sign(D ab) |X| / (H + |D|)      (= sin 2theta / (1 + cos 2theta)),      c = 1 / sqrt(1 + t^2),      s = c t.
// Orthogonality (c^2 + s^2 = 1 to rounding, what backward stability needs) rests on the ONE full-accuracy reciprocal
// square root that gives c; t itself only has to be a good angle -- an error of 1e-13 in it leaves a residual inner
// product of that relative size, which the quadratically convergent iteration removes in the next sweep -- so H and the
// reciprocal take one Newton step from the hardware seeds.  The Gram entries are first multiplied by an approximate
// 1 / max(aa, bb) (hardware seed, any scale factor would do) so that no square over- or underflows.  Straight-line code:
// two rotations computed back to back interleave in the instruction stream.
__device__ __forceinline__ Rot jacobi_rotation(double aa, double bb, double ab, double tol2, double floor2) {
  Rot r;
  const double m = fmax(aa, bb);
  double rm;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rm) : "d"(m));
  const double a1 = aa * rm, b1 = bb * rm, x1 = ab * rm;
  const double x2 = x1 * x1;
  // pairs already orthogonal to working accuracy, rows in the noise floor, zero / inf / nan norms: skip
  const bool ok = (x2 > tol2 * (a1 * b1)) && (aa > floor2) && (bb > floor2);
  const double d = b1 - a1;
  const double h2 = fma(d, d, 4.0 * x2);
  double rh;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(rh) : "d"(h2));
  rh = rh * fma(-(0.5 * h2 * rh), rh, 1.5);
  const double den = fma(h2, rh, fabs(d));  // H + |D|
  double rd;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rd) : "d"(den));
  rd = fma(rd, fma(-den, rd, 1.0), rd);
  // sign(D ab) 2 |x1| / den
  const double ta = (fabs(x1) + fabs(x1)) * rd;
  const int sgn = (__double2hiint(d) ^ __double2hiint(ab)) & 0x80000000;
  const double t = __hiloint2double(__double2hiint(ta) | sgn, __double2loint(ta));
  const double c = rsqrt_pos(fma(t, t, 1.0));
  const double sn = c * t;
  const bool fin = ok && (sn == sn) && (c == c) && sn != 0.0;
  r.c = c;
  r.s = sn;
  r.t = t;
  r.apply = fin;
  r.big = fin && x2 > 1e-15 * (a1 * b1);
  return r;
}
__device__ __forceinline__ double warp_sum1(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
