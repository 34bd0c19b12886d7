// Device helpers shared by the cluster-resident block Jacobi (jacobi.cu) and the L2-streamed one (sbj.cu).
#pragma once
#include <cuda_runtime.h>

struct Rot {
  double c, s, t;
  bool apply, big;
};
// rotation that orthogonalises two rows with Gram entries (aa, bb, ab):  a' = c a - s b,  b' = s a + c b
__device__ __forceinline__ Rot jacobi_rotation(double aa, double bb, double ab, double tol2, double floor2) {
  Rot r;
  r.c = 1.0; r.s = 0.0; r.t = 0.0;
  r.apply = false; r.big = false;
  const double ab2 = ab * ab, nn = aa * bb;
  if (!(ab2 > tol2 * nn) || !(aa > floor2) || !(bb > floor2)) return r;
  const double d = bb - aa;
  // t = sign(zeta) / (|zeta| + sqrt(1 + zeta^2)),  zeta = d / (2 ab)
  const double t = copysign(2.0, d) * ab / (fabs(d) + sqrt(d * d + 4.0 * ab2));
  if (!(t == t)) return r;
  const double w = 1.0 + t * t;
  double c = rsqrt(w);
  c = c * (1.5 - 0.5 * w * c * c);  // one Newton step: full fp64 accuracy
  r.c = c;
  r.s = c * t;
  r.t = t;
  r.apply = r.s != 0.0;
  r.big = ab2 > 1e-15 * nn;
  return r;
}
__device__ __forceinline__ double warp_sum1(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

