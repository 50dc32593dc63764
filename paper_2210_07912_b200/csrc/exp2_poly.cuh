// fp64 exponential of the fused kernels' time marginal (lnl_mma.cu, the distance-marginalised lnl_direct variant).
#pragma once
#include <cuda_runtime.h>

// 2^y for y <~ 0 (NaN propagates): y = n + r, |r| <= 1/2, 2^r by a degree-8 polynomial (interpolation at Chebyshev nodes,
// relative error 1.1e-12), 2^n through the exponent field (n clamped at -1000: 2^-1000 stands in for smaller terms).
// 12 FP64-pipe operations with the argument FMA of the caller; the coefficients are constant-bank operands.
static __constant__ double RIFT_EXP2_C[9] = {1.0,
                                             0x1.62e42fef84cf0p-1,
                                             0x1.ebfbdff823cedp-3,
                                             0x1.c6b08dd6fd239p-5,
                                             0x1.3b2ab7181b784p-7,
                                             0x1.5d8745a727ee4p-10,
                                             0x1.4308ac85a5afep-13,
                                             0x1.00dc4a5363675p-16,
                                             0x1.63d1363b4014fp-20};
__device__ __forceinline__ double poly_exp2(double y) {
  const double t = y + 6755399441055744.0;                       // 1.5 * 2^52: the low word of t holds rint(y)
  const int n = max(__double2loint(t), -1000);
  const double r = y - (t - 6755399441055744.0);
  double p = RIFT_EXP2_C[8];
#pragma unroll
  for (int i = 7; i >= 0; --i) p = fma(p, r, RIFT_EXP2_C[i]);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}
