// Two small pieces of SURVEY.md section 8(f) NEXT-4 (include/rift_sky.h, rift_ile_rho_guess in include/rift_ile.h).
//
// 1. Rotated detector-network-frame sky coordinates: the nominal north pole is the vector connecting two
//    interferometers.  Readings F1-F2 of DESIGN.md section 14:
//      n(ra, dec) = (cos dec cos(ra - gmst), cos dec sin(ra - gmst), sin dec)             Earth-fixed direction (as in step a3)
//      z' = (r_b - r_a)/|r_b - r_a|,  x' = (e_z x z')/|e_z x z'| (e_x if the baseline is polar),  y' = z' x x',  R = [x' y' z']
//      n = R (cos beta cos lambda, cos beta sin lambda, sin beta)
//    Elementwise fp64 kernels (sincos, asin, atan2): 32 bytes of traffic per sample, HBM-bound.
// 2. rho_guess, Eq. (D7) with reading A14: (2.3 rho_guess)^2 = sum_k sum_lm max_t |Q_{k,lm}(t)|^2 / |U_{k,lm,lm}|
//    from the handle's device copies of Q and U: one block per intrinsic point, rows in a fixed order (deterministic).
#include <cmath>

#include "rift_internal.h"
#include "rift_sky.h"

namespace {

struct Rot {
  double r[9];   // row-major: r[3 i + j] = R_ij
};

__global__ void network_to_radec_kernel(int64_t n, Rot R, double gmst, const double *__restrict__ lam, const double *__restrict__ beta,
                                        double *__restrict__ ra, double *__restrict__ dec) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double sl, cl, sb, cb;
    sincos(lam[i], &sl, &cl);
    sincos(beta[i], &sb, &cb);
    const double v0 = cb * cl, v1 = cb * sl, v2 = sb;
    const double n0 = R.r[0] * v0 + R.r[1] * v1 + R.r[2] * v2;
    const double n1 = R.r[3] * v0 + R.r[4] * v1 + R.r[5] * v2;
    const double n2 = R.r[6] * v0 + R.r[7] * v1 + R.r[8] * v2;
    dec[i] = asin(fmin(1.0, fmax(-1.0, n2)));
    double a = fmod(atan2(n1, n0) + gmst, 6.283185307179586476925286766559);
    if (a < 0.0) a += 6.283185307179586476925286766559;
    if (a >= 6.283185307179586476925286766559) a = 0.0;
    ra[i] = a;
  }
}

__global__ void radec_to_network_kernel(int64_t n, Rot R, double gmst, const double *__restrict__ ra, const double *__restrict__ dec,
                                        double *__restrict__ lam, double *__restrict__ beta) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double sh, ch, sd, cd;
    sincos(ra[i] - gmst, &sh, &ch);
    sincos(dec[i], &sd, &cd);
    const double n0 = cd * ch, n1 = cd * sh, n2 = sd;
    const double v0 = R.r[0] * n0 + R.r[3] * n1 + R.r[6] * n2;                 // R^T n
    const double v1 = R.r[1] * n0 + R.r[4] * n1 + R.r[7] * n2;
    const double v2 = R.r[2] * n0 + R.r[5] * n1 + R.r[8] * n2;
    beta[i] = asin(fmin(1.0, fmax(-1.0, v2)));
    double a = atan2(v1, v0);
    if (a < 0.0) a += 6.283185307179586476925286766559;
    if (a >= 6.283185307179586476925286766559) a = 0.0;
    lam[i] = a;
  }
}

template <typename C2>
__global__ void __launch_bounds__(256) rho_guess_kernel(const C2 *__restrict__ Q, int64_t point_stride, int n_t, int n_tp, int K, int M,
                                                        const double2 *__restrict__ U, double *__restrict__ out) {
  __shared__ double s_max[8];
  const int p = blockIdx.x;
  const C2 *q = Q + (int64_t)p * point_stride;
  double total = 0.0;
  for (int row = 0; row < K * M; ++row) {
    double mx = 0.0;
    for (int t = threadIdx.x; t < n_t; t += blockDim.x) {
      const C2 v = q[(int64_t)row * n_tp + t];
      const double re = (double)v.x, im = (double)v.y;
      mx = fmax(mx, re * re + im * im);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int w = 1; w < 8; ++w) mx = fmax(mx, s_max[w]);
      const int k = row / M, a = row - k * M;
      const double2 u = U[(((int64_t)p * K + k) * M + a) * M + a];
      const double ua = sqrt(u.x * u.x + u.y * u.y);
      if (ua > 0.0) total += mx / ua;
    }
  }
  if (threadIdx.x == 0) out[p] = sqrt(total) / 2.3;
}

inline int grid_for(int64_t n) {
  int64_t g = (n + 255) / 256;
  if (g > 148 * 8) g = 148 * 8;
  return g < 1 ? 1 : (int)g;
}

}  // namespace

cudaError_t launch_rho_guess(const QStore &q, bool q_fp32, const double *U, int32_t P, int32_t K, int32_t M, double *out,
                             cudaStream_t s) {
  const int64_t csz = q_fp32 ? 8 : 16;
  if (q_fp32)
    rho_guess_kernel<float2><<<P, 256, 0, s>>>(reinterpret_cast<const float2 *>(q.data), q.point_stride_bytes / csz, q.n_t, q.n_tp, K,
                                               M, reinterpret_cast<const double2 *>(U), out);
  else
    rho_guess_kernel<double2><<<P, 256, 0, s>>>(reinterpret_cast<const double2 *>(q.data), q.point_stride_bytes / csz, q.n_t, q.n_tp,
                                                K, M, reinterpret_cast<const double2 *>(U), out);
  return cudaGetLastError();
}

extern "C" int rift_sky_network_frame(const double *loc_a_m, const double *loc_b_m, double *R) {
  if (!loc_a_m || !loc_b_m || !R) return RIFT_EINVAL;
  double z[3], nz = 0.0;
  for (int i = 0; i < 3; ++i) {
    z[i] = loc_b_m[i] - loc_a_m[i];
    nz += z[i] * z[i];
  }
  nz = std::sqrt(nz);
  if (!(nz > 0.0) || !std::isfinite(nz)) return RIFT_EINVAL;
  for (int i = 0; i < 3; ++i) z[i] /= nz;
  double x[3] = {-z[1], z[0], 0.0};                                  // e_z x z'
  double nx = std::sqrt(x[0] * x[0] + x[1] * x[1]);
  if (nx < 1e-12) {
    x[0] = 1.0, x[1] = 0.0, x[2] = 0.0;
    nx = 1.0;
  }
  for (int i = 0; i < 3; ++i) x[i] /= nx;
  const double y[3] = {z[1] * x[2] - z[2] * x[1], z[2] * x[0] - z[0] * x[2], z[0] * x[1] - z[1] * x[0]};   // z' x x'
  for (int i = 0; i < 3; ++i) {
    R[3 * i + 0] = x[i];
    R[3 * i + 1] = y[i];
    R[3 * i + 2] = z[i];
  }
  return RIFT_OK;
}

extern "C" int rift_sky_network_to_radec(int64_t n, const double *R, double gmst_rad, const double *lambda, const double *beta,
                                         double *ra, double *dec, void *cuda_stream) {
  if (n < 0 || !R || (n > 0 && (!lambda || !beta || !ra || !dec))) return RIFT_EINVAL;
  if (n == 0) return RIFT_OK;
  Rot r;
  for (int i = 0; i < 9; ++i) r.r[i] = R[i];
  network_to_radec_kernel<<<grid_for(n), 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(n, r, gmst_rad, lambda, beta, ra, dec);
  return cudaGetLastError() == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}

extern "C" int rift_sky_radec_to_network(int64_t n, const double *R, double gmst_rad, const double *ra, const double *dec,
                                         double *lambda, double *beta, void *cuda_stream) {
  if (n < 0 || !R || (n > 0 && (!lambda || !beta || !ra || !dec))) return RIFT_EINVAL;
  if (n == 0) return RIFT_OK;
  Rot r;
  for (int i = 0; i < 9; ++i) r.r[i] = R[i];
  radec_to_network_kernel<<<grid_for(n), 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(n, r, gmst_rad, ra, dec, lambda, beta);
  return cudaGetLastError() == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}
