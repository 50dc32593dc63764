// Create-time layout conversion of Q, and the FMA-pipe microbenchmark used as the roofline denominator (H7).
#include "rift_internal.h"

namespace {

// Q rows: [rows][n_t] complex128  ->  [rows][n_tp] complex<float|double>, padding zero-filled.
template <typename CT>
__global__ void convert_q_kernel(const double2 *__restrict__ src, CT *__restrict__ dst, int64_t rows, int n_t, int n_tp) {
  const int64_t total = rows * n_tp;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / n_tp;
    const int t = (int)(i % n_tp);
    CT v;
    v.x = 0;
    v.y = 0;
    if (t < n_t) {
      const double2 s = src[r * n_t + t];
      v.x = s.x;
      v.y = s.y;
    }
    dst[i] = v;
  }
}

// Q rows: [rows][n_t] complex128 -> [rows][n_te] complex<float|double>; columns n_t..n_t+RIFT_EXT-1 repeat columns
// 0..RIFT_EXT-1 circularly, the rest is zero.
template <typename CT>
__global__ void convert_q_ext_kernel(const double2 *__restrict__ src, CT *__restrict__ dst, int64_t rows, int n_t,
                                     int n_te) {
  const int64_t total = rows * n_te;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / n_te;
    const int t = (int)(i % n_te);
    CT v;
    v.x = 0;
    v.y = 0;
    if (t < n_t + RIFT_EXT) {
      const double2 s = src[r * n_t + (t % n_t)];
      v.x = s.x;
      v.y = s.y;
    }
    dst[i] = v;
  }
}

// Q rows: [rows][n_t] complex128 -> planar rows [2*rows][n_tp] Real (2r = Re, 2r+1 = Im); columns n_t..n_t+RIFT_EXT-1
// repeat columns 0..RIFT_EXT-1 circularly, the rest is zero.
template <typename T>
__global__ void convert_q_planar_kernel(const double2 *__restrict__ src, T *__restrict__ dst, int64_t rows, int n_t,
                                        int n_tp) {
  const int64_t total = 2 * rows * n_tp;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r2 = i / n_tp;
    const int t = (int)(i % n_tp);
    T v = 0;
    if (t < n_t + RIFT_EXT) {
      const double2 s = src[(r2 >> 1) * n_t + (t % n_t)];
      v = (T)((r2 & 1) ? s.y : s.x);
    }
    dst[i] = v;
  }
}

template <typename T>
__global__ void __launch_bounds__(256) fma_peak_kernel(int iters, T seed, T *sink) {
  T a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = seed + (T)(threadIdx.x + i);
  const T m = (T)0.999999, c = (T)1e-6;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = fma(a[i], m, c);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i];
  if (s == (T)123.456) sink[0] = s;   // never true; keeps the chain alive
}

// Register-tiled variant: 7 x 8 accumulators, x[i][j] += q[i] * c[j] with every operand in a register (the operand
// pattern of the fused lnL kernels).  mode 1 of run_fma_peak.
__global__ void __launch_bounds__(256) fma_tile_kernel(int iters, const float *__restrict__ src, float *sink) {
  float q[7], c[8], x[7][8];
#pragma unroll
  for (int i = 0; i < 7; ++i) q[i] = src[threadIdx.x + 32 * i];
#pragma unroll
  for (int j = 0; j < 8; ++j) c[j] = src[300 + j];
#pragma unroll
  for (int i = 0; i < 7; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) x[i][j] = 0.f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
      for (int i = 0; i < 7; ++i) x[i][j] = fmaf(q[i], c[j], x[i][j]);
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 7; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) s += x[i][j];
  if (s == 123.456f) sink[0] = s;
}

}  // namespace

cudaError_t launch_convert_q(const double *Q_c128, void *dst, int64_t rows, int32_t n_t, int32_t n_tp, bool to_fp32,
                             cudaStream_t s) {
  const int64_t total = rows * n_tp;
  int grid = (int)((total + 255) / 256);
  if (grid > 148 * 16) grid = 148 * 16;
  if (grid < 1) grid = 1;
  if (to_fp32)
    convert_q_kernel<float2><<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                  reinterpret_cast<float2 *>(dst), rows, n_t, n_tp);
  else
    convert_q_kernel<double2><<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                   reinterpret_cast<double2 *>(dst), rows, n_t, n_tp);
  return cudaGetLastError();
}

cudaError_t launch_convert_q_ext(const double *Q_c128, void *dst, int64_t rows, int32_t n_t, int32_t n_te, bool to_fp32,
                                 cudaStream_t s) {
  const int64_t total = rows * n_te;
  int grid = (int)((total + 255) / 256);
  if (grid > 148 * 16) grid = 148 * 16;
  if (grid < 1) grid = 1;
  if (to_fp32)
    convert_q_ext_kernel<float2><<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                      reinterpret_cast<float2 *>(dst), rows, n_t, n_te);
  else
    convert_q_ext_kernel<double2><<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                       reinterpret_cast<double2 *>(dst), rows, n_t, n_te);
  return cudaGetLastError();
}

cudaError_t launch_convert_q_planar(const double *Q_c128, void *dst, int64_t rows, int32_t n_t, int32_t n_tp,
                                    bool to_fp32, cudaStream_t s) {
  const int64_t total = 2 * rows * n_tp;
  int grid = (int)((total + 255) / 256);
  if (grid > 148 * 16) grid = 148 * 16;
  if (grid < 1) grid = 1;
  if (to_fp32)
    convert_q_planar_kernel<float><<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                        reinterpret_cast<float *>(dst), rows, n_t, n_tp);
  else
    convert_q_planar_kernel<double><<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                         reinterpret_cast<double *>(dst), rows, n_t, n_tp);
  return cudaGetLastError();
}

cudaError_t run_fma_peak(int mode, int iters, double *tflops, cudaStream_t s) {
  const bool fp64 = mode == 1;
  int dev = 0, n_sm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  void *sink = nullptr;
  void *src = nullptr;
  cudaError_t e = cudaMalloc(&sink, 64);
  if (e != cudaSuccess) return e;
  e = cudaMalloc(&src, 4096);
  if (e != cudaSuccess) return e;
  cudaMemsetAsync(src, 0, 4096, s);
  cudaEvent_t t0, t1;
  cudaEventCreate(&t0);
  cudaEventCreate(&t1);
  const int grid = n_sm * 8, threads = 256;
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(t0, s);
    if (mode == 2)
      fma_tile_kernel<<<grid, threads, 0, s>>>(iters, reinterpret_cast<const float *>(src), reinterpret_cast<float *>(sink));
    else if (fp64)
      fma_peak_kernel<double><<<grid, threads, 0, s>>>(iters, 1.0, reinterpret_cast<double *>(sink));
    else
      fma_peak_kernel<float><<<grid, threads, 0, s>>>(iters, 1.0f, reinterpret_cast<float *>(sink));
    cudaEventRecord(t1, s);
    e = cudaEventSynchronize(t1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(t0);
  cudaEventDestroy(t1);
  cudaFree(sink);
  cudaFree(src);
  if (e != cudaSuccess) return e;
  *tflops = 2.0 * (mode == 2 ? 56.0 : 8.0) * (double)iters * grid * threads / (best * 1e-3) / 1e12;
  return cudaGetLastError();
}
