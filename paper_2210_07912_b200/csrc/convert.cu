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


// FP64 tensor-core (DMMA) microbenchmarks: `mma.sync.aligned.m8n8k4.f64` and the larger sm_90+ shapes m16n8k8 / m16n8k16,
// NACC independent accumulator tiles per warp, all operands in registers.  modes 3, 4, 5 of run_fma_peak; mode 6 interleaves
// m8n8k4 with as many independent DFMA per thread (do the two share a pipe?).
__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ void dmma1688(double (&d)[4], const double (&a)[4], const double (&b)[2]) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+d"(d[0]), "+d"(d[1]), "+d"(d[2]), "+d"(d[3])
               : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(b[0]), "d"(b[1]));
}
__device__ __forceinline__ void dmma16816(double (&d)[4], const double (&a)[8], const double (&b)[4]) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, {%12,%13,%14,%15}, {%0,%1,%2,%3};"
               : "+d"(d[0]), "+d"(d[1]), "+d"(d[2]), "+d"(d[3])
               : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(a[4]), "d"(a[5]), "d"(a[6]), "d"(a[7]), "d"(b[0]), "d"(b[1]),
                 "d"(b[2]), "d"(b[3]));
}

// legacy tensor-core path (HMMA): mma.sync m16n8k16, fp16 operands, fp32 accumulate; mode 7 of run_fma_peak
__global__ void __launch_bounds__(256) hmma_peak_kernel(int iters, const uint32_t *__restrict__ src, float *sink) {
  uint32_t a[4], b[2];
#pragma unroll
  for (int i = 0; i < 4; ++i) a[i] = src[threadIdx.x + 32 * i];
  b[0] = src[300 + threadIdx.x];
  b[1] = src[400 + threadIdx.x];
  float d[8][4];
#pragma unroll
  for (int t = 0; t < 8; ++t) d[t][0] = d[t][1] = d[t][2] = d[t][3] = 0.f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int t = 0; t < 8; ++t)
      asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                   : "+f"(d[t][0]), "+f"(d[t][1]), "+f"(d[t][2]), "+f"(d[t][3])
                   : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
  }
  float s = 0;
#pragma unroll
  for (int t = 0; t < 8; ++t) s += d[t][0] + d[t][1] + d[t][2] + d[t][3];
  if (s == 123.456f) sink[0] = s;
}

template <int MODE>
__global__ void __launch_bounds__(256) dmma_peak_kernel(int iters, const double *__restrict__ src, double *sink) {
  constexpr int NACC = 8;
  double a[8], b[4];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = src[threadIdx.x + 32 * i];
#pragma unroll
  for (int i = 0; i < 4; ++i) b[i] = src[300 + threadIdx.x + 32 * i];
  double s = 0;
  if (MODE == 3 || MODE == 6) {
    double d[NACC][2], f[NACC];
#pragma unroll
    for (int t = 0; t < NACC; ++t) d[t][0] = d[t][1] = 0.0, f[t] = a[t & 7];
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int t = 0; t < NACC; ++t) {
        dmma884(d[t], a[t & 7], b[t & 3]);
        if (MODE == 6) f[t] = fma(f[t], 0.999999, 1e-6);
      }
    }
#pragma unroll
    for (int t = 0; t < NACC; ++t) s += d[t][0] + d[t][1] + (MODE == 6 ? f[t] : 0.0);
  } else {
    double d[NACC][4];
#pragma unroll
    for (int t = 0; t < NACC; ++t) d[t][0] = d[t][1] = d[t][2] = d[t][3] = 0.0;
    const double a4[4] = {a[0], a[1], a[2], a[3]}, b2[2] = {b[0], b[1]};
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int t = 0; t < NACC; ++t) {
        if (MODE == 4) dmma1688(d[t], a4, b2);
        else dmma16816(d[t], a, b);
      }
    }
#pragma unroll
    for (int t = 0; t < NACC; ++t) s += d[t][0] + d[t][1] + d[t][2] + d[t][3];
  }
  if (s == 123.456) sink[0] = s;
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

__global__ void fill_f64_kernel(double *dst, int64_t n, double value) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) dst[i] = value;
}
cudaError_t launch_fill_f64(double *dst, int64_t n, double value, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  int grid = (int)((n + 255) / 256);
  if (grid > 148 * 8) grid = 148 * 8;
  fill_f64_kernel<<<grid, 256, 0, s>>>(dst, n, value);
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
  e = cudaMalloc(&src, 8192);
  if (e != cudaSuccess) return e;
  cudaMemsetAsync(src, 0, 8192, s);
  cudaEvent_t t0, t1;
  cudaEventCreate(&t0);
  cudaEventCreate(&t1);
  const int grid = n_sm * 8, threads = 256;
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(t0, s);
    if (mode == 2)
      fma_tile_kernel<<<grid, threads, 0, s>>>(iters, reinterpret_cast<const float *>(src), reinterpret_cast<float *>(sink));
    else if (mode == 3)
      dmma_peak_kernel<3><<<grid, threads, 0, s>>>(iters, reinterpret_cast<const double *>(src), reinterpret_cast<double *>(sink));
    else if (mode == 4)
      dmma_peak_kernel<4><<<grid, threads, 0, s>>>(iters, reinterpret_cast<const double *>(src), reinterpret_cast<double *>(sink));
    else if (mode == 5)
      dmma_peak_kernel<5><<<grid, threads, 0, s>>>(iters, reinterpret_cast<const double *>(src), reinterpret_cast<double *>(sink));
    else if (mode == 7)
      hmma_peak_kernel<<<grid, threads, 0, s>>>(iters, reinterpret_cast<const uint32_t *>(src), reinterpret_cast<float *>(sink));
    else if (mode == 6)
      dmma_peak_kernel<6><<<grid, threads, 0, s>>>(iters, reinterpret_cast<const double *>(src), reinterpret_cast<double *>(sink));
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
  // flop per thread and iteration: 8 FMA chains; 56 in the register tile; DMMA: 8 tiles x (m n k / 32 lanes) FMA
  //   m8n8k4 8, m16n8k8 32, m16n8k16 64 FMA per lane and tile; mode 6 reports the DMMA part only (+ 8 DFMA ride along)
  const double fma_per_it = mode == 2 ? 56.0 : mode == 3 || mode == 6 ? 64.0 : mode == 4 ? 256.0 : mode == 5 ? 512.0 : mode == 7 ? 8.0 * 64.0 : 8.0;
  *tflops = 2.0 * fma_per_it * (double)iters * grid * threads / (best * 1e-3) / 1e12;
  return cudaGetLastError();
}
