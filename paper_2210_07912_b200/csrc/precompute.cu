// NEXT-3: the inner products held fixed per intrinsic point, Eq. (D4a-c), from the
// frequency series of the modes and the data (include/rift_ile.h: rift_ile_precompute; reading E1 of DESIGN.md section 13):
//   Q[p,k,a,j] = sum_n w[k,n] exp(2 pi i f[n] t_j) conj(h[p,k,a,n]) d[p,k,n],   t_j = (j - (n_t - 1)/2) delta_t
//   U[p,k,a,b] = sum_n w[k,n] conj(h[p,k,a,n]) h[p,k,b,n],     V[p,k,a,b] = sum_n w[k,n] h[p,k,a,n] h[p,k,b,n]
// Q is a direct transform onto the n_t window times (n_t << number of bins of a full FFT grid, and the bins need not lie on
// one): a thread owns one window time and PQ_COLS (detector, mode) columns; the phase exp(2 pi i f_n t_j) is evaluated
// exactly (sincospi of the reduced argument) at the start of every run of 32 bins and carried across the run by rotations
// when the bins are equally spaced (checked on the host), so one phase serves all columns; X = w conj(h) d is staged in
// shared memory per run.  fp64 throughout.
#include "rift_internal.h"

namespace {

constexpr int PQ_THREADS = 128, PQ_COLS = 8, PQ_RUN = 32;

// exp(2 pi i f t): the argument is reduced in units of full turns so that sincospi sees |x| <= 1/2
__device__ __forceinline__ void phase(double f, double t, double &c, double &s) {
  const double x = f * t;                       // turns
  const double hi = rint(x);
  const double lo = fma(f, t, -hi);             // exact remainder of the product
  sincospi(2.0 * lo, &s, &c);
}

__global__ void __launch_bounds__(PQ_THREADS)
precompute_q_kernel(const double2 *__restrict__ h, const double2 *__restrict__ d, const double *__restrict__ w,
                    const double *__restrict__ f, int K, int M, int64_t n_cols, int n_freq, int n_t, double delta_t,
                    int equal_spacing, double df, double2 *__restrict__ Q) {
  __shared__ double2 xs[PQ_COLS][PQ_RUN];
  __shared__ double fs[PQ_RUN];
  const int64_t col0 = (int64_t)blockIdx.y * PQ_COLS;                       // column = (point * K + k) * M + a
  const int j = blockIdx.x * PQ_THREADS + threadIdx.x;
  const double t = ((double)j - 0.5 * (double)(n_t - 1)) * delta_t;
  double2 acc[PQ_COLS];
#pragma unroll
  for (int c = 0; c < PQ_COLS; ++c) acc[c] = make_double2(0.0, 0.0);
  double rc = 1.0, rs = 0.0;
  if (equal_spacing) phase(df, t, rc, rs);                                  // rotation per bin
  for (int n0 = 0; n0 < n_freq; n0 += PQ_RUN) {
    __syncthreads();
    for (int i = threadIdx.x; i < PQ_COLS * PQ_RUN; i += PQ_THREADS) {
      const int c = i / PQ_RUN, n = n0 + (i % PQ_RUN);
      double2 x = make_double2(0.0, 0.0);
      const int64_t col = col0 + c;
      if (n < n_freq && col < n_cols) {
        const int64_t pk = col / M;                                         // point * K + k
        const int k = (int)(pk % K);
        const double2 hv = h[col * n_freq + n], dv = d[pk * n_freq + n];
        const double wv = w[(int64_t)k * n_freq + n];
        x.x = wv * (hv.x * dv.x + hv.y * dv.y);                             // conj(h) d
        x.y = wv * (hv.x * dv.y - hv.y * dv.x);
      }
      xs[c][i % PQ_RUN] = x;
    }
    if (threadIdx.x < PQ_RUN) fs[threadIdx.x] = n0 + threadIdx.x < n_freq ? f[n0 + threadIdx.x] : 0.0;
    __syncthreads();
    if (j < n_t) {
      double ec, es;
      phase(fs[0], t, ec, es);
#pragma unroll 4
      for (int r = 0; r < PQ_RUN; ++r) {
        if (!equal_spacing && r > 0) phase(fs[r], t, ec, es);
#pragma unroll
        for (int c = 0; c < PQ_COLS; ++c) {
          const double2 x = xs[c][r];
          acc[c].x = fma(ec, x.x, fma(-es, x.y, acc[c].x));
          acc[c].y = fma(ec, x.y, fma(es, x.x, acc[c].y));
        }
        if (equal_spacing) {
          const double nc = ec * rc - es * rs;
          es = ec * rs + es * rc;
          ec = nc;
        }
      }
    }
  }
  if (j < n_t) {
#pragma unroll
    for (int c = 0; c < PQ_COLS; ++c)
      if (col0 + c < n_cols) Q[(col0 + c) * n_t + j] = acc[c];
  }
}

// one block per (point, detector, a, b): U and V entries by a block reduction over the bins
__global__ void __launch_bounds__(128) precompute_uv_kernel(const double2 *__restrict__ h, const double *__restrict__ w, int K,
                                                            int M, int n_freq, double2 *__restrict__ U, double2 *__restrict__ V) {
  const int64_t e = blockIdx.x;                                             // ((pk * M) + a) * M + b
  const int b = (int)(e % M), a = (int)((e / M) % M);
  const int64_t pk = e / ((int64_t)M * M);
  const int k = (int)(pk % K);
  const double2 *ha = h + (pk * M + a) * n_freq, *hb = h + (pk * M + b) * n_freq;
  const double *wk = w + (int64_t)k * n_freq;
  double ur = 0, ui = 0, vr = 0, vi = 0;
  for (int n = threadIdx.x; n < n_freq; n += 128) {
    const double2 x = ha[n], y = hb[n];
    const double wv = wk[n];
    ur += wv * (x.x * y.x + x.y * y.y);                                     // conj(x) y
    ui += wv * (x.x * y.y - x.y * y.x);
    vr += wv * (x.x * y.x - x.y * y.y);                                     // x y
    vi += wv * (x.x * y.y + x.y * y.x);
  }
  __shared__ double red[4][4];
  double v4[4] = {ur, ui, vr, vi};
#pragma unroll
  for (int q = 0; q < 4; ++q) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v4[q] += __shfl_xor_sync(0xffffffffu, v4[q], o);
    if ((threadIdx.x & 31) == 0) red[q][threadIdx.x >> 5] = v4[q];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    U[e] = make_double2(red[0][0] + red[0][1] + red[0][2] + red[0][3], red[1][0] + red[1][1] + red[1][2] + red[1][3]);
    V[e] = make_double2(red[2][0] + red[2][1] + red[2][2] + red[2][3], red[3][0] + red[3][1] + red[3][2] + red[3][3]);
  }
}

}  // namespace

cudaError_t launch_precompute(int32_t P, int32_t K, int32_t M, int32_t n_freq, const void *h, const void *d, const double *w,
                              const double *f, int equal_spacing, double df, int32_t n_t, double delta_t, void *Q, void *U,
                              void *V, cudaStream_t s) {
  const int64_t cols = (int64_t)P * K * M;
  dim3 grid((unsigned)((n_t + PQ_THREADS - 1) / PQ_THREADS), (unsigned)((cols + PQ_COLS - 1) / PQ_COLS));
  precompute_q_kernel<<<grid, PQ_THREADS, 0, s>>>(reinterpret_cast<const double2 *>(h), reinterpret_cast<const double2 *>(d), w, f,
                                                  K, M, cols, n_freq, n_t, delta_t, equal_spacing, df,
                                                  reinterpret_cast<double2 *>(Q));
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  precompute_uv_kernel<<<(unsigned)(cols * M), 128, 0, s>>>(reinterpret_cast<const double2 *>(h), w, K, M, n_freq,
                                                            reinterpret_cast<double2 *>(U), reinterpret_cast<double2 *>(V));
  return cudaGetLastError();
}
