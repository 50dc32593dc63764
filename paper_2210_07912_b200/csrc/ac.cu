// On-device adaptive-cartesian (AC) sampler, include/rift_ac.h (arXiv 2210.07912 section IV.C.2, Eq. (22)).
// The draw is one thread per sample: a counter-based random number per dimension, inverse CDF by binary search over the bin
// table staged in shared memory, position uniform inside the bin.  The histogram refresh is host-side (n_dim x n_bins
// numbers per round, the "minimal data transfer as needed to orchestrate the integration" of :352).
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "rift_ac.h"
#include "rift_ile.h"

#include <cuda_runtime.h>

struct rift_ac {
  int device = 0;
  int n_dim = 0, n_bins = 0;
  std::vector<double> lo, hi, masses;      // host copies
  double *d_tab = nullptr;                 // device: [n_dim][n_bins] masses, then [n_dim][n_bins] cdf, then lo[n_dim], hi[n_dim]
  double **d_xptr = nullptr;               // device array of n_dim output pointers
};

namespace {

constexpr int AC_THREADS = 256;
constexpr int AC_MAX_DIM = 16;

__device__ __forceinline__ double ac_u01(uint64_t seed, uint64_t index) {
  uint64_t z = seed + (index + 1ull) * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z = z ^ (z >> 31);
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}

__global__ void __launch_bounds__(AC_THREADS)
ac_draw_kernel(int n_dim, int n_bins, const double *__restrict__ tab, double *const *__restrict__ xptr,
               double *__restrict__ ln_ps, int64_t n, uint64_t seed, uint64_t offset) {
  extern __shared__ double sh[];           // masses, cdf, lo, hi
  const int n_tab = 2 * n_dim * n_bins + 2 * n_dim;
  for (int i = threadIdx.x; i < n_tab; i += AC_THREADS) sh[i] = tab[i];
  __syncthreads();
  const double *mass = sh, *cdf = sh + n_dim * n_bins, *lo = sh + 2 * n_dim * n_bins, *hi = lo + n_dim;
  const int64_t i = (int64_t)blockIdx.x * AC_THREADS + threadIdx.x;
  if (i >= n) return;
  double lp = 0.0;
  for (int d = 0; d < n_dim; ++d) {
    const double u = ac_u01(seed, (offset + (uint64_t)i) * (uint64_t)n_dim + (uint64_t)d);
    const double *c = cdf + d * n_bins;
    int a = 0, b = n_bins - 1;             // last bin with cdf[bin] <= u (cdf[0] = 0 <= u always)
    while (a < b) {
      const int m = (a + b + 1) >> 1;
      if (c[m] <= u) a = m; else b = m - 1;
    }
    // the masses sum to 1 only up to rounding: a draw past the last positive-mass bin (or into a bin emptied by floor = 0)
    // steps back to the nearest bin that can be drawn, so that ln p_s stays finite
    while (a > 0 && !(mass[d * n_bins + a] > 0.0)) --a;
    const double ms = mass[d * n_bins + a];
    const double w = __ddiv_rn(__dsub_rn(hi[d], lo[d]), (double)n_bins);
    double frac = __ddiv_rn(__dsub_rn(u, c[a]), ms);
    frac = fmin(frac, 0.99999999999999989);                                 // nextafter(1, 0): stay inside the bin
    xptr[d][i] = __dadd_rn(__dmul_rn(__dadd_rn((double)a, frac), w), lo[d]);
    lp += log(__ddiv_rn(ms, w));
  }
  ln_ps[i] = lp;
}

struct Params6 {
  const double *p[6];
};

__global__ void __launch_bounds__(AC_THREADS)
ac_ile_ln_weight_kernel(int64_t n, Params6 P, double d_min, double d_max, const double *__restrict__ ln_ps,
                        double *__restrict__ ln_w) {
  const int64_t i = (int64_t)blockIdx.x * AC_THREADS + threadIdx.x;
  if (i >= n) return;
  const double ra = P.p[0][i], dec = P.p[1][i], psi = P.p[2][i], iota = P.p[3][i], phi = P.p[4][i], dist = P.p[5][i];
  const double pi = 3.14159265358979323846, two_pi = 2.0 * pi;
  const bool ok = ra >= 0.0 && ra < two_pi && fabs(dec) <= 0.5 * pi && psi >= 0.0 && psi < pi && iota >= 0.0 && iota <= pi &&
                  phi >= 0.0 && phi < two_pi && dist >= d_min && dist <= d_max;
  double lp = -log(two_pi) + log(cos(dec) / 2.0) - log(pi) + log(sin(iota) / 2.0) - log(two_pi) +
              log(3.0 * dist * dist / (d_max * d_max * d_max - d_min * d_min * d_min));
  if (!ok || !isfinite(lp)) lp = -INFINITY;
  ln_w[i] = lp - ln_ps[i];
}

int upload(rift_ac *h) {
  const int nd = h->n_dim, nb = h->n_bins;
  std::vector<double> tab((size_t)2 * nd * nb + 2 * nd);
  for (int d = 0; d < nd; ++d) {
    double acc = 0.0;                      // cdf accumulated left to right, as the oracle does
    for (int b = 0; b < nb; ++b) {
      tab[(size_t)d * nb + b] = h->masses[(size_t)d * nb + b];
      tab[(size_t)nd * nb + (size_t)d * nb + b] = acc;
      acc = acc + h->masses[(size_t)d * nb + b];
    }
    tab[(size_t)2 * nd * nb + d] = h->lo[d];
    tab[(size_t)2 * nd * nb + nd + d] = h->hi[d];
  }
  return cudaMemcpy(h->d_tab, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice) == cudaSuccess ? RIFT_OK
                                                                                                                : RIFT_ECUDA;
}

}  // namespace

extern "C" {

int rift_ac_create(int32_t n_dim, int32_t n_bins, const double *lo, const double *hi, rift_ac_t **out) {
  if (!out || !lo || !hi || n_dim < 1 || n_dim > AC_MAX_DIM || n_bins < 1 || n_bins > 1024) return RIFT_EINVAL;
  if (((size_t)2 * n_dim * n_bins + 2 * n_dim) * sizeof(double) > 200u * 1024u) return RIFT_EINVAL;   // the draw kernel's table
  for (int d = 0; d < n_dim; ++d)
    if (!(hi[d] > lo[d]) || !std::isfinite(lo[d]) || !std::isfinite(hi[d])) return RIFT_EINVAL;
  rift_ac *h = new (std::nothrow) rift_ac();
  if (!h) return RIFT_ENOMEM;
  h->n_dim = n_dim;
  h->n_bins = n_bins;
  h->lo.assign(lo, lo + n_dim);
  h->hi.assign(hi, hi + n_dim);
  h->masses.assign((size_t)n_dim * n_bins, 1.0 / n_bins);
  const size_t tab_bytes = ((size_t)2 * n_dim * n_bins + 2 * n_dim) * sizeof(double);
  if (cudaGetDevice(&h->device) != cudaSuccess || cudaMalloc(&h->d_tab, tab_bytes) != cudaSuccess ||
      cudaMalloc(&h->d_xptr, sizeof(double *) * n_dim) != cudaSuccess || upload(h) != RIFT_OK) {
    cudaGetLastError();
    cudaFree(h->d_tab);
    cudaFree(h->d_xptr);
    delete h;
    return RIFT_ECUDA;
  }
  *out = h;
  return RIFT_OK;
}

int rift_ac_draw(rift_ac_t *h, int64_t n, uint64_t seed, uint64_t offset, double *const *x, double *ln_ps,
                 void *cuda_stream) {
  if (!h || n < 0) return RIFT_EINVAL;
  if (n == 0) return RIFT_OK;
  if (!x || !ln_ps) return RIFT_EINVAL;
  for (int d = 0; d < h->n_dim; ++d)
    if (!x[d]) return RIFT_EINVAL;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (cudaMemcpyAsync(h->d_xptr, x, sizeof(double *) * h->n_dim, cudaMemcpyHostToDevice, s) != cudaSuccess) return RIFT_ECUDA;
  const size_t smem = ((size_t)2 * h->n_dim * h->n_bins + 2 * h->n_dim) * sizeof(double);
  if (smem > 48u * 1024u &&
      cudaFuncSetAttribute(ac_draw_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RIFT_ECUDA;
  ac_draw_kernel<<<(unsigned)((n + AC_THREADS - 1) / AC_THREADS), AC_THREADS, smem, s>>>(h->n_dim, h->n_bins, h->d_tab,
                                                                                        h->d_xptr, ln_ps, n, seed, offset);
  return cudaGetLastError() == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}

int rift_ac_update(rift_ac_t *h, const double *hist, double floor_mix, double temper) {
  return rift_ac_update_dims(h, hist, floor_mix, temper, nullptr);
}

int rift_ac_update_dims(rift_ac_t *h, const double *hist, double floor_mix, double temper, const int32_t *adapt) {
  if (!h || !hist || !(floor_mix >= 0.0 && floor_mix <= 1.0) || !(temper > 0.0)) return RIFT_EINVAL;
  const int nd = h->n_dim, nb = h->n_bins;
  std::vector<double> t(nb);
  for (int d = 0; d < nd; ++d) {
    if (adapt && !adapt[d]) continue;        // frozen dimension: keeps its masses
    double s = 0.0;
    for (int b = 0; b < nb; ++b) {
      const double v = hist[(size_t)d * nb + b];
      t[b] = std::pow(v > 0.0 ? v : 0.0, temper);
      s = s + t[b];
    }
    for (int b = 0; b < nb; ++b)
      h->masses[(size_t)d * nb + b] = (s > 0.0 && std::isfinite(s)) ? (1.0 - floor_mix) * (t[b] / s) + floor_mix / nb : 1.0 / nb;
  }
  // masses of exactly zero (floor_mix = 0) would make a bin undrawable but also divide by zero if rounding selects it
  for (double &m : h->masses)
    if (!(m > 0.0)) m = 0.0;
  return upload(h);
}

int rift_ac_get_masses(const rift_ac_t *h, double *masses) {
  if (!h || !masses) return RIFT_EINVAL;
  memcpy(masses, h->masses.data(), h->masses.size() * sizeof(double));
  return RIFT_OK;
}

int rift_ac_ile_ln_weight(int64_t n, const double *const params[6], double d_min_mpc, double d_max_mpc, const double *ln_ps,
                          double *ln_weight, void *cuda_stream) {
  if (n < 0 || !(d_max_mpc > d_min_mpc) || !(d_min_mpc > 0.0)) return RIFT_EINVAL;
  if (n == 0) return RIFT_OK;
  if (!params || !ln_ps || !ln_weight) return RIFT_EINVAL;
  Params6 P;
  for (int d = 0; d < 6; ++d) {
    if (!params[d]) return RIFT_EINVAL;
    P.p[d] = params[d];
  }
  ac_ile_ln_weight_kernel<<<(unsigned)((n + AC_THREADS - 1) / AC_THREADS), AC_THREADS, 0,
                            reinterpret_cast<cudaStream_t>(cuda_stream)>>>(n, P, d_min_mpc, d_max_mpc, ln_ps, ln_weight);
  return cudaGetLastError() == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}

int rift_ac_destroy(rift_ac_t *h) {
  if (!h) return RIFT_EINVAL;
  cudaFree(h->d_tab);
  cudaFree(h->d_xptr);
  delete h;
  return RIFT_OK;
}

}  // extern "C"
