// Gaussian-mixture adaptive sampler (include/rift_gmm.h): PAPER.md section IV.C.1 (:315-334)
// and Appendix A (:562-625), readings G1-G6 of DESIGN.md section 14.
//
// Device work (per sample, embarrassingly parallel, HBM-bound at 8 (n_dim + 1) bytes per sample and pass):
//   gmm_max_kernel     max of the log-weights (block partials; gmm_maxfin_kernel takes their maximum into the fit's state)
//   gmm_ess_kernel     sum w^t, sum w^2t of reading G7; gmm_ess_step_kernel: one bisection step on the device
//   gmm_em_kernel      one E-step fused with the sums of the M-step: r_nk = N_k pi_k / sum_j N_j pi_j by log-sum-exp, then per
//                      component sum w r, sum w r (x - mu_old), sum w r (x - mu_old)(x - mu_old)^T, plus sum w ln P and sum w,
//                      in registers, reduced by warp shuffles and shared memory to one partial row per block; the model is read
//                      from the fit's device-resident state (EmState)
//   gmm_sum_kernel     the partial rows added in a fixed order (deterministic)
//   gmm_mstep_kernel   Eq. (A4)-(A6), the convergence test and the validity checks, one thread (<= 8 components): the next
//                      E-step's model is written to the device state, no host round trip inside an iteration
//   gmm_draw_kernel    Eq. (A12)-(A13): component by inverse CDF of pi, box proposal z_j = Phi^-1(Phi(a_j) + u (Phi(b_j) -
//                      Phi(a_j))), x = mu + A z, retried until x lies in the domain; ln p_s of the accepted point
//   gmm_density_kernel ln p_s(x) = ln sum_k pi_k N_k(x) / Z_k
// Host work (n_comp <= 8 numbers of each kind, once per fit / model change): the 2 x 2 eigen-decomposition, the proposal boxes,
// the component masses Z_k (Gauss-Legendre), the permutation search of Eq. (A8) and the merge of Eq. (A9)-(A11).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

#include "rift_internal.h"
#include "rift_gmm.h"

namespace {

constexpr int GM_MAXK = RIFT_GMM_MAX_COMP;
constexpr int GM_TRIES = RIFT_GMM_MAX_TRIES;
constexpr int GM_THREADS = 256;
constexpr int GM_BLOCKS = 296;                     // 2 per SM
constexpr int GM_ROW = GM_MAXK * 6 + 2;            // per component: s0, s1[2], s2[3]; then sum w ln P, sum w

struct GmmDev {                                    // kernel parameter (about 1.3 KB)
  int d, K;
  double lo[2], hi[2];
  double mu[GM_MAXK][2];
  double prec[GM_MAXK][3];                         // Sigma^-1: xx, xy, yy
  double lnc[GM_MAXK];                             // ln pi - (1/2) ln det Sigma - (d/2) ln 2 pi   (-inf for pi = 0)
  double lnz[GM_MAXK];                             // ln Z_k
  double A[GM_MAXK][4];                            // row-major [i][j]: x_i = mu_i + sum_j A_ij z_j
  double pa[GM_MAXK][2], pw[GM_MAXK][2];           // Phi(a_j), Phi(b_j) - Phi(a_j) of the proposal box
  double cum[GM_MAXK];                             // running sum of pi
};

struct Model {
  double mu[GM_MAXK][2], cov[GM_MAXK][3], pi[GM_MAXK];   // cov: xx, xy, yy
};

inline double Phi(double t) { return 0.5 * std::erfc(-t * 0.70710678118654752440); }

// G4: A = phi lambda^(1/2), eigenvalues ascending, eigenvectors signed so that the component of largest magnitude is positive
void transform2(const double c[3], double A[4]) {
  const double a = c[0], b = c[1], cc = c[2];
  double l0, l1, v1x, v1y;
  if (b == 0.0) {
    if (a <= cc) {
      l0 = a, l1 = cc, v1x = 0.0, v1y = 1.0;
    } else {
      l0 = cc, l1 = a, v1x = 1.0, v1y = 0.0;
    }
  } else {
    const double h = 0.5 * (a - cc), r = std::hypot(h, b);
    l1 = 0.5 * (a + cc) + r;
    l0 = (a * cc - b * b) / l1;
    if (h >= 0.0) {
      v1x = h + r, v1y = b;
    } else {
      v1x = b, v1y = r - h;
    }
    const double nv = std::hypot(v1x, v1y);
    v1x /= nv, v1y /= nv;
  }
  double v0x = -v1y, v0y = v1x;
  auto fix = [](double &x, double &y) {
    const double m = std::fmax(std::fabs(x), std::fabs(y)) * (1.0 - 1e-12);
    const double lead = std::fabs(x) > m ? x : y;
    if (lead < 0.0) x = -x, y = -y;
  };
  fix(v0x, v0y);
  fix(v1x, v1y);
  const double s0 = std::sqrt(l0), s1 = std::sqrt(l1);
  A[0] = v0x * s0, A[1] = v1x * s1;
  A[2] = v0y * s0, A[3] = v1y * s1;
}

const double GL8_X[8] = {-0.9602898564975363, -0.7966664774136267, -0.5255324099163290, -0.1834346424956498,
                         0.1834346424956498,  0.5255324099163290,  0.7966664774136267,  0.9602898564975363};
const double GL8_W[8] = {0.1012285362903763, 0.2223810344533745, 0.3137066458778873, 0.3626837833783620,
                         0.3626837833783620, 0.3137066458778873, 0.2223810344533745, 0.1012285362903763};

// Z = integral of N(x | mu, cov) over the domain.  d = 2: the integral over x_2 is a difference of two normal CDFs at the
// conditional mean m(x_1) and deviation sc; the integral over x_1 is cut at the two kinks (m(x_1) = lo_2, hi_2) and each piece
// takes 512 panels of 8-point Gauss-Legendre
double box_mass(int d, const double mu[2], const double c[3], const double lo[2], const double hi[2]) {
  const double s0 = std::sqrt(c[0]);
  if (d == 1) return Phi((hi[0] - mu[0]) / s0) - Phi((lo[0] - mu[0]) / s0);
  const double slope = c[1] / c[0], sc = std::sqrt(c[2] - c[1] * c[1] / c[0]);
  const double a = std::fmax(lo[0], mu[0] - 12.0 * s0), b = std::fmin(hi[0], mu[0] + 12.0 * s0);
  if (!(b > a)) return 0.0;
  double cut[4] = {a, b, b, b};
  int nc = 1;
  if (slope != 0.0) {
    double p[2] = {mu[0] + (lo[1] - mu[1]) / slope, mu[0] + (hi[1] - mu[1]) / slope};
    if (p[0] > p[1]) std::swap(p[0], p[1]);
    for (double q : p)
      if (q > cut[nc - 1] && q < b) cut[nc++] = q;
  }
  cut[nc] = b;
  const int panels = 512;
  const double norm = 1.0 / (s0 * 2.50662827463100050242);
  double total = 0.0;
  for (int piece = 0; piece < nc; ++piece) {
    const double w = (cut[piece + 1] - cut[piece]) / panels;
    double acc = 0.0;
    for (int p = 0; p < panels; ++p) {
      const double mid = cut[piece] + (p + 0.5) * w;
      for (int g = 0; g < 8; ++g) {
        const double x1 = mid + 0.5 * w * GL8_X[g], t = (x1 - mu[0]) / s0, m = mu[1] + slope * (x1 - mu[0]);
        acc += GL8_W[g] * std::exp(-0.5 * t * t) * (Phi((hi[1] - m) / sc) - Phi((lo[1] - m) / sc));
      }
    }
    total += acc * 0.5 * w * norm;
  }
  return total;
}

bool model_valid(int d, int K, const Model &m) {
  double sum = 0.0;
  for (int k = 0; k < K; ++k) {
    if (!(m.pi[k] >= 0.0) || !std::isfinite(m.pi[k])) return false;
    sum += m.pi[k];
    for (int j = 0; j < d; ++j)
      if (!std::isfinite(m.mu[k][j])) return false;
    if (!(m.cov[k][0] > 0.0) || !std::isfinite(m.cov[k][0])) return false;
    if (d == 2) {
      const double det = m.cov[k][0] * m.cov[k][2] - m.cov[k][1] * m.cov[k][1];
      if (!(m.cov[k][2] > 0.0) || !(det > 0.0) || !std::isfinite(det)) return false;
    }
  }
  return std::fabs(sum - 1.0) < 1e-9;
}

// Everything the kernels need from a model.  with_boxes = false skips the proposal boxes and the masses (the EM kernel reads
// neither)
void derive(int d, int K, const double lo[2], const double hi[2], const Model &m, bool with_boxes, GmmDev &g) {
  std::memset(&g, 0, sizeof(g));
  g.d = d, g.K = K;
  for (int j = 0; j < 2; ++j) g.lo[j] = lo[j], g.hi[j] = hi[j];
  double run = 0.0;
  for (int k = 0; k < K; ++k) {
    g.mu[k][0] = m.mu[k][0], g.mu[k][1] = m.mu[k][1];
    const double a = m.cov[k][0], b = d == 2 ? m.cov[k][1] : 0.0, c = d == 2 ? m.cov[k][2] : 1.0;
    const double det = a * c - b * b;
    g.prec[k][0] = c / det, g.prec[k][1] = -b / det, g.prec[k][2] = a / det;
    g.lnc[k] = (m.pi[k] > 0.0 ? std::log(m.pi[k]) : -INFINITY) - 0.5 * std::log(det) - 0.5 * d * 1.8378770664093454836;
    run += m.pi[k];
    g.cum[k] = run;
    if (!with_boxes) continue;
    if (d == 1) {
      g.A[k][0] = std::sqrt(a);
    } else {
      const double cv[3] = {a, b, c};
      transform2(cv, g.A[k]);
    }
    // Eq. (A13): r = A^-1, bounding box of r (corner - mu)
    double zl[2] = {INFINITY, INFINITY}, zh[2] = {-INFINITY, -INFINITY};
    if (d == 1) {
      zl[0] = (lo[0] - m.mu[k][0]) / g.A[k][0], zh[0] = (hi[0] - m.mu[k][0]) / g.A[k][0];
    } else {
      const double dA = g.A[k][0] * g.A[k][3] - g.A[k][1] * g.A[k][2];
      const double r00 = g.A[k][3] / dA, r01 = -g.A[k][1] / dA, r10 = -g.A[k][2] / dA, r11 = g.A[k][0] / dA;
      for (int cnr = 0; cnr < 4; ++cnr) {
        const double cx = ((cnr & 1) ? hi[0] : lo[0]) - m.mu[k][0], cy = ((cnr & 2) ? hi[1] : lo[1]) - m.mu[k][1];
        const double t0 = r00 * cx + r01 * cy, t1 = r10 * cx + r11 * cy;
        zl[0] = std::fmin(zl[0], t0), zh[0] = std::fmax(zh[0], t0);
        zl[1] = std::fmin(zl[1], t1), zh[1] = std::fmax(zh[1], t1);
      }
    }
    for (int j = 0; j < d; ++j) {
      g.pa[k][j] = Phi(zl[j]);
      g.pw[k][j] = Phi(zh[j]) - g.pa[k][j];
    }
    const double cv[3] = {a, b, c};
    const double Z = box_mass(d, m.mu[k], cv, lo, hi);
    g.lnz[k] = Z > 0.0 ? std::log(Z) : -INFINITY;
  }
}

}  // namespace

struct rift_gmm {
  int device = 0, d = 0, K = 0;
  double lo[2] = {0, 0}, hi[2] = {1, 1};
  Model model{};
  double n_trained = 0.0;
  GmmDev dev{};                                    // derived from `model` (boxes included) when dev_ok
  bool dev_ok = false;
  double *d_partial = nullptr;                     // [GM_BLOCKS][GM_ROW]
  double *d_sums = nullptr;                        // [GM_ROW]
  void *d_em = nullptr;                            // EmState of a running fit
  unsigned long long *d_fail = nullptr;
};

namespace {

__device__ __forceinline__ double gm_u01(uint64_t seed, uint64_t c) {            // G6
  uint64_t z = seed + (c + 1ull) * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z ^= z >> 31;
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}

// ln(N_k(x) pi_k) for every component, their log-sum-exp in `lse`; `extra[k]` is subtracted (ln Z_k for the density, 0 for EM)
template <bool WITH_Z>
__device__ __forceinline__ double gm_log_terms(const GmmDev &g, double x0, double x1, double (&lp)[GM_MAXK]) {
  double m = -INFINITY;
#pragma unroll
  for (int k = 0; k < GM_MAXK; ++k) {
    lp[k] = -INFINITY;
    if (k < g.K) {
      const double d0 = x0 - g.mu[k][0], d1 = g.d == 2 ? x1 - g.mu[k][1] : 0.0;
      const double q = g.prec[k][0] * d0 * d0 + 2.0 * g.prec[k][1] * d0 * d1 + (g.d == 2 ? g.prec[k][2] * d1 * d1 : 0.0);
      lp[k] = g.lnc[k] - 0.5 * q - (WITH_Z ? g.lnz[k] : 0.0);
      m = fmax(m, lp[k]);
    }
  }
  if (!(m > -INFINITY)) return -INFINITY;
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < GM_MAXK; ++k)
    if (k < g.K) s += exp(lp[k] - m);
  return m + log(s);
}

// The model of a running EM fit, kept on the device across iterations (no host round trip per iteration)
struct EmState {
  double mu[GM_MAXK][2], cov[GM_MAXK][3], pi[GM_MAXK];   // Eq. (A4)-(A6) of the last M-step
  double prec[GM_MAXK][3], lnc[GM_MAXK];                 // what the next E-step reads
  double ll, prev;                                       // ln L of the last E-step, and of the one before the last M-step
  int it, done, bad;                                     // M-steps done; converged / stopped; an empty component or a bad covariance
  double w_max, temper;                                  // maximum of the log-weights; the exponent of reading G7
  double b_lo, b_hi, beta;                               // bisection bracket and the exponent under test
  int temper_set;
};

__device__ __forceinline__ void em_derive(int d, int k, EmState &st) {
  const double a = st.cov[k][0], b = d == 2 ? st.cov[k][1] : 0.0, c = d == 2 ? st.cov[k][2] : 1.0;
  const double det = a * c - b * b;
  st.prec[k][0] = c / det, st.prec[k][1] = -b / det, st.prec[k][2] = a / det;
  st.lnc[k] = (st.pi[k] > 0.0 ? log(st.pi[k]) : -INFINITY) - 0.5 * log(det) - 0.5 * d * 1.8378770664093454836;
}

// Eq. (A4)-(A6) from the sums about the old means, the convergence test and the validity checks: one thread (<= 8 components)
__global__ void gmm_mstep_kernel(const double *__restrict__ sums, EmState *__restrict__ stp, int d, int K, double reg, double tol) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  EmState &st = *stp;
  if (st.done) return;
  const double W = sums[GM_MAXK * 6 + 1];
  if (!(W > 0.0)) {
    st.bad = st.done = 1;
    return;
  }
  const double ll = sums[GM_MAXK * 6] / W;
  st.ll = ll;
  if (st.it > 0 && fabs(ll - st.prev) < tol) {
    st.done = 1;
    return;
  }
  double mu[GM_MAXK][2], cov[GM_MAXK][3], pi[GM_MAXK], psum = 0.0;
  bool ok = true;
  for (int k = 0; k < K; ++k) {
    const double *a = sums + 6 * k;
    if (!(a[0] > 0.0)) ok = false;                               // an empty component
    const double e0 = a[1] / a[0], e1 = a[2] / a[0];
    mu[k][0] = st.mu[k][0] + e0;
    mu[k][1] = d == 2 ? st.mu[k][1] + e1 : 0.0;
    cov[k][0] = a[3] / a[0] - e0 * e0 + reg;
    cov[k][1] = d == 2 ? a[4] / a[0] - e0 * e1 : 0.0;
    cov[k][2] = d == 2 ? a[5] / a[0] - e1 * e1 + reg : 1.0;
    pi[k] = a[0] / W;
    psum += pi[k];
    const double det = cov[k][0] * cov[k][2] - cov[k][1] * cov[k][1];
    if (!(pi[k] >= 0.0) || !isfinite(pi[k]) || !isfinite(mu[k][0]) || !isfinite(mu[k][1]) || !(cov[k][0] > 0.0) || !isfinite(cov[k][0]) ||
        (d == 2 && (!(cov[k][2] > 0.0) || !(det > 0.0) || !isfinite(det))))
      ok = false;
  }
  if (!ok || !(fabs(psum - 1.0) < 1e-9)) {
    st.bad = st.done = 1;                                        // the model of the last valid M-step stays
    return;
  }
  for (int k = 0; k < K; ++k) {
    st.mu[k][0] = mu[k][0], st.mu[k][1] = mu[k][1];
    st.cov[k][0] = cov[k][0], st.cov[k][1] = cov[k][1], st.cov[k][2] = cov[k][2];
    st.pi[k] = pi[k];
    em_derive(d, k, st);
  }
  st.prev = ll;
  st.it += 1;
}

__global__ void __launch_bounds__(GM_THREADS) gmm_max_kernel(int64_t n, const double *__restrict__ ln_w, double *__restrict__ partial) {
  __shared__ double s_w[GM_THREADS / 32];
  double m = -INFINITY;
  for (int64_t i = (int64_t)blockIdx.x * GM_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GM_THREADS) {
    const double v = ln_w[i];
    if (v == v) m = fmax(m, v);                                                  // NaN counts as -inf
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < GM_THREADS / 32; ++w) m = fmax(m, s_w[w]);
    partial[blockIdx.x] = m;
  }
}

// maximum of the block maxima; no finite weight at all stops the fit
__global__ void gmm_maxfin_kernel(int n_blocks, const double *__restrict__ partial, EmState *__restrict__ stp) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double m = -INFINITY;
  for (int b = 0; b < n_blocks; ++b) m = fmax(m, partial[b]);
  stp->w_max = m;
  if (!(m > -INFINITY) || !isfinite(m)) stp->bad = stp->done = 1;
}

// one step of reading G7 on the device: step 0 tests temper = 1, steps 1..20 bisect [0, 1]; the exponent under test is
// stp->beta, the sums of the pass just made are in `partial`
__global__ void gmm_ess_step_kernel(int n_blocks, const double *__restrict__ partial, EmState *__restrict__ stp, double ess_min,
                                    int step) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  EmState &st = *stp;
  if (st.done || st.temper_set) return;
  double s1 = 0.0, s2 = 0.0;
  for (int b = 0; b < n_blocks; ++b) s1 += partial[2 * b], s2 += partial[2 * b + 1];
  const double ess = s2 > 0.0 ? s1 * s1 / s2 : 0.0;
  if (step == 0) {
    if (ess >= ess_min) {
      st.temper = 1.0;
      st.temper_set = 1;
    } else {
      st.b_lo = 0.0, st.b_hi = 1.0, st.beta = 0.5;
    }
    return;
  }
  if (ess >= ess_min) st.b_lo = st.beta;
  else st.b_hi = st.beta;
  st.beta = 0.5 * (st.b_lo + st.b_hi);
  if (step == 20) {
    st.temper = st.b_lo;
    st.temper_set = 1;
  }
}

// sum w^beta and sum w^(2 beta), w = exp(ln_w - w_max): the tempered effective sample size (sum)^2 / (sum of squares)
__global__ void __launch_bounds__(GM_THREADS) gmm_ess_kernel(int64_t n, const double *__restrict__ ln_w,
                                                             const EmState *__restrict__ stp, double *__restrict__ partial) {
  __shared__ double s_w[GM_THREADS / 32][2];
  if (stp->done || stp->temper_set) return;
  const double w_max = stp->w_max, beta = stp->beta;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * GM_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GM_THREADS) {
    const double v = ln_w[i];
    if (v == v && v > -INFINITY) {
      const double w = exp(beta * (v - w_max));
      s1 += w;
      s2 += w * w;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
  }
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5][0] = s1, s_w[threadIdx.x >> 5][1] = s2;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < GM_THREADS / 32; ++w) s1 += s_w[w][0], s2 += s_w[w][1];
    partial[2 * blockIdx.x] = s1;
    partial[2 * blockIdx.x + 1] = s2;
  }
}

__global__ void __launch_bounds__(GM_THREADS) gmm_em_kernel(int64_t n, const double *__restrict__ x0p, const double *__restrict__ x1p,
                                                            const double *__restrict__ ln_w,
                                                            const EmState *__restrict__ stp, int d, int K,
                                                            double *__restrict__ partial) {
  __shared__ double s_red[GM_THREADS / 32][GM_ROW];
  __shared__ GmmDev g;                                           // the fields the E-step reads, from the device-resident model
  if (stp->done) return;                                         // converged or stopped: the remaining launches are no-ops
  const double w_max = stp->w_max, temper = stp->temper;
  if (threadIdx.x == 0) g.d = d, g.K = K;
  if (threadIdx.x < GM_MAXK) {
    const int k = threadIdx.x;
    g.mu[k][0] = stp->mu[k][0], g.mu[k][1] = stp->mu[k][1];
    g.prec[k][0] = stp->prec[k][0], g.prec[k][1] = stp->prec[k][1], g.prec[k][2] = stp->prec[k][2];
    g.lnc[k] = stp->lnc[k];
  }
  __syncthreads();
  double acc[GM_ROW];
#pragma unroll
  for (int j = 0; j < GM_ROW; ++j) acc[j] = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * GM_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GM_THREADS) {
    double w = 1.0;
    if (ln_w) {
      const double v = ln_w[i];
      w = v == v ? exp(temper * (v - w_max)) : 0.0;
      if (v == -INFINITY) w = 0.0;                       // also when temper = 0
    }
    if (w == 0.0) continue;
    const double x0 = x0p[i], x1 = g.d == 2 ? x1p[i] : 0.0;
    double lp[GM_MAXK];
    const double lse = gm_log_terms<false>(g, x0, x1, lp);
    acc[GM_MAXK * 6] += w * lse;
    acc[GM_MAXK * 6 + 1] += w;
#pragma unroll
    for (int k = 0; k < GM_MAXK; ++k) {
      if (k < g.K) {
        const double p = w * exp(lp[k] - lse);
        const double d0 = x0 - g.mu[k][0], d1 = x1 - g.mu[k][1];
        acc[6 * k + 0] += p;
        acc[6 * k + 1] += p * d0;
        acc[6 * k + 2] += p * d1;
        acc[6 * k + 3] += p * d0 * d0;
        acc[6 * k + 4] += p * d0 * d1;
        acc[6 * k + 5] += p * d1 * d1;
      }
    }
  }
#pragma unroll
  for (int j = 0; j < GM_ROW; ++j) {
    double v = acc[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5][j] = v;
  }
  __syncthreads();
  if (threadIdx.x < GM_ROW) {
    double v = 0.0;
    for (int w = 0; w < GM_THREADS / 32; ++w) v += s_red[w][threadIdx.x];
    partial[(int64_t)blockIdx.x * GM_ROW + threadIdx.x] = v;
  }
}

__global__ void gmm_sum_kernel(int n_blocks, const double *__restrict__ partial, double *__restrict__ sums) {
  if (threadIdx.x < GM_ROW) {
    double v = 0.0;
    for (int b = 0; b < n_blocks; ++b) v += partial[(int64_t)b * GM_ROW + threadIdx.x];
    sums[threadIdx.x] = v;
  }
}

__global__ void __launch_bounds__(GM_THREADS) gmm_draw_kernel(int64_t n, uint64_t seed, uint64_t offset, const GmmDev g,
                                                              double *__restrict__ x0p, double *__restrict__ x1p,
                                                              double *__restrict__ ln_ps, unsigned long long *__restrict__ n_fail) {
  for (int64_t i = (int64_t)blockIdx.x * GM_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GM_THREADS) {
    const uint64_t idx = offset + (uint64_t)i;
    const double uc = gm_u01(seed, idx * (uint64_t)(GM_TRIES * 4));
    int k = 0;
    while (k < g.K - 1 && !(g.cum[k] > uc)) ++k;                                  // the first component with cum > u
    double x0 = 0.0, x1 = 0.0;
    bool ok = false;
    for (int t = 0; t < GM_TRIES && !ok; ++t) {
      const uint64_t c = (idx * (uint64_t)GM_TRIES + (uint64_t)t) * 4ull;
      const double z0 = normcdfinv(g.pa[k][0] + gm_u01(seed, c + 1) * g.pw[k][0]);
      if (g.d == 2) {
        const double z1 = normcdfinv(g.pa[k][1] + gm_u01(seed, c + 2) * g.pw[k][1]);
        x0 = g.mu[k][0] + (g.A[k][0] * z0 + g.A[k][1] * z1);
        x1 = g.mu[k][1] + (g.A[k][2] * z0 + g.A[k][3] * z1);
        ok = x0 >= g.lo[0] && x0 < g.hi[0] && x1 >= g.lo[1] && x1 < g.hi[1];
      } else {
        x0 = g.mu[k][0] + g.A[k][0] * z0;
        ok = x0 >= g.lo[0] && x0 < g.hi[0];
      }
    }
    if (!ok) {
      x0 = fmin(fmax(g.mu[k][0], g.lo[0]), nextafter(g.hi[0], g.lo[0]));
      if (g.d == 2) x1 = fmin(fmax(g.mu[k][1], g.lo[1]), nextafter(g.hi[1], g.lo[1]));
      atomicAdd(n_fail, 1ull);
    }
    x0p[i] = x0;
    if (g.d == 2) x1p[i] = x1;
    if (ln_ps) {
      double lp[GM_MAXK];
      ln_ps[i] = gm_log_terms<true>(g, x0, x1, lp);
    }
  }
}

__global__ void __launch_bounds__(GM_THREADS) gmm_density_kernel(int64_t n, const GmmDev g, const double *__restrict__ x0p,
                                                                 const double *__restrict__ x1p, double *__restrict__ ln_ps) {
  for (int64_t i = (int64_t)blockIdx.x * GM_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GM_THREADS) {
    const double x0 = x0p[i], x1 = g.d == 2 ? x1p[i] : 0.0;
    bool in = x0 >= g.lo[0] && x0 < g.hi[0];
    if (g.d == 2) in = in && x1 >= g.lo[1] && x1 < g.hi[1];
    double lp[GM_MAXK];
    ln_ps[i] = in ? gm_log_terms<true>(g, x0, x1, lp) : -INFINITY;
  }
}

struct SumTerms {
  const double *t[8];
};
__global__ void __launch_bounds__(GM_THREADS) gmm_add_kernel(int64_t n, int n_terms, SumTerms T, double *__restrict__ out) {
  for (int64_t i = (int64_t)blockIdx.x * GM_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GM_THREADS) {
    double v = T.t[0][i];
    for (int j = 1; j < n_terms; ++j) v += T.t[j][i];
    out[i] = v;
  }
}

inline int gm_grid(int64_t n) {
  int64_t b = (n + GM_THREADS - 1) / GM_THREADS;
  if (b > GM_BLOCKS) b = GM_BLOCKS;
  return b < 1 ? 1 : (int)b;
}

struct GmGuard {                                   // make the handle's device current for the call
  int prev = -1;
  explicit GmGuard(int dev) {
    cudaGetDevice(&prev);
    if (prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~GmGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

void ensure_dev(rift_gmm *h) {
  if (!h->dev_ok) {
    derive(h->d, h->K, h->lo, h->hi, h->model, true, h->dev);
    h->dev_ok = true;
  }
}

}  // namespace

extern "C" int rift_gmm_create(int32_t n_dim, int32_t n_comp, const double *lo, const double *hi, rift_gmm_t **out) {
  if (!out) return RIFT_EINVAL;
  *out = nullptr;
  if ((n_dim != 1 && n_dim != 2) || n_comp < 1 || n_comp > GM_MAXK || !lo || !hi) return RIFT_EINVAL;
  for (int j = 0; j < n_dim; ++j)
    if (!(hi[j] > lo[j]) || !std::isfinite(lo[j]) || !std::isfinite(hi[j])) return RIFT_EINVAL;
  rift_gmm *h = new (std::nothrow) rift_gmm();
  if (!h) return RIFT_ENOMEM;
  h->d = n_dim, h->K = n_comp;
  for (int j = 0; j < n_dim; ++j) h->lo[j] = lo[j], h->hi[j] = hi[j];
  for (int k = 0; k < n_comp; ++k) {
    h->model.pi[k] = 1.0 / n_comp;
    for (int j = 0; j < n_dim; ++j) h->model.mu[k][j] = lo[j] + (k + 0.5) / n_comp * (hi[j] - lo[j]);
    const double s0 = (hi[0] - lo[0]) / n_comp, s1 = n_dim == 2 ? (hi[1] - lo[1]) / n_comp : 1.0;
    h->model.cov[k][0] = s0 * s0, h->model.cov[k][1] = 0.0, h->model.cov[k][2] = s1 * s1;
  }
  if (cudaGetDevice(&h->device) != cudaSuccess || cudaMalloc(&h->d_partial, sizeof(double) * GM_BLOCKS * GM_ROW) != cudaSuccess ||
      cudaMalloc(&h->d_sums, sizeof(double) * GM_ROW) != cudaSuccess || cudaMalloc(&h->d_em, 4096) != cudaSuccess || cudaMalloc(&h->d_fail, sizeof(unsigned long long)) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(h->d_partial);
    cudaFree(h->d_sums);
    cudaFree(h->d_em);
    cudaFree(h->d_fail);
    delete h;
    return RIFT_ENOMEM;
  }
  *out = h;
  return RIFT_OK;
}

extern "C" int rift_gmm_destroy(rift_gmm_t *h) {
  if (!h) return RIFT_EINVAL;
  GmGuard g(h->device);
  cudaFree(h->d_partial);
  cudaFree(h->d_sums);
  cudaFree(h->d_em);
  cudaFree(h->d_fail);
  delete h;
  return RIFT_OK;
}

extern "C" int rift_gmm_set_model(rift_gmm_t *h, const double *mu, const double *cov, const double *pi, double n_trained) {
  if (!h || !mu || !cov || !pi || !(n_trained >= 0.0)) return RIFT_EINVAL;
  Model m{};
  const int d = h->d;
  for (int k = 0; k < h->K; ++k) {
    for (int j = 0; j < d; ++j) m.mu[k][j] = mu[k * d + j];
    const double *c = cov + (size_t)k * d * d;
    m.cov[k][0] = c[0];
    m.cov[k][1] = d == 2 ? 0.5 * (c[1] + c[2]) : 0.0;
    m.cov[k][2] = d == 2 ? c[3] : 1.0;
    if (d == 2 && std::fabs(c[1] - c[2]) > 1e-12 * std::sqrt(std::fabs(c[0] * c[3]))) return RIFT_EINVAL;   // not symmetric
    m.pi[k] = pi[k];
  }
  if (!model_valid(d, h->K, m)) return RIFT_EINVAL;
  h->model = m;
  h->n_trained = n_trained;
  h->dev_ok = false;
  return RIFT_OK;
}

extern "C" int rift_gmm_get_model(const rift_gmm_t *h, double *mu, double *cov, double *pi, double *n_trained) {
  if (!h) return RIFT_EINVAL;
  const int d = h->d;
  for (int k = 0; k < h->K; ++k) {
    if (mu)
      for (int j = 0; j < d; ++j) mu[k * d + j] = h->model.mu[k][j];
    if (cov) {
      double *c = cov + (size_t)k * d * d;
      c[0] = h->model.cov[k][0];
      if (d == 2) c[1] = c[2] = h->model.cov[k][1], c[3] = h->model.cov[k][2];
    }
    if (pi) pi[k] = h->model.pi[k];
  }
  if (n_trained) *n_trained = h->n_trained;
  return RIFT_OK;
}

namespace {

double mahalanobis(int d, const double a[2], const double b[2], const double c[3]) {
  const double d0 = a[0] - b[0];
  if (d == 1) return std::sqrt(std::fmax(0.0, d0 * d0 / c[0]));
  const double d1 = a[1] - b[1], det = c[0] * c[2] - c[1] * c[1];
  return std::sqrt(std::fmax(0.0, (c[2] * d0 * d0 - 2.0 * c[1] * d0 * d1 + c[0] * d1 * d1) / det));
}

// Eq. (A8)-(A11), G3: `nw` (trained on n_new samples) merged into `old` (n_old samples); the result is indexed like `old`
void merge_models(int d, int K, const Model &old, double n_old, const Model &nw, double n_new, Model &out) {
  double cost[GM_MAXK][GM_MAXK];
  for (int i = 0; i < K; ++i)
    for (int j = 0; j < K; ++j)
      cost[i][j] = mahalanobis(d, old.mu[j], nw.mu[i], nw.cov[i]) + mahalanobis(d, nw.mu[i], old.mu[j], old.cov[j]);
  int perm[GM_MAXK], best_perm[GM_MAXK];
  for (int i = 0; i < K; ++i) perm[i] = best_perm[i] = i;
  double best = INFINITY;
  do {                                                     // lexicographic order; the first minimum is kept
    double c = 0.0;
    for (int i = 0; i < K; ++i) c += cost[i][perm[i]];
    if (c < best) {
      best = c;
      std::copy(perm, perm + K, best_perm);
    }
  } while (std::next_permutation(perm, perm + K));
  out = old;
  for (int i = 0; i < K; ++i) {
    const int j = best_perm[i];
    const double a = n_old * old.pi[j], b = n_new * nw.pi[i], s = a + b;
    double m[2];
    for (int q = 0; q < 2; ++q) m[q] = (a * old.mu[j][q] + b * nw.mu[i][q]) / s;
    const int ix[3][2] = {{0, 0}, {0, 1}, {1, 1}};
    for (int e = 0; e < 3; ++e) {
      const int p = ix[e][0], q = ix[e][1];
      out.cov[j][e] = (a * old.cov[j][e] + b * nw.cov[i][e]) / s + (a * old.mu[j][p] * old.mu[j][q] + b * nw.mu[i][p] * nw.mu[i][q]) / s -
                      m[p] * m[q];
    }
    if (d == 1) out.cov[j][1] = 0.0, out.cov[j][2] = 1.0;
    out.mu[j][0] = m[0], out.mu[j][1] = m[1];
    out.pi[j] = s / (n_old + n_new);
  }
}

}  // namespace

namespace {
int gmm_fit_impl(rift_gmm_t *h, int64_t n, const double *const *x, const double *ln_w, double ess_min, int32_t n_iter, double tol,
                 double reg, int32_t merge, double *temper_used, int32_t *iters_done, double *loglik, void *cuda_stream) {
  if (!h || n < 1 || !x || !x[0] || (h->d == 2 && !x[1]) || n_iter < 0 || !(tol >= 0.0) || !(reg >= 0.0) || !(ess_min >= 0.0))
    return RIFT_EINVAL;
  GmGuard guard(h->device);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int d = h->d, K = h->K, grid = gm_grid(n);
  // the model lives on the device for the whole fit: E-step + sums, a fixed-order add, the M-step kernel; the host looks at the
  // state every 8 iterations (converged / stopped?) and once at the end
  static_assert(sizeof(EmState) <= 4096, "EmState buffer");
  EmState st;
  std::memset(&st, 0, sizeof(st));
  {
    GmmDev g;
    derive(d, K, h->lo, h->hi, h->model, false, g);
    for (int k = 0; k < K; ++k) {
      for (int j = 0; j < 2; ++j) st.mu[k][j] = h->model.mu[k][j];
      for (int j = 0; j < 3; ++j) st.cov[k][j] = h->model.cov[k][j], st.prec[k][j] = g.prec[k][j];
      st.pi[k] = h->model.pi[k];
      st.lnc[k] = g.lnc[k];
    }
    st.ll = -INFINITY;
    st.w_max = 0.0, st.temper = 1.0, st.beta = 1.0, st.temper_set = (ln_w && ess_min > 0.0) ? 0 : 1;
  }
  EmState *d_st = static_cast<EmState *>(h->d_em);
  if (cudaMemcpyAsync(d_st, &st, sizeof(st), cudaMemcpyHostToDevice, s) != cudaSuccess) return RIFT_ECUDA;
  if (ln_w) {
    gmm_max_kernel<<<grid, GM_THREADS, 0, s>>>(n, ln_w, h->d_partial);
    gmm_maxfin_kernel<<<1, 32, 0, s>>>(grid, h->d_partial, d_st);
    // G7: the largest temper in [0, 1] (20 bisection steps) whose tempered effective sample size reaches ess_min -- 21 passes
    // over the log-weights, decided on the device (later passes are no-ops once temper = 1 is accepted)
    if (ess_min > 0.0)
      for (int step = 0; step <= 20; ++step) {
        gmm_ess_kernel<<<grid, GM_THREADS, 0, s>>>(n, ln_w, d_st, h->d_partial);
        gmm_ess_step_kernel<<<1, 32, 0, s>>>(grid, h->d_partial, d_st, ess_min, step);
      }
  }
  for (int it0 = 0; it0 < n_iter && !st.done; it0 += 8) {
    // n_iter M-steps need n_iter E-steps; a tolerance stop is detected by the E-step after the last M-step it follows
    const int todo = std::min(8, n_iter - it0);
    for (int j = 0; j < todo; ++j) {
      gmm_em_kernel<<<grid, GM_THREADS, 0, s>>>(n, x[0], d == 2 ? x[1] : nullptr, ln_w, d_st, d, K, h->d_partial);
      gmm_sum_kernel<<<1, 64, 0, s>>>(grid, h->d_partial, h->d_sums);
      gmm_mstep_kernel<<<1, 32, 0, s>>>(h->d_sums, d_st, d, K, reg, tol);
    }
    if (cudaGetLastError() != cudaSuccess || cudaMemcpyAsync(&st, d_st, sizeof(st), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess)
      return RIFT_ECUDA;
  }
  if (n_iter == 0 && (cudaMemcpyAsync(&st, d_st, sizeof(st), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
                      cudaStreamSynchronize(s) != cudaSuccess))
    return RIFT_ECUDA;
  if (st.bad) return RIFT_ESTATE;                                 // every weight zero, an empty component or a bad covariance
  const double temper = st.temper;
  Model m = h->model;
  for (int k = 0; k < K; ++k) {
    for (int j = 0; j < 2; ++j) m.mu[k][j] = st.mu[k][j];
    for (int j = 0; j < 3; ++j) m.cov[k][j] = st.cov[k][j];
    m.pi[k] = st.pi[k];
  }
  if (n_iter > 0 && !model_valid(d, K, m)) return RIFT_ESTATE;
  const int it = st.it;
  const double ll = st.ll;
  if (merge && h->n_trained > 0.0) {
    Model out;
    merge_models(d, K, h->model, h->n_trained, m, (double)n, out);
    if (!model_valid(d, K, out)) return RIFT_ESTATE;
    h->model = out;
    h->n_trained += (double)n;
  } else {
    h->model = m;
    h->n_trained = (double)n;
  }
  h->dev_ok = false;
  if (iters_done) *iters_done = it;
  if (loglik) *loglik = ll;
  if (temper_used) *temper_used = temper;
  return RIFT_OK;
}
}  // namespace

extern "C" int rift_gmm_fit(rift_gmm_t *h, int64_t n, const double *const *x, const double *ln_w, int32_t n_iter, double tol,
                            double reg, int32_t merge, int32_t *iters_done, double *loglik, void *cuda_stream) {
  return gmm_fit_impl(h, n, x, ln_w, 0.0, n_iter, tol, reg, merge, nullptr, iters_done, loglik, cuda_stream);
}

extern "C" int rift_gmm_fit_tempered(rift_gmm_t *h, int64_t n, const double *const *x, const double *ln_w, double ess_min,
                                     int32_t n_iter, double tol, double reg, int32_t merge, double *temper_used,
                                     int32_t *iters_done, double *loglik, void *cuda_stream) {
  return gmm_fit_impl(h, n, x, ln_w, ess_min, n_iter, tol, reg, merge, temper_used, iters_done, loglik, cuda_stream);
}

extern "C" int rift_gmm_draw(rift_gmm_t *h, int64_t n, uint64_t seed, uint64_t offset, double *const *x, double *ln_ps,
                             int64_t *n_failed, void *cuda_stream) {
  if (!h || n < 0 || !x || (n > 0 && (!x[0] || (h->d == 2 && !x[1])))) return RIFT_EINVAL;
  GmGuard guard(h->device);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  ensure_dev(h);
  if (cudaMemsetAsync(h->d_fail, 0, sizeof(unsigned long long), s) != cudaSuccess) return RIFT_ECUDA;
  if (n > 0) gmm_draw_kernel<<<gm_grid(n), GM_THREADS, 0, s>>>(n, seed, offset, h->dev, x[0], h->d == 2 ? x[1] : nullptr, ln_ps, h->d_fail);
  if (cudaGetLastError() != cudaSuccess) return RIFT_ECUDA;
  if (n_failed) {
    unsigned long long f = 0;
    if (cudaMemcpyAsync(&f, h->d_fail, sizeof(f), cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
      return RIFT_ECUDA;
    *n_failed = (int64_t)f;
  }
  return RIFT_OK;
}

extern "C" int rift_gmm_ln_density(rift_gmm_t *h, int64_t n, const double *const *x, double *ln_ps, void *cuda_stream) {
  if (!h || n < 0 || !x || (n > 0 && (!x[0] || (h->d == 2 && !x[1]) || !ln_ps))) return RIFT_EINVAL;
  if (n == 0) return RIFT_OK;
  GmGuard guard(h->device);
  ensure_dev(h);
  gmm_density_kernel<<<gm_grid(n), GM_THREADS, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(n, h->dev, x[0], h->d == 2 ? x[1] : nullptr,
                                                                                            ln_ps);
  return cudaGetLastError() == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}

extern "C" int rift_gmm_box_mass(rift_gmm_t *h, double *Z) {
  if (!h || !Z) return RIFT_EINVAL;
  ensure_dev(h);
  for (int k = 0; k < h->K; ++k) Z[k] = std::exp(h->dev.lnz[k]);
  return RIFT_OK;
}

extern "C" int rift_gmm_add(int64_t n, int32_t n_terms, const double *const *terms, double *out, void *cuda_stream) {
  if (n < 0 || n_terms < 1 || n_terms > 8 || !terms || (n > 0 && !out)) return RIFT_EINVAL;
  SumTerms T{};
  for (int j = 0; j < n_terms; ++j) {
    if (!terms[j]) return RIFT_EINVAL;
    T.t[j] = terms[j];
  }
  if (n == 0) return RIFT_OK;
  int64_t b = (n + GM_THREADS - 1) / GM_THREADS;
  if (b > 148 * 8) b = 148 * 8;
  gmm_add_kernel<<<(int)b, GM_THREADS, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(n, n_terms, T, out);
  return cudaGetLastError() == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}
