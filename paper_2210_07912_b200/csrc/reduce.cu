// Sample-axis reduce, step a8 of DESIGN.md section 1 (fp64 throughout, HBM-bound).
//   ln omega_i = lnL_i + ln w_i;  lnZ = ln[(1/N) sum omega]  (Eq. (3));  n_eff = sum omega / max omega (B1);
//   n_ess = (sum omega)^2 / sum omega^2 (B2);  rel_err^2 = (N/n_ess - 1)/(N-1) (B3, reading A20);
//   weighted 1-D histograms per parameter (Eq. (22), reading A13).
// Two kernels: per-block partial states (block max, sums and histograms relative to the block max; warp-shuffle
// reductions), then one block per segment merges the partials with the stored state (Eq. (20)-(21): pooled sums).
#include <cstdio>
#include <mutex>

#include "rift_internal.h"

namespace {

constexpr int RED_THREADS = 256;
constexpr int PARTIAL_HDR = 4;   // m, s1, s2, nan flag

__device__ __forceinline__ double block_reduce(double v, double *scratch, bool is_max) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double u = __shfl_xor_sync(0xffffffffu, v, o);
    v = is_max ? fmax(v, u) : v + u;
  }
  __syncthreads();
  if (lane == 0) scratch[warp] = v;
  __syncthreads();
  double r = scratch[0];
  for (int i = 1; i < RED_THREADS / 32; ++i) r = is_max ? fmax(r, scratch[i]) : r + scratch[i];
  return r;
}

struct HistArgs {
  const double *p[6];
  double lo[6], hi[6];
};

__global__ void __launch_bounds__(RED_THREADS)
reduce_partial_kernel(int64_t n_per_seg, const double *__restrict__ lnL, const double *__restrict__ ln_w, HistArgs ha,
                      int has_params, int n_bins, double *__restrict__ partial) {
  extern __shared__ double sh[];
  double *scratch = sh;                 // [8]
  double *hist = sh + 8;                // [6][n_bins]
  const int seg = blockIdx.y, bx = blockIdx.x, nbx = gridDim.x;
  const int64_t chunk = (n_per_seg + nbx - 1) / nbx;
  const int64_t i0 = (int64_t)bx * chunk, i1 = min(n_per_seg, i0 + chunk);
  const int64_t base = (int64_t)seg * n_per_seg;
  const int pstride = PARTIAL_HDR + 6 * n_bins;
  double *out = partial + ((int64_t)seg * nbx + bx) * pstride;

  for (int i = threadIdx.x; i < 6 * n_bins; i += RED_THREADS) hist[i] = 0.0;

  double mx = -INFINITY;
  int nan_seen = 0;
  for (int64_t i = i0 + threadIdx.x; i < i1; i += RED_THREADS) {
    const double v = lnL[base + i] + (ln_w ? ln_w[base + i] : 0.0);
    if (isnan(v)) nan_seen = 1;
    mx = fmax(mx, v);
  }
  mx = block_reduce(mx, scratch, true);
  const double nanf = block_reduce((double)nan_seen, scratch, false);
  __syncthreads();

  double s1 = 0.0, s2 = 0.0;
  if (mx > -INFINITY && nanf == 0.0) {
    for (int64_t i = i0 + threadIdx.x; i < i1; i += RED_THREADS) {
      const double v = lnL[base + i] + (ln_w ? ln_w[base + i] : 0.0);
      const double w = exp(v - mx);
      s1 += w;
      s2 += w * w;
      if (has_params && w > 1e-25) {       // smaller weights cannot move a normalised bin by 1e-25 (the block max has w = 1)
#pragma unroll
        for (int d = 0; d < 6; ++d) {
          const double x = ha.p[d][base + i];
          int bin = (int)floor(((double)n_bins * (x - ha.lo[d])) / (ha.hi[d] - ha.lo[d]));
          if (!(bin >= 0)) bin = 0;
          if (bin > n_bins - 1) bin = n_bins - 1;
          atomicAdd(&hist[d * n_bins + bin], w);
        }
      }
    }
  }
  s1 = block_reduce(s1, scratch, false);
  s2 = block_reduce(s2, scratch, false);
  __syncthreads();
  if (threadIdx.x == 0) {
    out[0] = mx;
    out[1] = s1;
    out[2] = s2;
    out[3] = nanf;
  }
  for (int i = threadIdx.x; i < 6 * n_bins; i += RED_THREADS) out[PARTIAL_HDR + i] = hist[i];
}

__global__ void __launch_bounds__(128)
reduce_merge_kernel(int64_t n_per_seg, int n_seg, int nbx, int n_bins, int merge, const double *__restrict__ partial,
                    ReduceState *__restrict__ state, double *__restrict__ state_hist, double *__restrict__ out_scalars,
                    double *__restrict__ out_hist) {
  const int seg = blockIdx.x;
  const int pstride = PARTIAL_HDR + 6 * n_bins;
  const double *P = partial + (int64_t)seg * nbx * pstride;
  __shared__ double s_m, s_s1;
  __shared__ int s_nan;
  __shared__ double s_f[4096];                     // exp(m_b - m) per partial block (nbx <= 4096, reduce_blocks_per_seg)
  __shared__ double s_red[3][4];
  __shared__ int s_red_nan[4];
  ReduceState old;
  old.m = -INFINITY;
  old.s1 = old.s2 = 0.0;
  old.n = 0;
  if (merge) old = state[seg];
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;

  // pass 1 (all threads): NaN flag and maximum over the stored state and the partial blocks
  double m = old.m;
  int nan_seen = isnan(old.m) ? 1 : 0;
  for (int b = threadIdx.x; b < nbx; b += 128) {
    if (P[b * pstride + 3] != 0.0) nan_seen = 1;
    m = fmax(m, P[b * pstride]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    nan_seen |= __shfl_xor_sync(0xffffffffu, nan_seen, o);
  }
  if (lane == 0) {
    s_red[0][wrp] = m;
    s_red_nan[wrp] = nan_seen;
  }
  __syncthreads();
  m = fmax(fmax(s_red[0][0], s_red[0][1]), fmax(s_red[0][2], s_red[0][3]));
  nan_seen = s_red_nan[0] | s_red_nan[1] | s_red_nan[2] | s_red_nan[3];
  __syncthreads();
  // pass 2: rescaled sums
  double s1 = 0.0, s2 = 0.0;
  const bool live0 = !nan_seen && m > -INFINITY;
  for (int b = threadIdx.x; b < nbx; b += 128) {
    const double mb = P[b * pstride];
    double f = 0.0;
    if (live0 && mb > -INFINITY) {
      f = exp(mb - m);
      s1 += P[b * pstride + 1] * f;
      s2 += P[b * pstride + 2] * f * f;
    }
    s_f[b] = f;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
  }
  if (lane == 0) {
    s_red[1][wrp] = s1;
    s_red[2][wrp] = s2;
  }
  __syncthreads();

  if (threadIdx.x == 0) {
    s1 = (s_red[1][0] + s_red[1][1]) + (s_red[1][2] + s_red[1][3]);
    s2 = (s_red[2][0] + s_red[2][1]) + (s_red[2][2] + s_red[2][3]);
    if (live0 && old.m > -INFINITY) {
      const double f = exp(old.m - m);
      s1 += old.s1 * f;
      s2 += old.s2 * f * f;
    }
    const int64_t n = old.n + n_per_seg;
    ReduceState st;
    st.m = nan_seen ? __longlong_as_double(0x7ff8000000000000LL) : m;
    st.s1 = s1;
    st.s2 = s2;
    st.n = n;
    state[seg] = st;
    const double N = (double)n;
    double lnZ, rel, neff, ness;
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    if (nan_seen) {
      lnZ = rel = neff = ness = qnan;
    } else if (n == 0 || !(m > -INFINITY)) {
      lnZ = (n == 0) ? qnan : m;
      rel = qnan;
      neff = ness = 0.0;
    } else {
      lnZ = m + log(s1) - log(N);
      neff = s1;
      ness = s1 * s1 / s2;
      if (n > 1) {
        const double r2 = (N / ness - 1.0) / (N - 1.0);
        rel = sqrt(r2 > 0.0 ? r2 : 0.0);
      } else {
        rel = 0.0;
      }
    }
    out_scalars[0 * n_seg + seg] = lnZ;
    out_scalars[1 * n_seg + seg] = rel;
    out_scalars[2 * n_seg + seg] = neff;
    out_scalars[3 * n_seg + seg] = ness;
    s_m = m;
    s_s1 = s1;
    s_nan = nan_seen;
  }
  __syncthreads();
  if (state_hist == nullptr) return;
  const double mfin = s_m, s1fin = s_s1;
  const bool live = !s_nan && mfin > -INFINITY;
  const double f_old = (merge && live && old.m > -INFINITY) ? exp(old.m - mfin) : 0.0;
  for (int i = threadIdx.x; i < 6 * n_bins; i += blockDim.x) {
    double h = 0.0;
    if (live) {
      if (f_old != 0.0) h = state_hist[(int64_t)seg * 6 * n_bins + i] * f_old;
      double h4[4] = {0.0, 0.0, 0.0, 0.0};                  // four independent chains: the loads of a bin are 4.8 KB apart
      int b = 0;
      for (; b + 4 <= nbx; b += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) h4[u] += P[(b + u) * pstride + PARTIAL_HDR + i] * s_f[b + u];
      }
      for (; b < nbx; ++b) h4[0] += P[b * pstride + PARTIAL_HDR + i] * s_f[b];
      h += (h4[0] + h4[1]) + (h4[2] + h4[3]);
    }
    state_hist[(int64_t)seg * 6 * n_bins + i] = h;
    if (out_hist) out_hist[(int64_t)seg * 6 * n_bins + i] = (live && s1fin > 0.0) ? h / s1fin : 0.0;
  }
}

}  // namespace

// ~2048 samples per block, at most ~4096 blocks over all segments (the partial buffer is n_seg * blocks * (4 + 6 n_bins))
int32_t reduce_blocks_per_seg(int64_t n_per_seg, int32_t n_seg) {
  int64_t b = (n_per_seg + 2047) / 2048;
  const int64_t cap = 4096 / (n_seg > 0 ? n_seg : 1);
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int32_t)b;
}

size_t reduce_partial_doubles(int32_t n_seg, int32_t blocks_per_seg, int32_t n_bins) {
  return (size_t)n_seg * blocks_per_seg * (PARTIAL_HDR + 6 * (size_t)n_bins);
}

cudaError_t launch_reduce(int32_t n_seg, int64_t n_per_seg, const double *lnL, const double *ln_w,
                          const double *const params[6], const double lo[6], const double hi[6], int32_t n_bins,
                          int merge, ReduceState *state, double *state_hist, double *partial, int32_t blocks_per_seg,
                          double *out_scalars, double *out_hist, cudaStream_t s, int *n_launch) {
  HistArgs ha;
  const bool hp = params != nullptr && n_bins > 0;
  for (int d = 0; d < 6; ++d) {
    ha.p[d] = hp ? params[d] : nullptr;
    ha.lo[d] = hp ? lo[d] : 0.0;
    ha.hi[d] = hp ? hi[d] : 1.0;
  }
  const int nb = hp ? n_bins : 0;
  const size_t smem = (8 + 6 * (size_t)nb) * sizeof(double);
  if (smem > 48u * 1024u) {            // 1023-1024 bins: 64 + 48 n_bins bytes pass the default dynamic limit
    cudaError_t ea = cudaFuncSetAttribute(reduce_partial_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (ea != cudaSuccess) return ea;
  }
  dim3 grid(blocks_per_seg, n_seg);
  reduce_partial_kernel<<<grid, RED_THREADS, smem, s>>>(n_per_seg, lnL, ln_w, ha, hp ? 1 : 0, nb, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  reduce_merge_kernel<<<n_seg, 128, 0, s>>>(n_per_seg, n_seg, blocks_per_seg, nb, merge, partial, state,
                                            hp ? state_hist : nullptr, out_scalars, hp ? out_hist : nullptr);
  if (n_launch) *n_launch += 2;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ allocation-free reduce
// rift_ile_reduce_static (include/rift_ile.h): the same two kernels as launch_reduce, scalar outputs only, with the
// per-block partial states and the per-segment state in a file-scope device array instead of buffers owned by a handle, so
// that the call allocates nothing (CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc).  Every GPU that
// loads the library holds the array (160 KiB) until the process exits.  In host code `g_static_scratch` is only a stand-in
// for the symbol: the device address comes from cudaGetSymbolAddress, once per device with that device current.

namespace {

constexpr int STATIC_MAX_SEG = RIFT_REDUCE_STATIC_MAX_SEG;          // per-segment states
constexpr int STATIC_MAX_BLOCKS = 4096;                             // partial blocks over all segments (reduce_blocks_per_seg)
constexpr size_t STATIC_STATE_DOUBLES = (size_t)STATIC_MAX_SEG * sizeof(ReduceState) / sizeof(double);
constexpr size_t STATIC_DOUBLES = STATIC_STATE_DOUBLES + (size_t)STATIC_MAX_BLOCKS * PARTIAL_HDR;
static_assert(sizeof(ReduceState) % sizeof(double) == 0, "ReduceState is a whole number of doubles");
static_assert(STATIC_MAX_SEG <= STATIC_MAX_BLOCKS, "one partial block per segment at least");

static __device__ __align__(256) double g_static_scratch[STATIC_DOUBLES];   // [state | partial]

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
double *g_static_ptr[STATIC_MAX_DEVICES] = {};                       // device address of g_static_scratch, per device
thread_local char g_static_error[160] = "";

int static_fail(int code, const char *msg) {
  snprintf(g_static_error, sizeof(g_static_error), "%s", msg);
  return code;
}

}  // namespace

extern "C" const char *rift_ile_reduce_static_error(void) { return g_static_error; }

extern "C" int rift_ile_reduce_static(int32_t n_seg, int64_t n_per_seg, const double *lnL, const double *ln_weight,
                                      double *out, void *cuda_stream) {
  g_static_error[0] = 0;
  if (n_seg < 1 || n_per_seg < 0) return static_fail(RIFT_EINVAL, "bad n_seg / n_per_seg");
  if (n_seg > STATIC_MAX_SEG)
    return static_fail(RIFT_EINVAL, "n_seg exceeds RIFT_REDUCE_STATIC_MAX_SEG (1024): the static scratch array holds no more "
                                    "segment states; use rift_ile_reduce");
  if ((n_per_seg > 0 && !lnL) || !out) return static_fail(RIFT_EINVAL, "null pointer");
  const int32_t bps = reduce_blocks_per_seg(n_per_seg, n_seg);
  if ((int64_t)bps * n_seg > STATIC_MAX_BLOCKS) return static_fail(RIFT_EINVAL, "partial blocks exceed the static scratch array");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= STATIC_MAX_DEVICES)
    return static_fail(RIFT_ECUDA, "cudaGetDevice failed or device ordinal >= 64");
  double *scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {                                        // set-up, once per device, that device current
      void *p = nullptr;
      const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
      if (e != cudaSuccess || !p) {
        cudaGetLastError();
        return static_fail(RIFT_ECUDA, "cudaGetSymbolAddress(g_static_scratch) failed");
      }
      g_static_ptr[dev] = static_cast<double *>(p);
    }
    scratch = g_static_ptr[dev];
  }
  // merge = 0: the merge kernel overwrites the segment states without reading them and the partial kernel writes every
  // partial slot the merge kernel reads, so nothing of the previous call's contents is used and nothing needs clearing
  ReduceState *state = reinterpret_cast<ReduceState *>(scratch);
  double *partial = scratch + STATIC_STATE_DOUBLES;
  const cudaError_t e = launch_reduce(n_seg, n_per_seg, lnL, ln_weight, nullptr, nullptr, nullptr, 0, 0, state, nullptr, partial,
                                      bps, out, nullptr, reinterpret_cast<cudaStream_t>(cuda_stream), nullptr);
  if (e != cudaSuccess) return static_fail(RIFT_ECUDA, cudaGetErrorString(e));
  return RIFT_OK;
}
