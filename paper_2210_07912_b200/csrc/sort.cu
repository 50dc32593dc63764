// Grouping of extrinsic samples by their RELATIVE integer shift tuple d_k = s_k - s_0 (step a3, reading G4).
// Samples of one segment that share the tuple read exactly the same Q rows at the same offsets, so the fused
// lnL kernel can serve several samples from one shared-memory load.  Three small kernels:
//   key_hist   : per sample, shifts -> bucket id (exact mixed-radix index of the tuple when it fits, else a hash),
//                histogram by atomics
//   scan       : exclusive scan of each segment's bucket counts (one block per segment of the chunk)
//   scatter    : perm[slot] = sample; order inside a bucket is arbitrary (results do not depend on it)
#include "rift_internal.h"

namespace {

constexpr int SORT_THREADS = 256;

__device__ __forceinline__ uint32_t mix32(uint32_t h, uint32_t v) {
  h ^= v + 0x9e3779b9u + (h << 6) + (h >> 2);
  return h;
}

__global__ void __launch_bounds__(SORT_THREADS)
key_hist_kernel(DetGeom g, SortPlan sp, Batch b, const double *__restrict__ p_ra, const double *__restrict__ p_dec,
                int32_t *__restrict__ bucket_of, uint32_t *__restrict__ hist) {
  const int64_t w = (int64_t)blockIdx.x * SORT_THREADS + threadIdx.x;
  if (w >= b.n) return;
  const int64_t gi = b.g0 + w;
  const int32_t seg_local = (int32_t)(gi / b.n_per_seg - b.g0 / b.n_per_seg);
  double sd, cd, sh, ch;
  sincos(p_dec[gi], &sd, &cd);
  sincos(p_ra[gi] - g.gmst, &sh, &ch);
  const double nx = __dmul_rn(cd, ch), ny = __dmul_rn(cd, sh), nz = sd;
  int32_t s0 = 0;
  uint32_t idx = 0, hsh = 0x811c9dc5u;
  for (int k = 0; k < g.n_det; ++k) {
    const double dot = __dadd_rn(__dadd_rn(__dmul_rn(g.loc[k][0], nx), __dmul_rn(g.loc[k][1], ny)),
                                 __dmul_rn(g.loc[k][2], nz));
    const double dt = -__ddiv_rn(dot, RIFT_C_LIGHT);
    const double x = __ddiv_rn(dt, g.delta_t);
    const double f = floor(__dadd_rn(x, 0.5));
    const int32_t s = (f == f && fabs(f) < 1e9) ? (int32_t)f : 0;      // NaN / inf sky angles: any bucket will do
    if (k == 0) {
      s0 = s;
    } else {
      const int32_t d = s - s0;
      int32_t u = d + sp.half[k];
      u = u < 0 ? 0 : (u >= sp.range[k] ? sp.range[k] - 1 : u);
      idx = idx * (uint32_t)sp.range[k] + (uint32_t)u;
      hsh = mix32(hsh, (uint32_t)d);
    }
  }
  const uint32_t bkt = sp.exact ? idx : (hsh & (uint32_t)(sp.n_buckets - 1));
  const int32_t slot = seg_local * sp.n_buckets + (int32_t)(bkt < (uint32_t)sp.n_buckets ? bkt : 0);
  bucket_of[w] = slot;
  atomicAdd(&hist[slot], 1u);
}

// one block per segment of the chunk: hist[seg][0..NB) -> exclusive prefix + first workspace slot of the segment
__global__ void __launch_bounds__(SORT_THREADS) scan_kernel(SortPlan sp, Batch b, uint32_t *__restrict__ hist) {
  __shared__ uint32_t warp_tot[SORT_THREADS / 32];
  __shared__ uint32_t carry;
  const int seg_local = blockIdx.x;
  const int64_t seg = b.g0 / b.n_per_seg + seg_local;
  const int64_t seg_begin = seg * b.n_per_seg - b.g0;
  uint32_t *h = hist + (int64_t)seg_local * sp.n_buckets;
  if (threadIdx.x == 0) carry = (uint32_t)(seg_begin > 0 ? seg_begin : 0);
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int base = 0; base < sp.n_buckets; base += SORT_THREADS) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < sp.n_buckets ? h[i] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    uint32_t off = carry;
    for (int j = 0; j < warp; ++j) off += warp_tot[j];
    if (i < sp.n_buckets) h[i] = off + inc - v;
    __syncthreads();
    if (threadIdx.x == SORT_THREADS - 1) carry = off + inc;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(SORT_THREADS)
scatter_kernel(Batch b, const int32_t *__restrict__ bucket_of, uint32_t *__restrict__ cursor, int32_t *__restrict__ perm) {
  const int64_t w = (int64_t)blockIdx.x * SORT_THREADS + threadIdx.x;
  if (w >= b.n) return;
  const uint32_t pos = atomicAdd(&cursor[bucket_of[w]], 1u);
  perm[pos] = (int32_t)w;
}

}  // namespace

cudaError_t launch_group_sort(const DetGeom &g, const SortPlan &sp, const Batch &b, const double *const params[6],
                              int32_t *bucket_of, uint32_t *hist, int32_t n_seg_chunk, int32_t *perm, cudaStream_t s,
                              int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  cudaError_t e = cudaMemsetAsync(hist, 0, sizeof(uint32_t) * (size_t)n_seg_chunk * sp.n_buckets, s);
  if (e != cudaSuccess) return e;
  const unsigned grid = (unsigned)((b.n + SORT_THREADS - 1) / SORT_THREADS);
  key_hist_kernel<<<grid, SORT_THREADS, 0, s>>>(g, sp, b, params[0], params[1], bucket_of, hist);
  scan_kernel<<<n_seg_chunk, SORT_THREADS, 0, s>>>(sp, b, hist);
  scatter_kernel<<<grid, SORT_THREADS, 0, s>>>(b, bucket_of, hist, perm);
  if (n_launch) *n_launch += 3;
  return cudaGetLastError();
}
