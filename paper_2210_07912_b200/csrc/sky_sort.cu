// Sky-cell bucketing ahead of lnl_sky (lnl_sky.cu): a counting sort of the samples of a chunk by (segment, sky cell).
// Every delay dt_k = -r_k.n/c (step a3) is a Lipschitz function of the source direction n with constant |r_k - r_0|/c for
// the RELATIVE delay, so samples of one small sky cell have relative shifts d_k = s_k - s_0 within a few samples of one
// another: a batch of one cell can be contracted by the tensor cores from ONE row range of Q per detector (the batch's
// smallest shift applied as the row offset) with residual per-sample shifts below e_max (SKY_E for lnl_sky, SKY64_E for lnl_sky64).  Cells: rings of constant width
// delta in declination, each cut into ceil(2 pi cos_max / delta) equal steps of hour angle, so that two directions of a cell
// are at most sqrt(2) delta apart; delta = (e_max - 1) / (sqrt(2) max_k |r_k - r_0| / (c delta_t)) bounds the spread of every
// d_k inside a cell by e_max - 1 (rounding included).
#include "rift_internal.h"

namespace {

__device__ __forceinline__ int sky_cell(const SkyCells &c, double ra, double dec, double gmst) {
  if (!(ra == ra) || !(dec == dec)) return 0;                             // NaN angles: any cell (the sample's lnL is NaN)
  int ring = (int)floor((dec + 1.5707963267948966) / c.delta);
  ring = ring < 0 ? 0 : (ring >= c.n_rings ? c.n_rings - 1 : ring);
  const int n_phi = c.ring_off[ring + 1] - c.ring_off[ring];
  double phi = fmod(ra - gmst, 6.283185307179586);
  if (phi < 0) phi += 6.283185307179586;
  int j = (int)(phi * (n_phi / 6.283185307179586));
  j = j < 0 ? 0 : (j >= n_phi ? n_phi - 1 : j);
  return c.ring_off[ring] + j;
}

// pass 1: bucket = local segment * n_cells + cell; the atomic's return value is the sample's position in its bucket
__global__ void __launch_bounds__(256) sky_key_kernel(SkyCells cells, double gmst, Batch b, const double *__restrict__ p_ra,
                                                      const double *__restrict__ p_dec, int32_t *__restrict__ key,
                                                      int32_t *__restrict__ pos, int32_t *__restrict__ count) {
  const int64_t w = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (w >= b.n) return;
  const int64_t gi = b.g0 + w;
  const int lseg = (int)(gi / b.n_per_seg - b.g0 / b.n_per_seg);
  const int bucket = lseg * cells.n_cells + sky_cell(cells, p_ra[gi], p_dec[gi], gmst);
  key[w] = bucket;
  pos[w] = atomicAdd(count + bucket, 1);
}

// pass 2 (one block): batches of SKY_NB slots per bucket, their exclusive prefix, the total
__global__ void __launch_bounds__(1024) sky_scan_kernel(const int32_t *__restrict__ count, int32_t *__restrict__ base, int n,
                                                        int32_t *__restrict__ n_batches) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int i0 = 0; i0 < n; i0 += 1024) {
    const int i = i0 + threadIdx.x;
    const int nb = i < n ? (count[i] + SKY_NB - 1) / SKY_NB : 0;
    int v = nb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += t;
    }
    if (lane == 31) s_warp[warp] = v;
    __syncthreads();
    if (warp == 0) {
      int t = s_warp[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, t, o);
        if (lane >= o) t += u;
      }
      s_warp[lane] = t;
    }
    __syncthreads();
    const int excl = s_carry + (warp ? s_warp[warp - 1] : 0) + v - nb;
    if (i < n) base[i] = excl;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = excl + nb;
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_batches = s_carry;
}

// pass 3: sorted slot of every sample = first slot of its bucket + position in the bucket; perm was preset to -1 (padding)
__global__ void __launch_bounds__(256) sky_fill_kernel(int64_t n, const int32_t *__restrict__ key, const int32_t *__restrict__ pos,
                                                       const int32_t *__restrict__ base, int32_t *__restrict__ perm) {
  const int64_t w = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (w >= n) return;
  perm[(int64_t)base[key[w]] * SKY_NB + pos[w]] = (int32_t)w;
}

}  // namespace

// Cells for a bound `dmax` (samples) on |d s_k / d n|: rings and their hour-angle steps.  Returns false if too many rings.
bool sky_make_cells(double dmax_samples, int e_max, SkyCells &c) {
  c = SkyCells{};
  double delta = (e_max - 1) / (1.4142135623730951 * (dmax_samples > 1.0 ? dmax_samples : 1.0));
  if (delta > 0.5) delta = 0.5;
  const int n_rings = (int)std::ceil(3.141592653589793 / delta);
  if (n_rings > SKY_MAX_RINGS) return false;
  c.delta = 3.141592653589793 / n_rings;
  c.n_rings = n_rings;
  int off = 0;
  for (int i = 0; i < n_rings; ++i) {
    const double d0 = -1.5707963267948966 + i * c.delta, d1 = d0 + c.delta;
    const double cmax = (d0 < 0 && d1 > 0) ? 1.0 : std::fmax(std::cos(d0), std::cos(d1));
    int n_phi = (int)std::ceil(6.283185307179586 * cmax / c.delta);
    if (n_phi < 1) n_phi = 1;
    c.ring_off[i] = off;
    off += n_phi;
  }
  c.ring_off[n_rings] = off;
  c.n_cells = off;
  return true;
}

// key / pos: [n]; count / base: [n_lseg * n_cells]; perm: [cap_slots]; n_batches: device int
cudaError_t launch_sky_sort(const SkyCells &cells, double gmst, const Batch &b, const double *const params[6], int n_lseg,
                            int32_t *key, int32_t *pos, int32_t *count, int32_t *base, int32_t *perm, int64_t cap_slots,
                            int32_t *n_batches, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  const int nbk = n_lseg * cells.n_cells;
  cudaError_t e = cudaMemsetAsync(count, 0, sizeof(int32_t) * (size_t)nbk, s);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(perm, 0xff, sizeof(int32_t) * (size_t)cap_slots, s);
  if (e != cudaSuccess) return e;
  const unsigned grid = (unsigned)((b.n + 255) / 256);
  sky_key_kernel<<<grid, 256, 0, s>>>(cells, gmst, b, params[0], params[1], key, pos, count);
  sky_scan_kernel<<<1, 1024, 0, s>>>(count, base, nbk, n_batches);
  sky_fill_kernel<<<grid, 256, 0, s>>>(b.n, key, pos, base, perm);
  if (n_launch) *n_launch += 3;
  return cudaGetLastError();
}
