// Fused lnL kernel of the mixed mode for windows of any length: steps a6-a7 of DESIGN.md section 1 on sky-sorted batches.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// The samples of a chunk arrive bucketed by sky cell (sky_sort.cu): the 64 samples of a batch have relative shifts
// d_{n,k} = s_k - s_0 = b_k + r_{n,k} with one base b_k per detector and residuals 0 <= r < SKY_E.  Circular window
// (N_tau = N_t), detector-0 time: x_j = sum_k P_k[(j + b_k + r_{n,k}) mod N_t, n], P_k[t, n] = sum_kappa A_k[t, kappa] B_k[kappa, n].
// Time is tiled in blocks of 224 window entries.  Per (block, detector) a chunk of 256 consecutive operand rows starting at
// row  block start + b_k  of the circularly extended fp16 operand [Q_hi | Q_lo | Q_hi] arrives by one bulk copy (three ring
// slots); 16 warps contract it with the coefficient operand [B_hi | B_hi | B_lo] of the batch (reading B8: fp16 pieces,
// products exact in the fp32 accumulator) by mma.sync.m16n8k16 -- 4 row tiles x 2 sample tiles per warp, A fragments by
// ldmatrix from rows whose 16-byte chunks are XOR-swizzled in global memory already; the tiles are stored unshifted into an
// exchange buffer [256 rows][64 samples] (32-byte groups swizzled by row: conflict-free 8-byte stores); after a barrier
// every thread adds  P_k[j + r_{n,k}][n]  for its sample n (= lane: one bank per lane whatever the shifts) and its 28 window
// entries j = 8 e + warp/2 of the block into registers.  After the last detector the block joins the thread's running
// (max, sum) of 2^(c log2e (x - max)) -- an on-line log-sum-exp, so the window never exists anywhere as a whole.
// Nothing but Q rows, 23 KB of coefficients per batch and one lnL per sample moves through L2 / HBM.
#include <cuda_fp16.h>

#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

constexpr int SKY_WARPS = 16, SKY_THREADS = SKY_WARPS * 32, SKY_SLOTS = 3;
constexpr int SKY_NE = SKY_TBO / 8;                 // window entries per thread and time block
constexpr float SKY_BSCALE = 8192.f;               // 2^13: scale of the coefficient operand (|F_k Y_lm| < 2) into the fp16 range

struct SkySmem {                                   // byte offsets inside dynamic shared memory
  uint32_t bars, cl2, cval, qval, orig, resid, bk, part, bs, bs_pitch, xb, ring, slot_bytes, total;
};

__host__ __device__ inline SkySmem sky_smem(const SkyPlan &p) {
  SkySmem L;
  L.bars = 0;                                                          // full[3]
  L.cl2 = 64;                                                          // float [64]
  L.cval = L.cl2 + SKY_NB * 4;                                         // double [64] c = D_ref / D
  L.qval = L.cval + SKY_NB * 8;                                        // double [64] q
  L.orig = L.qval + SKY_NB * 8;                                        // int [64] caller's sample (chunk-local), -1 = padding
  L.resid = L.orig + SKY_NB * 4;                                       // int [K][64] residual shifts
  L.bk = L.resid + (uint32_t)p.K * SKY_NB * 4;                         // int [8] base shifts, [8] = intrinsic point
  L.part = (L.bk + 64 + 15u) & ~15u;                                   // float2 [8][64] per-warp-pair (max, sum)
  L.bs = (L.part + 8 * SKY_NB * 8 + 127u) & ~127u;                     // fp16 [K][64][bs_pitch / 2]
  L.bs_pitch = (uint32_t)p.kp * 2 + 16;                                // + 16 bytes: fragment loads of 8 samples hit 32 banks
  L.xb = (L.bs + (uint32_t)p.K * SKY_NB * L.bs_pitch + 127u) & ~127u;  // float [256][64]
  L.ring = L.xb + SKY_TBR * SKY_NB * 4;
  L.slot_bytes = SKY_TBR * (uint32_t)p.rowb;
  L.total = L.ring + SKY_SLOTS * L.slot_bytes;
  return L;
}

struct SkyArgs {
  SkyPlan p;
  SkySmem L;
  const unsigned char *q;          // [P][K][rows_ext][rowb] fp16, 16-byte chunks swizzled by (row & 7) inside 128-byte segments
  const float *qscale;             // [P] power-of-two scale of each point's Q
  Batch b;
  Workspace ws;                    // sorted slots: coef (fp32), scale_c, quad, shift, orig
  const int32_t *n_batches;        // device: batches of SKY_NB slots
  double *lnL_out;
};

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void hmma(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

template <int KS>
__global__ void __launch_bounds__(SKY_THREADS, 1) lnl_sky_kernel(const SkyArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const SkyPlan &P = A.p;
  const SkySmem &L = A.L;
  const Batch &b = A.b;
  const Workspace &ws = A.ws;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + L.bars);
  float *cl2_s = reinterpret_cast<float *>(smem_raw + L.cl2);
  double *cval_s = reinterpret_cast<double *>(smem_raw + L.cval);
  double *qval_s = reinterpret_cast<double *>(smem_raw + L.qval);
  int *orig_s = reinterpret_cast<int *>(smem_raw + L.orig);
  int *resid_s = reinterpret_cast<int *>(smem_raw + L.resid);
  int *bk_s = reinterpret_cast<int *>(smem_raw + L.bk);
  float2 *part_s = reinterpret_cast<float2 *>(smem_raw + L.part);
  unsigned char *bs = smem_raw + L.bs;
  unsigned char *xb = smem_raw + L.xb;
  unsigned char *ring = smem_raw + L.ring;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K = P.K, n_t = P.n_t, km2 = 2 * P.M * K, m2 = 2 * P.M;
  if (tid == 0)
    for (int i = 0; i < SKY_SLOTS; ++i) mbar_init(full + i, 1);
  __syncthreads();

  // MMA role: sample tiles 2 np, 2 np + 1; row tiles rg + 4 i
  const int g = lane >> 2, t4 = lane & 3, np = warp & 3, rg = warp >> 2;
  const uint32_t xb_u32 = smem_u32(xb), ring_u32 = smem_u32(ring);
  // ldmatrix row of this lane inside a 16-row tile, and its 16-byte chunk inside a k-step
  const int lm_row = (lane & 7) + 8 * ((lane >> 3) & 1), lm_chunk = lane >> 4;
  // store role: rows 16 rt + g (+ 8), columns 8 nt + 2 t4 (+ 1); the 32-byte groups of a row are XORed with row & 7 = g
  const uint32_t st0 = (uint32_t)(16 * rg + g) * 256u + (uint32_t)(((2 * np) ^ g) * 32 + t4 * 8);
  const uint32_t st1 = (uint32_t)(16 * rg + g) * 256u + (uint32_t)(((2 * np + 1) ^ g) * 32 + t4 * 8);
  // reader role: sample n_mine = 32 (warp & 1) + lane, window entries ph + 8 e of the block
  const int n_mine = 32 * (warp & 1) + lane, ph = warp >> 1;
  const double ln_ntau = log((double)n_t);
  const int n_chunks = P.n_blocks * K;

  const int total_batches = *A.n_batches;
  const int bt_begin = (int)(((int64_t)total_batches * blockIdx.x) / gridDim.x);
  const int bt_end = (int)(((int64_t)total_batches * (blockIdx.x + 1)) / gridDim.x);
  uint32_t cnt = 0;                                              // chunks consumed so far (ring position and phase)

  for (int bt = bt_begin; bt < bt_end; ++bt) {
    const int64_t slot0 = (int64_t)bt * SKY_NB;
    // ---- stage the batch
    if (tid < 8) bk_s[tid] = INT32_MAX;
    __syncthreads();                                             // previous batch fully consumed; bk reset
    if (tid < SKY_NB) {
      const int o = ws.orig[slot0 + tid];
      orig_s[tid] = o;
      cval_s[tid] = ws.scale_c[slot0 + tid];
      qval_s[tid] = ws.quad[slot0 + tid];
    }
    if (tid == 0) {
      const int o0 = ws.orig[slot0];                             // the first slot of a batch is never padding
      bk_s[8] = b.ids[(b.g0 + (o0 < 0 ? 0 : o0)) / b.n_per_seg];
    }
    int my_d = INT32_MAX;
    if (tid < SKY_NB * K) {
      const int k = tid / SKY_NB, n = tid - k * SKY_NB;
      const int sk = ws.shift[(slot0 + n) * K + k];
      if (sk != INT32_MAX) {
        my_d = sk - ws.shift[(slot0 + n) * K];
        atomicMin(bk_s + k, my_d);
      }
    }
    // coefficient operand [B_hi | B_hi | B_lo] as fp16 rows of kp elements per (detector, sample)
    for (int idx = tid; idx < SKY_NB * K * P.kp; idx += SKY_THREADS) {
      const int kap = idx % P.kp, nk = idx / P.kp, k = nk % K, n = nk / K;
      __half h = __float2half_rn(0.f);
      const int region = kap / m2;
      if (region < 3) {
        const float v = reinterpret_cast<const float *>(ws.coef)[(slot0 + n) * ws.coef_stride + k * m2 + (kap - region * m2)] * SKY_BSCALE;
        const __half hi = __float2half_rn(v);
        h = region < 2 ? hi : __float2half_rn(v - __half2float(hi));
      }
      *reinterpret_cast<__half *>(bs + (size_t)(k * SKY_NB + n) * L.bs_pitch + kap * 2) = h;
    }
    __syncthreads();
    const int point = bk_s[8];
    if (tid < SKY_NB * K) {
      int r = my_d == INT32_MAX ? 0 : my_d - bk_s[tid / SKY_NB];
      r = r < 0 ? 0 : (r > SKY_E - 1 ? SKY_E - 1 : r);           // out of range only for a sample with NaN angles
      resid_s[tid] = r;
    }
    if (tid < SKY_NB) cl2_s[tid] = (float)(cval_s[tid] * 1.4426950408889634 / ((double)A.qscale[point] * SKY_BSCALE));
    const unsigned char *qpoint = A.q + (int64_t)point * P.point_stride;
    auto issue = [&](int i, uint32_t c) {                        // chunk i = (block i / K, detector i % K) into ring slot c % 3
      const int blk = i / K, k = i - blk * K;
      const int bk = bk_s[k] == INT32_MAX ? 0 : bk_s[k];
      const int64_t row = (int64_t)k * P.rows_ext + P.R0 + blk * SKY_TBO + bk;
      const uint32_t slot = c % SKY_SLOTS;
      mbar_expect_tx(full + slot, L.slot_bytes);
      bulk_g2s(ring + slot * L.slot_bytes, qpoint + row * P.rowb, L.slot_bytes, full + slot);
    };
    if (tid == 0)
      for (int i = 0; i < SKY_SLOTS && i < n_chunks; ++i) issue(i, cnt + i);
    __syncthreads();

    float m_run = -INFINITY, s_run = 0.f;
    const float cl2n = cl2_s[n_mine];
    for (int blk = 0; blk < P.n_blocks; ++blk) {
      float x[SKY_NE];
      for (int k = 0; k < K; ++k, ++cnt) {
        const int i = blk * K + k;
        const uint32_t slot = cnt % SKY_SLOTS;
        // ---- coefficient fragments of this detector for the warp's two sample tiles
        uint32_t bf[KS][2][2];
#pragma unroll
        for (int s = 0; s < KS; ++s)
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const unsigned char *p = bs + (size_t)(k * SKY_NB + 8 * (2 * np + j) + g) * L.bs_pitch + (16 * s + 2 * t4) * 2;
            bf[s][j][0] = *reinterpret_cast<const uint32_t *>(p);
            bf[s][j][1] = *reinterpret_cast<const uint32_t *>(p + 16);
          }
        mbar_wait(full + slot, (cnt / SKY_SLOTS) & 1u);
        // the chunk's first row in the extended operand decides the swizzle of its rows
        const int bkk = bk_s[k] == INT32_MAX ? 0 : bk_s[k];
        const int rs = P.R0 + blk * SKY_TBO + bkk;
        const uint32_t sw = (uint32_t)((rs + lane) & 7);
        const uint32_t a_base = ring_u32 + slot * L.slot_bytes + (uint32_t)(16 * rg + lm_row) * (uint32_t)P.rowb;
        float acc[4][2][4];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int j = 0; j < 2; ++j) acc[ii][j][0] = acc[ii][j][1] = acc[ii][j][2] = acc[ii][j][3] = 0.f;
#pragma unroll
        for (int s = 0; s < KS; ++s) {
          const uint32_t c = 2 * s + lm_chunk;
          const uint32_t coff = (c >> 3) * 128u + (((c & 7u) ^ sw) << 4);
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            uint32_t af[4];
            ldsm_x4(a_base + (uint32_t)(64 * ii) * (uint32_t)P.rowb + coff, af);
            hmma(acc[ii][0], af, bf[s][0][0], bf[s][0][1]);
            hmma(acc[ii][1], af, bf[s][1][0], bf[s][1][1]);
          }
        }
        __syncthreads();                                         // every reader is done with the previous detector's rows
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) {
          unsigned char *d = xb + ii * (64 * 256);
          *reinterpret_cast<float2 *>(d + st0) = make_float2(acc[ii][0][0], acc[ii][0][1]);
          *reinterpret_cast<float2 *>(d + st0 + 2048) = make_float2(acc[ii][0][2], acc[ii][0][3]);
          *reinterpret_cast<float2 *>(d + st1) = make_float2(acc[ii][1][0], acc[ii][1][1]);
          *reinterpret_cast<float2 *>(d + st1 + 2048) = make_float2(acc[ii][1][2], acc[ii][1][3]);
        }
        __syncthreads();                                         // the rows of detector k are complete; chunk i is consumed
        if (tid == 0 && i + SKY_SLOTS < n_chunks) issue(i + SKY_SLOTS, cnt + SKY_SLOTS);
        // ---- shifted read: x_j += P_k[j + r][n], lane = sample: one bank per lane
        {
          const int row = ph + resid_s[k * SKY_NB + n_mine];
          const unsigned char *src = xb + (uint32_t)row * 256u + (uint32_t)((((n_mine >> 3) ^ (row & 7)) << 5) + ((n_mine & 7) << 2));
          if (k == 0) {
#pragma unroll
            for (int e = 0; e < SKY_NE; ++e) x[e] = *reinterpret_cast<const float *>(src + e * 2048);
          } else {
#pragma unroll
            for (int e = 0; e < SKY_NE; ++e) x[e] += *reinterpret_cast<const float *>(src + e * 2048);
          }
        }
      }
      // ---- the block joins the running log-sum-exp of this thread
      const int j0 = blk * SKY_TBO + ph;
      float bm = -INFINITY;
#pragma unroll
      for (int e = 0; e < SKY_NE; ++e)
        if (j0 + 8 * e < n_t) bm = fmaxf(bm, x[e]);
      const float m_new = fmaxf(m_run, bm);
      float s = s_run * fast_exp2((m_run - m_new) * cl2n);
      if (m_run == -INFINITY) s = 0.f;
#pragma unroll
      for (int e = 0; e < SKY_NE; ++e)
        if (j0 + 8 * e < n_t) s += fast_exp2((x[e] - m_new) * cl2n);
      s_run = s;
      m_run = m_new;
    }
    part_s[ph * SKY_NB + n_mine] = make_float2(m_run, s_run);
    __syncthreads();
    if (tid < SKY_NB && orig_s[tid] >= 0) {
      float m = -INFINITY;
#pragma unroll
      for (int p8 = 0; p8 < 8; ++p8) m = fmaxf(m, part_s[p8 * SKY_NB + tid].x);
      const float c2 = cl2_s[tid];
      float s = 0.f;
#pragma unroll
      for (int p8 = 0; p8 < 8; ++p8) {
        const float2 v = part_s[p8 * SKY_NB + tid];
        if (v.x > -INFINITY) s += v.y * fast_exp2((v.x - m) * c2);
      }
      const double c = cval_s[tid];
      const double inv = 1.0 / ((double)A.qscale[point] * SKY_BSCALE);
      A.lnL_out[b.g0 + orig_s[tid]] = c * ((double)m * inv) + log((double)s) - ln_ntau - qval_s[tid];
    }
  }
}

// ---- create-time operand: per point scale, then rows [Q_hi | Q_lo | Q_hi] with swizzled 16-byte chunks
__global__ void sky_absmax_kernel(const double *__restrict__ q, int64_t per_point, int64_t n, uint32_t *__restrict__ mx) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    atomicMax(mx + i / per_point, __float_as_uint(fabsf((float)q[i])));
}
__global__ void sky_scale_kernel(const uint32_t *__restrict__ mx, float *__restrict__ scale, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float m = __uint_as_float(mx[i]);
  // a power of two that puts max |Q| into [2^13, 2^14): the fp16 pieces hi + lo then carry 22 bits of every value
  scale[i] = (m > 0.f && m < 3.0e38f) ? exp2f(13.f - floorf(log2f(m))) : 1.f;
}
__global__ void convert_q_sky_kernel(const double2 *__restrict__ src, __half *__restrict__ dst, const float *__restrict__ scale,
                                     SkyPlan p, int64_t total) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int kap = (int)(i % p.kp);
    const int64_t rowi = i / p.kp;
    const int r = (int)(rowi % p.rows_ext);
    const int64_t pk = rowi / p.rows_ext;                                  // point * K + detector
    int t = (r - p.R0) % p.n_t;
    if (t < 0) t += p.n_t;
    const int m2 = 2 * p.M, region = kap / m2;
    __half h = __float2half_rn(0.f);
    if (region < 3) {
      const int kk = kap - region * m2;
      const double2 v2 = src[(pk * p.M + (kk >> 1)) * p.n_t + t];
      const float v = (float)(((kk & 1) ? v2.y : v2.x) * (double)scale[pk / p.K]);
      const __half hi = __float2half_rn(v);
      h = region == 1 ? __float2half_rn(v - __half2float(hi)) : hi;
    }
    const int c = kap >> 3;
    const int pos = (c >> 3) * 64 + (((c & 7) ^ (r & 7)) << 3) + (kap & 7);
    dst[rowi * p.kp + pos] = h;
  }
}

}  // namespace

size_t lnl_sky_smem_bytes(const SkyPlan &p) { return sky_smem(p).total; }

cudaError_t launch_convert_q_sky(const double *Q_c128, void *dst, float *qscale, const SkyPlan &p, int32_t n_points,
                                 cudaStream_t s) {
  const int64_t per_point = (int64_t)p.K * p.M * p.n_t * 2, n_src = per_point * n_points;
  cudaError_t e = cudaMemsetAsync(qscale, 0, sizeof(float) * n_points, s);
  if (e != cudaSuccess) return e;
  sky_absmax_kernel<<<148 * 8, 256, 0, s>>>(Q_c128, per_point, n_src, reinterpret_cast<uint32_t *>(qscale));
  sky_scale_kernel<<<(n_points + 127) / 128, 128, 0, s>>>(reinterpret_cast<const uint32_t *>(qscale), qscale, n_points);
  const int64_t total = (int64_t)n_points * p.K * p.rows_ext * p.kp;
  convert_q_sky_kernel<<<148 * 16, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), reinterpret_cast<__half *>(dst), qscale,
                                                p, total);
  return cudaGetLastError();
}

cudaError_t launch_lnl_sky(const SkyPlan &p, const void *q, const float *qscale, const Batch &b, const Workspace &ws,
                           const int32_t *n_batches_dev, int64_t max_batches, double *lnL_out, int n_sm, cudaStream_t s,
                           int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  SkyArgs a;
  a.p = p;
  a.L = sky_smem(p);
  a.q = reinterpret_cast<const unsigned char *>(q);
  a.qscale = qscale;
  a.b = b;
  a.ws = ws;
  a.n_batches = n_batches_dev;
  a.lnL_out = lnL_out;
  void (*kern)(SkyArgs) = nullptr;
  switch (p.ks) {
    case 4: kern = lnl_sky_kernel<4>; break;
    case 8: kern = lnl_sky_kernel<8>; break;
    default: return cudaErrorInvalidValue;
  }
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)a.L.total);
  if (e != cudaSuccess) return e;
  int64_t grid = n_sm;
  if (grid > max_batches) grid = max_batches;
  if (grid < 1) grid = 1;
  kern<<<(unsigned)grid, SKY_THREADS, a.L.total, s>>>(a);
  if (n_launch) ++*n_launch;
  return cudaGetLastError();
}
