// Fused lnL kernel, tensor-core variant (tcgen05 / TMEM): steps a6-a7 of DESIGN.md section 1 in mixed precision.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// The contraction over the modes is a GEMM per detector in UNSHIFTED detector time,
//     P_k[t, n] = sum_kappa Q'_k[t, kappa] B'_k[kappa, n],     t = 0..N_t-1 (rows, M of the UMMA), n = 16 samples (N),
// with fp32-level accuracy from two TF32 pieces per operand (hi + lo; the lo*lo product is dropped): the A operand
// Q' = [Q_hi | Q_lo] (ka columns) lives in TENSOR MEMORY for the whole intrinsic point, the B operands
// B1 = [B_hi | B_hi], B2 = [B_lo | 0] come from shared memory (bulk-copied batch blobs written by the geometry kernel),
// accumulators P_k (K detectors x nt row tiles x 16 columns) are in TMEM.  In circular mode (N_tau = N_t) the time
// marginal is invariant under a common rotation, so with t = (j + s_0) mod N_t
//     x[t] = P_0[t] + sum_{k>=1} P_k[(t + d_k) mod N_t],     d_k = s_k - s_0  (|d_k| <= dmax_k, light travel time),
// and the per-sample shift is applied by a shared-memory exchange: every epilogue thread owns TMEM lane = row t, writes
// its P_k[t, n] (k >= 1) to Xb[k][n][t + H] (plus wrap-around duplicates inside the halo H) and reads back
// Xb[k][n][t + d_k + H] -- contiguous across lanes, conflict-free.  Each warp then reduces its 32 lanes x nt rows to a
// (reference, sum) pair per sample; the four lane-quarters are combined in fp64 by lnl_tc_finalize_kernel.
//
// Warp roles (320 threads, one CTA per SM): warps 0-3 / 4-7 = two epilogue warpgroups (samples 0-7 / 8-15 of each batch;
// warp w reads TMEM lanes 32 (w%4)..), warp 8 = bulk-copy producer, warp 9 = UMMA issuer (and TMEM allocator).
#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

constexpr int TC_THREADS = 320;
constexpr int TC_STAGES = 3;
constexpr int NH = RIFT_TC_NB / 2;   // samples per epilogue warpgroup

// ---- tcgen05 wrappers ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem descriptor], kind::tf32, issued by one thread
__device__ __forceinline__ void tc_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// K-major, no swizzle: core matrix = 8 rows x 16 bytes, contiguous (128 B).  LBO = byte distance between the two
// 16-byte K chunks of one K=8 step, SBO = byte distance between 8-row groups; version 1 (Blackwell).
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
__device__ __forceinline__ void tc_ld8(uint32_t taddr, float (&r)[8]) {
  uint32_t u[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7])
               : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 8; ++i) r[i] = __uint_as_float(u[i]);
}
// wait for outstanding tcgen05.ld; the registers are tied to the wait so that no use is scheduled above it
__device__ __forceinline__ void tc_wait_ld8(float (&r)[8]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]), "+f"(r[4]), "+f"(r[5]), "+f"(r[6]), "+f"(r[7])::"memory");
}
__device__ __forceinline__ void tc_st8(uint32_t taddr, const float4 &a, const float4 &b) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
               "r"(__float_as_uint(a.x)), "r"(__float_as_uint(a.y)), "r"(__float_as_uint(a.z)), "r"(__float_as_uint(a.w)),
               "r"(__float_as_uint(b.x)), "r"(__float_as_uint(b.y)), "r"(__float_as_uint(b.z)), "r"(__float_as_uint(b.w))
               : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int n_threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}

struct TcArgs {
  TcPlan tp;
  TcChunk ch;
  const float *qtc;              // [P][K][nt*128][ka] tf32 words
};

// instruction descriptor: D fp32, A/B tf32, both K-major, N = 16, M = 128
constexpr uint32_t TC_IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(RIFT_TC_NB >> 3) << 17) | ((128u >> 4) << 24);

__global__ void __launch_bounds__(TC_THREADS, 1) lnl_tc_kernel(const TcArgs args) {
  const TcPlan &tp = args.tp;
  const TcChunk &ch = args.ch;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar_full = reinterpret_cast<uint64_t *>(smem_raw);            // [TC_STAGES]  blob landed
  uint64_t *bar_empty = bar_full + TC_STAGES;                             // [TC_STAGES]  blob consumed by the epilogue
  uint64_t *bar_tfull = bar_empty + TC_STAGES;                            // accumulators ready
  uint64_t *bar_tempty = bar_tfull + 1;                                   // accumulators drained
  uint32_t *tmem_ptr_s = reinterpret_cast<uint32_t *>(smem_raw + 96);
  float *blob_s = reinterpret_cast<float *>(smem_raw + 128);
  float *xb_s = blob_s + TC_STAGES * tp.blob_words;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K = tp.K, nt = tp.nt, ka = tp.ka;

  if (threadIdx.x == 0) {
    for (int i = 0; i < TC_STAGES; ++i) {
      mbar_init(bar_full + i, 1);
      mbar_init(bar_empty + i, 8);
    }
    mbar_init(bar_tfull, 1);
    mbar_init(bar_tempty, 8);
  }
  if (warp == 9) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_s)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr_s;

  const int64_t b_begin = (ch.n_batches * blockIdx.x) / gridDim.x;
  const int64_t b_end = (ch.n_batches * (blockIdx.x + 1)) / gridDim.x;
  uint32_t it = 0;                                                        // batches done by this CTA (all roles in step)
  int staged_point = -1;

  for (int64_t b0 = b_begin; b0 < b_end;) {
    const int64_t seg = (ch.gb0 + b0) / ch.nbps;
    const int64_t job_end = min(b_end, (seg + 1) * ch.nbps - ch.gb0);
    const int point = ch.ids[seg];
    const uint32_t nb = (uint32_t)(job_end - b0);

    // ---- the A operand of this intrinsic point -> tensor memory (thread = TMEM lane = row of the tile)
    __syncthreads();                       // every role is done with the previous job (all UMMAs have completed)
    if (point != staged_point && warp < 4) {
      const int rows = nt * 128;
      for (int k = 0; k < K; ++k)
        for (int i = 0; i < nt; ++i) {
          const int row = 128 * i + 32 * warp + lane;
          const float4 *src = reinterpret_cast<const float4 *>(args.qtc + (((int64_t)point * K + k) * rows + row) * ka);
          const uint32_t taddr = tmem_base + ((uint32_t)(32 * warp) << 16) + (uint32_t)((k * nt + i) * ka);
          for (int c8 = 0; c8 < ka; c8 += 8) {
            const float4 a = __ldg(src + (c8 >> 2)), b = __ldg(src + (c8 >> 2) + 1);
            tc_st8(taddr + c8, a, b);
          }
        }
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    staged_point = point;
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    if (warp == 8) {
      // ===== producer: one bulk copy per batch blob =====
      if (lane == 0) {
        for (uint32_t j = 0; j < nb; ++j) {
          const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
          mbar_wait(bar_empty + stage, ph ^ 1u);
          const uint32_t bytes = (uint32_t)tp.blob_words * 4u;
          mbar_expect_tx(bar_full + stage, bytes);
          bulk_g2s(blob_s + stage * tp.blob_words, ch.blob + (b0 + j) * tp.blob_words, bytes, bar_full + stage);
        }
      }
      __syncwarp();
    } else if (warp == 9) {
      // ===== UMMA issuer =====
      const int n1 = ka >> 3, n2 = tp.kb2 >> 3;                            // K=8 steps of B1, B2
      for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
        mbar_wait(bar_full + stage, ph);
        mbar_wait(bar_tempty, (g & 1u) ^ 1u);
        tc_fence_after();
        if (lane == 0) {
          for (int k = 0; k < K; ++k) {
            const uint32_t b1 = smem_u32(blob_s + stage * tp.blob_words + k * tp.nch * 64);
            const uint32_t b2 = b1 + (uint32_t)(ka >> 2) * 256u;
            for (int i = 0; i < nt; ++i) {
              const uint32_t d_t = tmem_base + (uint32_t)(tp.dcol0 + (k * nt + i) * RIFT_TC_NB);
              const uint32_t a_t = tmem_base + (uint32_t)((k * nt + i) * ka);
              for (int s = 0; s < n1; ++s)
                tc_mma_ts(d_t, a_t + 8 * s, tc_smem_desc(b1 + 512u * s, 256u, 128u), TC_IDESC, s > 0 ? 1u : 0u);
              for (int s = 0; s < n2; ++s)
                tc_mma_ts(d_t, a_t + 8 * s, tc_smem_desc(b2 + 512u * s, 256u, 128u), TC_IDESC, 1u);
            }
          }
          tc_commit(bar_tfull);
        }
        __syncwarp();
      }
    } else {
      // ===== epilogue warpgroups =====
      const int wg = warp >> 2, q = warp & 3;
      const int T = 32 * q + lane;
      const uint32_t lane_addr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(tp.dcol0 + NH * wg);
      const int n_t = tp.n_t, H = tp.H, pitch = tp.pitch;
      for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
        const float *blob = blob_s + stage * tp.blob_words;
        float *xb = xb_s + (size_t)((wg * 2 + (g & 1u)) * (K - 1)) * NH * pitch;
        mbar_wait(bar_full + stage, ph);
        mbar_wait(bar_tfull, g & 1u);
        tc_fence_after();

        // Phase A: P_k (k >= 1) -> exchange buffer, P_0 -> registers
        for (int k = 1; k < K; ++k) {
          const int dm = tp.dmax[k];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            if (i < nt) {
              float r[8];
              tc_ld8(lane_addr + (uint32_t)((k * nt + i) * RIFT_TC_NB), r);
              tc_wait_ld8(r);
              const int t = 128 * i + T;
              if (t < n_t) {
                float *dst = xb + (size_t)(k - 1) * NH * pitch + t + H;
#pragma unroll
                for (int n = 0; n < NH; ++n) dst[n * pitch] = r[n];
                if (t < dm) {
#pragma unroll
                  for (int n = 0; n < NH; ++n) dst[n * pitch + n_t] = r[n];
                }
                if (t >= n_t - dm) {
#pragma unroll
                  for (int n = 0; n < NH; ++n) dst[n * pitch - n_t] = r[n];
                }
              }
            }
          }
        }
        float x[4][NH];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          if (i < nt) {
            tc_ld8(lane_addr + (uint32_t)(i * RIFT_TC_NB), x[i]);
          } else {
#pragma unroll
            for (int n = 0; n < NH; ++n) x[i][n] = 0.f;
          }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) tc_wait_ld8(x[i]);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty);                            // the UMMAs of the next batch may overwrite D
        named_bar_sync(1 + wg, 128);                                       // exchange rows of this warpgroup are complete

        // Phase B: shifted sum over detectors, then per-warp (reference, sum) of the time marginal
        const int32_t *dsh = reinterpret_cast<const int32_t *>(blob + K * tp.nch * 64);
        const float *cl2s = blob + K * tp.nch * 64 + K * 16;
        float2 *part = ch.part + ((b0 + j) * RIFT_TC_NB + NH * wg) * 4 + q;
#pragma unroll
        for (int n = 0; n < NH; ++n) {
          for (int k = 1; k < K; ++k) {
            const int d = dsh[k * 16 + NH * wg + n];
            const float *src = xb + (size_t)((k - 1) * NH + n) * pitch + T + H + d;
#pragma unroll
            for (int i = 0; i < 4; ++i)
              if (128 * i + T < n_t) x[i][n] += src[128 * i];
          }
          float m = -INFINITY;
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            if (128 * i + T >= n_t) x[i][n] = -INFINITY;
            m = fmaxf(m, x[i][n]);
          }
          m = warp_max(m);
          const float cl2 = cl2s[NH * wg + n];
          // reference in log2 units, rounded once: sum_j 2^(x_j cl2 - off) = 2^res sum_j 2^((x_j - m) cl2), res = m cl2 - off
          const float off = (m == -INFINITY) ? 0.f : m * cl2;
          const float res = (m == -INFINITY) ? 0.f : fmaf(m, cl2, -off);
          float s = 0.f;
#pragma unroll
          for (int i = 0; i < 4; ++i) s += fast_exp2(fmaf(x[i][n], cl2, -off));
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
          if (lane == 0) part[n * 4] = make_float2(m, s * fast_exp2(-res));
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + stage);
      }
    }
    it += nb;
    b0 = job_end;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 9) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

// Combine the four lane-quarter partials of every sample (fp64): lnL = c M + ln sum_q s_q exp(c (m_q - M)) - ln N - quad
__global__ void lnl_tc_finalize_kernel(TcPlan tp, TcChunk ch, double *__restrict__ lnL_out) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= ch.n_batches * RIFT_TC_NB) return;
  const int64_t gb = ch.gb0 + w / RIFT_TC_NB;
  const int64_t seg = gb / ch.nbps;
  const int64_t i = (gb % ch.nbps) * RIFT_TC_NB + (w % RIFT_TC_NB);
  if (i >= ch.n_per_seg) return;
  const float4 *p = reinterpret_cast<const float4 *>(ch.part + w * 4);
  const float4 p0 = p[0], p1 = p[1];
  const double m[4] = {p0.x, p0.z, p1.x, p1.z}, s[4] = {p0.y, p0.w, p1.y, p1.w};
  const double c = ch.scale_c[w];
  double mm = -INFINITY;
  for (int a = 0; a < 4; ++a) mm = fmax(mm, m[a]);
  double sum = 0.0;
  for (int a = 0; a < 4; ++a)
    if (m[a] > -INFINITY) sum += s[a] * exp(c * (m[a] - mm));
  lnL_out[seg * ch.n_per_seg + i] = c * mm + log(sum) - log((double)tp.n_t) - ch.quad[w];
}

// Q [P][K][M][n_t] complex128  ->  A operand [P][K][nt*128][ka] tf32 words: columns [0, kh) = hi(Re, Im interleaved),
// [kh, 2 kh) = lo, zero padding; rows >= n_t are zero.
__global__ void convert_q_tc_kernel(const double2 *__restrict__ src, float *__restrict__ dst, TcPlan tp, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const int col = (int)(idx % tp.ka);
    const int64_t r = idx / tp.ka;
    const int rows = tp.nt * 128;
    const int t = (int)(r % rows);
    const int64_t pk = r / rows;                                           // point * K + k
    const int part = col / tp.kh, kap = col % tp.kh;
    float v = 0.f;
    if (t < tp.n_t && part < 2 && kap < 2 * tp.M) {
      const double2 qv = src[(pk * tp.M + (kap >> 1)) * tp.n_t + t];
      const double x = (kap & 1) ? qv.y : qv.x;
      uint32_t u = __float_as_uint((float)x);
      u += 0xFFFu + ((u >> 13) & 1u);
      u &= 0xFFFFE000u;
      const float hi = __uint_as_float(u);
      if (part == 0) {
        v = hi;
      } else {
        uint32_t ul = __float_as_uint((float)(x - (double)hi));
        ul += 0xFFFu + ((ul >> 13) & 1u);
        ul &= 0xFFFFE000u;
        v = __uint_as_float(ul);
      }
    }
    dst[idx] = v;
  }
}

}  // namespace

size_t lnl_tc_smem_bytes(const TcPlan &tp) {
  return 128 + (size_t)TC_STAGES * tp.blob_words * 4 + (size_t)4 * (tp.K - 1) * NH * tp.pitch * 4;
}

cudaError_t launch_convert_q_tc(const double *Q_c128, float *dst, const TcPlan &tp, int32_t n_points, cudaStream_t s) {
  const int64_t total = (int64_t)n_points * tp.K * tp.nt * 128 * tp.ka;
  if (total <= 0) return cudaSuccess;
  int64_t grid = (total + 255) / 256;
  if (grid > 148 * 32) grid = 148 * 32;
  convert_q_tc_kernel<<<(unsigned)grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), dst, tp, total);
  return cudaGetLastError();
}

cudaError_t launch_lnl_tc(const TcPlan &tp, const float *qtc, const TcChunk &c, double *lnL_out, int n_sm,
                          cudaStream_t s, int *n_launch) {
  if (c.n_batches <= 0) return cudaSuccess;
  const size_t smem = lnl_tc_smem_bytes(tp);
  cudaError_t e = cudaFuncSetAttribute(lnl_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  TcArgs a;
  a.tp = tp;
  a.ch = c;
  a.qtc = qtc;
  int64_t grid = n_sm;
  if (grid > c.n_batches) grid = c.n_batches;
  lnl_tc_kernel<<<(unsigned)grid, TC_THREADS, smem, s>>>(a);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const int64_t n = c.n_batches * RIFT_TC_NB;
  lnl_tc_finalize_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(tp, c, lnL_out);
  if (n_launch) *n_launch += 2;
  return cudaGetLastError();
}
