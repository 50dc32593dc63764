// Fused lnL kernel, tensor-core variant (tcgen05 / TMEM): steps a6-a7 of DESIGN.md section 1 in mixed precision.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// The contraction over the modes is a GEMM per detector in UNSHIFTED detector time,
//     P_k[t, n] = sum_kappa Q'_k[t, kappa] B'_k[kappa, n],     t = 0..N_t-1 (rows, M of the UMMA), n = 16 samples (N),
// with fp32-level accuracy from two fp16 pieces per operand (hi + lo, 11 significant bits each, operands pre-scaled by
// powers of two into the fp16 range; the lo*lo product is dropped; accumulation in fp32): the A operand
// Q' = [Q_hi | Q_lo | Q_hi] (kp elements) lives in TENSOR MEMORY for the whole intrinsic point, the B operand
// B' = [B_hi | B_hi | B_lo] comes from shared memory (bulk-copied batch blobs written by the geometry kernel),
// accumulators P_k (K detectors x nt row tiles x 16 columns) are in TMEM.  In circular mode (N_tau = N_t) the time
// marginal is invariant under a common rotation (in guard-band mode, N_tau < N_t, nothing wraps and rows outside the
// window [j0 + s_0, j0 + s_0 + N_tau) are masked), so with t = (j0 + j + s_0) mod N_t
//     x[t] = P_0[t] + sum_{k>=1} P_k[(t + d_k) mod N_t],     d_k = s_k - s_0  (|d_k| <= dmax_k, light travel time),
// and the per-sample shift is applied by a shared-memory exchange: every epilogue thread owns TMEM lane = row t, writes
// its P_k[t, n] (k >= 1) to Xb[k][n][t + H] (plus wrap-around duplicates inside the halo H) and reads back
// Xb[k][n][t + d_k + H] -- contiguous across lanes, conflict-free.  Each warp then reduces its 32 lanes x nt rows to a
// (reference, sum) pair per sample; the four lane-quarters are combined in fp64 by lnl_tc_finalize_kernel.
//
// Warp roles (320 threads, one CTA per SM): warps 0-3 / 4-7 = two epilogue warpgroups (samples 0-7 / 8-15 of each batch;
// warp w reads TMEM lanes 32 (w%4)..), warp 8 = bulk-copy producer, warp 9 = UMMA issuer (and TMEM allocator).
#include <cuda_fp16.h>

#include "tc_common.cuh"

namespace {

constexpr int TC_THREADS = 384;       // 8 epilogue warps, producer, UMMA issuer, 2 idle warps completing the third warpgroup
constexpr int TC_STAGES = 3;
constexpr int NH = RIFT_TC_NB / 2;   // samples per epilogue warpgroup

struct TcArgs {
  TcPlan tp;
  TcChunk ch;
  const uint32_t *qtc;           // [P][K][nt*128][acols] words of two fp16
};

// NT = row tiles of 128 (ceil(n_t / 128)); PITCH = floats per exchange row (>= n_t + 2 H), compile-time so that the
// exchange addresses are one register plus immediates.
// GUARD = guard-band window (N_tau < N_t): rows outside the window are masked.  PASS = RIFT_TC_PASS_*: with the modes split
// into subsets, every pass but the last writes its window sums x[t, n] to global memory instead of reducing them, every
// pass but the first adds the sums of the pass before.
template <int NT, int PITCH, bool GUARD, int PASS>
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
  const int K = tp.K, acols = tp.acols;

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

  // Jobs = runs of batches of one intrinsic point.  Every role walks the same job list; at a job boundary all warps
  // meet (all UMMAs of the previous job have completed) and warps 0-3 put the A operand of the new point into tensor
  // memory (thread = TMEM lane = row of the tile).
  auto for_each_job = [&](auto &&body) {
    uint32_t it = 0;                                                      // batches done by this CTA (all roles in step)
    int staged_point = -1;
    for (int64_t b0 = b_begin; b0 < b_end;) {
      const int64_t seg = (ch.gb0 + b0) / ch.nbps;
      const int64_t job_end = min(b_end, (seg + 1) * ch.nbps - ch.gb0);
      const int point = ch.ids[seg];
      const uint32_t nb = (uint32_t)(job_end - b0);
      __syncthreads();
      if (point != staged_point && warp < 4) {
        for (int k = 0; k < K; ++k)
          for (int i = 0; i < NT; ++i) {
            const int row = 128 * i + 32 * warp + lane;
            const float4 *src =
                reinterpret_cast<const float4 *>(args.qtc + (((int64_t)point * K + k) * (NT * 128) + row) * acols);
            const uint32_t taddr = tmem_base + ((uint32_t)(32 * warp) << 16) + (uint32_t)((k * NT + i) * acols);
            for (int c8 = 0; c8 < acols; c8 += 8) {
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
      body(point, b0, nb, it);
      it += nb;
      b0 = job_end;
    }
  };

  // Register budget: the service warpgroup (warps 8-11) keeps 40 registers per thread, the epilogue warpgroups take 208.
  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == 8) {
      // ===== producer: one bulk copy per batch blob =====
      for_each_job([&](int, int64_t b0, uint32_t nb, uint32_t it) {
      if (lane == 0) {
        for (uint32_t j = 0; j < nb; ++j) {
          const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
          mbar_wait_idle(bar_empty + stage, ph ^ 1u);
          const uint32_t bytes = (uint32_t)tp.blob_words * 4u;
          mbar_expect_tx(bar_full + stage, bytes);
          bulk_g2s(blob_s + stage * tp.blob_words, ch.blob + (b0 + j) * tp.blob_words, bytes, bar_full + stage);
        }
      }
      __syncwarp();
      });
    } else if (warp == 9) {
      // ===== UMMA issuer =====  (K=16 steps outermost: consecutive UMMAs accumulate into different tiles)
      const int n_steps = tp.kp >> 4;
      for_each_job([&](int, int64_t, uint32_t nb, uint32_t it) {
      for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
        mbar_wait_idle(bar_full + stage, ph);
        mbar_wait_idle(bar_tempty, (g & 1u) ^ 1u);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t desc0 = tc_smem_desc(smem_u32(blob_s + stage * tp.blob_words), 256u, 128u);
          for (int s = 0; s < n_steps; ++s) {
            for (int k = 0; k < K; ++k) {
              const uint64_t desc = desc0 + (uint64_t)((k * tp.nch * 256 + s * 512) >> 4);
#pragma unroll
              for (int i = 0; i < NT; ++i) {
                const uint32_t d_t = tmem_base + (uint32_t)(tp.dcol0 + (k * NT + i) * RIFT_TC_NB);
                const uint32_t a_t = tmem_base + (uint32_t)((k * NT + i) * acols + 8 * s);
                tc_mma_ts(d_t, a_t, desc, TC_IDESC, s > 0 ? 1u : 0u);
              }
            }
          }
          tc_commit(bar_tfull);
        }
        __syncwarp();
      }
      });
    } else {
      for_each_job([](int, int64_t, uint32_t, uint32_t) {});                // idle warps: job-boundary barriers only
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    for_each_job([&](int point, int64_t b0, uint32_t nb, uint32_t it) {
      // ===== epilogue warpgroups =====
      const int wg = warp >> 2, q = warp & 3;
      const int T = 32 * q + lane;
      const uint32_t lane_addr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(tp.dcol0 + NH * wg);
      const int n_t = tp.n_t, H = tp.H;
      const float inv_scale = 1.0f / (ch.qscale[point] * (float)RIFT_TC_BSCALE);   // accumulators carry x / inv_scale
      const bool last_valid = 128 * (NT - 1) + T < n_t;                    // tiles 0..NT-2 are full, the last one ragged
      const int last_clamp = last_valid ? 0 : (n_t - 1) - (128 * (NT - 1) + T);   // row offset that keeps reads in range

      auto load_tiles = [&](int k, float (&r)[NT][NH]) {
#pragma unroll
        for (int i = 0; i < NT; ++i) tc_ld8(lane_addr + (uint32_t)((k * NT + i) * RIFT_TC_NB), r[i]);
      };
      auto wait_tiles = [&](float (&r)[NT][NH]) {
#pragma unroll
        for (int i = 0; i < NT; ++i) tc_wait_ld8(r[i]);
      };
      auto store_tiles = [&](int k, float *xb, const float (&r)[NT][NH]) {
        const int dm = tp.dmax[k];
        float *base = xb + (size_t)(k - 1) * NH * PITCH + T + H;
#pragma unroll
        for (int i = 0; i < NT; ++i) {
          const int t = 128 * i + T;
          if (i < NT - 1 || last_valid) {
            float *dst = base + 128 * i;
#pragma unroll
            for (int n = 0; n < NH; ++n) dst[n * PITCH] = r[i][n];
            if (t < dm) {
              float *dh = dst + n_t;
#pragma unroll
              for (int n = 0; n < NH; ++n) dh[n * PITCH] = r[i][n];
            }
            if (t >= n_t - dm) {
              float *dl = dst - n_t;
#pragma unroll
              for (int n = 0; n < NH; ++n) dl[n * PITCH] = r[i][n];
            }
          }
        }
      };

      // Phase A of batch g (after its accumulators are ready): P_k (k >= 1) -> exchange buffer, P_0 -> registers xd; the
      // loads of the next detector are in flight while the current one is stored.  No spin inside, so that the caller can
      // fuse it with the reduction of the previous batch in one basic block.
      auto phase_a = [&](uint32_t g, float (&xd)[NT][NH]) {
        float *xb = xb_s + (size_t)((wg * 2 + (g & 1u)) * (K - 1)) * NH * PITCH;
        float ra[NT][NH];
        load_tiles(0, xd);                                                 // P_0 stays in registers
        for (int k = 1; k < K; ++k) {
          load_tiles(k, ra);
          wait_tiles(ra);
          store_tiles(k, xb, ra);
        }
        wait_tiles(xd);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty);                            // the UMMAs of the next batch may overwrite D
      };
      // Phase B: shifted sum over detectors
      auto phase_b = [&](uint32_t g, int64_t lb, float (&x)[NT][NH]) {
        float xp[NT][NH];
        if constexpr (PASS == RIFT_TC_PASS_MIDDLE || PASS == RIFT_TC_PASS_LAST) {   // in flight under the exchange reads
          const float *src = ch.xacc + ((size_t)(lb * RIFT_TC_NB + NH * wg)) * (NT * 128) + T;
#pragma unroll
          for (int n = 0; n < NH; ++n)
#pragma unroll
            for (int i = 0; i < NT; ++i) xp[i][n] = __ldcs(src + (size_t)n * (NT * 128) + 128 * i);
        }
        const float *blob = blob_s + (g % TC_STAGES) * tp.blob_words;
        const float *xb = xb_s + (size_t)((wg * 2 + (g & 1u)) * (K - 1)) * NH * PITCH;
        const int32_t *dsh = reinterpret_cast<const int32_t *>(blob + K * tp.nch * 64) + NH * wg;
        for (int k = 1; k < K; ++k) {
          const int4 d0 = *reinterpret_cast<const int4 *>(dsh + k * 16), d1 = *reinterpret_cast<const int4 *>(dsh + k * 16 + 4);
          const int d[NH] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
          const float *base = xb + (size_t)(k - 1) * NH * PITCH + T + H;
#pragma unroll
          for (int n = 0; n < NH; ++n) {
            const float *src = base + d[n] + n * PITCH;
#pragma unroll
            for (int i = 0; i < NT - 1; ++i) x[i][n] += src[128 * i];
            x[NT - 1][n] += src[128 * (NT - 1) + last_clamp];
          }
        }
        if constexpr (PASS == RIFT_TC_PASS_MIDDLE || PASS == RIFT_TC_PASS_LAST) {
#pragma unroll
          for (int n = 0; n < NH; ++n)
#pragma unroll
            for (int i = 0; i < NT; ++i) x[i][n] += xp[i][n];
        }
      };
      // per-warp (reference, sum) of the time marginal for the 8 samples of batch g (chunk-local batch index lb)
      auto reduce = [&](uint32_t g, int64_t lb, float (&x)[NT][NH]) {
        if constexpr (PASS == RIFT_TC_PASS_FIRST || PASS == RIFT_TC_PASS_MIDDLE) {   // hand the window sums to the next pass
          float *dst = ch.xacc + ((size_t)(lb * RIFT_TC_NB + NH * wg)) * (NT * 128) + T;
#pragma unroll
          for (int n = 0; n < NH; ++n)
#pragma unroll
            for (int i = 0; i < NT; ++i) __stcs(dst + (size_t)n * (NT * 128) + 128 * i, x[i][n]);
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_empty + g % TC_STAGES);
          return;
        }
        const uint32_t stage = g % TC_STAGES;
        const float *blob = blob_s + stage * tp.blob_words;
        const float *cl2s = blob + K * tp.nch * 64 + K * 16 + NH * wg;
        float m[NH];
        if constexpr (GUARD) {                // guard-band window: rows outside [j0 + s_0, j0 + s_0 + n_tau) do not count
          const int32_t *lo = reinterpret_cast<const int32_t *>(blob + K * tp.nch * 64) + NH * wg;
#pragma unroll
          for (int n = 0; n < NH; ++n) {
            const int l0 = lo[n];
#pragma unroll
            for (int i = 0; i < NT; ++i)
              if ((unsigned)(128 * i + T - l0) >= (unsigned)tp.n_tau) x[i][n] = -INFINITY;
          }
        }
#pragma unroll
        for (int n = 0; n < NH; ++n) {
          if (!last_valid) x[NT - 1][n] = -INFINITY;
          float mm = x[0][n];
#pragma unroll
          for (int i = 1; i < NT; ++i) mm = fmaxf(mm, x[i][n]);
          m[n] = mm;
        }
        const float mine = treduce8(m, lane, [](float a, float b) { return fmaxf(a, b); });
        const float4 c0 = *reinterpret_cast<const float4 *>(cl2s), c1 = *reinterpret_cast<const float4 *>(cl2s + 4);
        const float cl2[NH] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
        float sums[NH];
#pragma unroll
        for (int n = 0; n < NH; ++n) {
          const float mx = __shfl_sync(0xffffffffu, mine, ((n & 4) << 2) | ((n & 2) << 2) | ((n & 1) << 2));
          // reference in log2 units, rounded once (the residual is corrected below)
          const float off = (mx == -INFINITY) ? 0.f : mx * cl2[n];
          float s = 0.f;
#pragma unroll
          for (int i = 0; i < NT; ++i) s += fast_exp2(fmaf(x[i][n], cl2[n], -off));
          sums[n] = s;
        }
        const float ssum = treduce8(sums, lane, [](float a, float b) { return a + b; });
        if ((lane & 3) == 0) {
          const int nsel = lane >> 2;                                      // = 4 b4 + 2 b3 + b2
          const float cl = cl2s[nsel];
          // sum_j 2^(x_j cl - off) = 2^res sum_j 2^((x_j - m) cl),  res = m cl - off
          const float off = (mine == -INFINITY) ? 0.f : mine * cl;
          const float res = (mine == -INFINITY) ? 0.f : fmaf(mine, cl, -off);
          ch.part[(lb * RIFT_TC_NB + NH * wg + nsel) * 4 + q] = make_float2(mine * inv_scale, ssum * fast_exp2(-res));
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + stage);
      };

      // Software pipeline over the batches of this job: the reduction of batch g (shuffle / exponential latency chains)
      // and Phase A of batch g + 1 (tensor-memory loads, shared-memory stores) are issued from one basic block.
      float x[NT][NH];
      mbar_wait(bar_tfull, it & 1u);
      tc_fence_after();
      phase_a(it, x);
      for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t g = it + j;
        named_bar_sync(1 + wg, 128);                                       // exchange rows of batch g are complete
        mbar_wait(bar_full + g % TC_STAGES, (g / TC_STAGES) & 1u);         // shifts and exponent scales of batch g
        phase_b(g, b0 + j, x);
        if (j + 1 < nb) {
          mbar_wait(bar_tfull, (g + 1u) & 1u);
          tc_fence_after();
          float xn[NT][NH];
          phase_a(g + 1u, xn);
          reduce(g, b0 + j, x);
#pragma unroll
          for (int i = 0; i < NT; ++i)
#pragma unroll
            for (int n = 0; n < NH; ++n) x[i][n] = xn[i][n];
        } else {
          reduce(g, b0 + j, x);
        }
      }
    });
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
  lnL_out[seg * ch.n_per_seg + i] = c * mm + log(sum) - log((double)tp.n_tau) - ch.quad[w];
}

// Per point: max |Re Q|, |Im Q| over detectors, modes, time (bit pattern of the non-negative float, atomicMax)
__global__ void q_absmax_kernel(const double2 *__restrict__ src, uint32_t *__restrict__ mx, int64_t per_point, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const double2 v = src[idx];
    const float a = fmaxf(fabsf((float)v.x), fabsf((float)v.y));
    if (a > 0.f && a < INFINITY) atomicMax(mx + idx / per_point, __float_as_uint(a));
  }
}
// scale[p] = 2^e with scale * max|Q| in [2^13, 2^14)  (1 when the point is all zero)
__global__ void q_scale_kernel(const uint32_t *mx, float *scale, int n_points) {   // in place: mx aliases scale
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_points) return;
  const float a = __uint_as_float(mx[p]);
  int e = 0;
  if (a > 0.f) frexpf(a, &e);                                              // a = f 2^e, f in [0.5, 1)
  scale[p] = (a > 0.f) ? ldexpf(1.0f, 14 - e) : 1.0f;
}

// Q [P][K][M][n_t] complex128  ->  A operand [P][K][nt*128][acols] words of two fp16: contraction index kappa' over
// [Q_hi | Q_lo | Q_hi] (each 2M elements, Re/Im interleaved), zero padding up to kp; rows >= n_t are zero.
__global__ void convert_q_tc_kernel(const double2 *__restrict__ src, uint32_t *__restrict__ dst, const float *__restrict__ scale,
                                    TcPlan tp, int sub, int64_t total) {
  const int ms = tp.m_sub, a0 = sub * tp.m_sub;                            // modes [a0, a0 + ms) of this subset
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const int col = (int)(idx % tp.acols);
    const int64_t r = idx / tp.acols;
    const int rows = tp.nt * 128;
    const int t = (int)(r % rows);
    const int64_t pk = r / rows;                                           // point * K + k
    const double sc = (double)scale[pk / tp.K];
    uint32_t word = 0;
    if (t < tp.n_t) {
      for (int hlf = 0; hlf < 2; ++hlf) {
        const int kp_i = 2 * col + hlf;
        const int part = kp_i / (2 * ms), kap = kp_i % (2 * ms);
        const int a = a0 + (kap >> 1);
        if (part < 3 && a < tp.M) {
          const double2 qv = src[(pk * tp.M + a) * tp.n_t + t];
          const double x = ((kap & 1) ? qv.y : qv.x) * sc;
          const __half hi = __double2half(x);
          const __half out = (part == 1) ? __double2half(x - (double)__half2float(hi)) : hi;
          word |= (uint32_t)__half_as_ushort(out) << (16 * hlf);
        }
      }
    }
    dst[idx] = word;
  }
}

}  // namespace

size_t lnl_tc_smem_bytes(const TcPlan &tp) {
  return 128 + (size_t)TC_STAGES * tp.blob_words * 4 + (size_t)4 * (tp.K - 1) * NH * tp.pitch * 4;
}

// exchange-row pitches the kernel is instantiated for; 0 if n_t + 2 H does not fit any
int lnl_tc_pitch(int n_t, int halo) {
  const int need = n_t + 2 * halo;
  const int opts[4] = {256, 512, 640, 768};
  for (int i = 0; i < 4; ++i)
    if (need <= opts[i]) return opts[i];
  return 0;
}

namespace {
template <int NT>
cudaError_t launch_nt(const TcArgs &a, int pass, unsigned grid, size_t smem, cudaStream_t s) {
#define RIFT_TC_CASE(P)                                                                                          \
  case P: {                                                                                                      \
    void (*kern)(TcArgs) = nullptr;                                                                              \
    if (a.tp.n_tau < a.tp.n_t) {                                                                                 \
      if (pass != RIFT_TC_PASS_SINGLE) return cudaErrorInvalidValue;                                             \
      kern = lnl_tc_kernel<NT, P, true, RIFT_TC_PASS_SINGLE>;                                                    \
    } else {                                                                                                     \
      kern = pass == RIFT_TC_PASS_SINGLE  ? lnl_tc_kernel<NT, P, false, RIFT_TC_PASS_SINGLE>                     \
             : pass == RIFT_TC_PASS_FIRST ? lnl_tc_kernel<NT, P, false, RIFT_TC_PASS_FIRST>                      \
             : pass == RIFT_TC_PASS_MIDDLE ? lnl_tc_kernel<NT, P, false, RIFT_TC_PASS_MIDDLE>                    \
                                           : lnl_tc_kernel<NT, P, false, RIFT_TC_PASS_LAST>;                     \
    }                                                                                                            \
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
    if (e != cudaSuccess) return e;                                                                              \
    kern<<<grid, TC_THREADS, smem, s>>>(a);                                                                      \
    return cudaGetLastError();                                                                                   \
  }
  switch (a.tp.pitch) {
    RIFT_TC_CASE(256)
    RIFT_TC_CASE(512)
    RIFT_TC_CASE(640)
    RIFT_TC_CASE(768)
    default: return cudaErrorInvalidValue;
  }
#undef RIFT_TC_CASE
}
}  // namespace

cudaError_t launch_convert_q_tc(const double *Q_c128, uint32_t *dst, float *qscale, const TcPlan &tp, int32_t n_points,
                                cudaStream_t s) {
  const int64_t total = (int64_t)n_points * tp.K * tp.nt * 128 * tp.acols;
  if (total <= 0) return cudaSuccess;
  const int64_t per_point = (int64_t)tp.K * tp.M * tp.n_t, n_src = per_point * n_points;
  // qscale doubles as the scratch of the max reduction (bit patterns), then holds the scale
  cudaError_t e = cudaMemsetAsync(qscale, 0, sizeof(float) * n_points, s);
  if (e != cudaSuccess) return e;
  int64_t grid = (n_src + 255) / 256;
  if (grid > 148 * 32) grid = 148 * 32;
  q_absmax_kernel<<<(unsigned)grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128),
                                                 reinterpret_cast<uint32_t *>(qscale), per_point, n_src);
  q_scale_kernel<<<(n_points + 127) / 128, 128, 0, s>>>(reinterpret_cast<const uint32_t *>(qscale), qscale, n_points);
  grid = (total + 255) / 256;
  if (grid > 148 * 32) grid = 148 * 32;
  for (int sub = 0; sub < tp.n_sub; ++sub)
    convert_q_tc_kernel<<<(unsigned)grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), dst + (size_t)sub * total,
                                                       qscale, tp, sub, total);
  return cudaGetLastError();
}

cudaError_t launch_lnl_tc(const TcPlan &tp, const uint32_t *qtc, const TcChunk &c, int pass, double *lnL_out, int n_sm,
                          cudaStream_t s, int *n_launch) {
  if (c.n_batches <= 0) return cudaSuccess;
  const size_t smem = lnl_tc_smem_bytes(tp);
  cudaError_t e;
  TcArgs a;
  a.tp = tp;
  a.ch = c;
  a.qtc = qtc;
  int64_t grid = n_sm;
  if (grid > c.n_batches) grid = c.n_batches;
  switch (tp.nt) {
    case 1: e = launch_nt<1>(a, pass, (unsigned)grid, smem, s); break;
    case 2: e = launch_nt<2>(a, pass, (unsigned)grid, smem, s); break;
    case 3: e = launch_nt<3>(a, pass, (unsigned)grid, smem, s); break;
    case 4: e = launch_nt<4>(a, pass, (unsigned)grid, smem, s); break;
    default: e = cudaErrorInvalidValue;
  }
  if (e != cudaSuccess) return e;
  if (n_launch) ++*n_launch;
  if (pass == RIFT_TC_PASS_FIRST || pass == RIFT_TC_PASS_MIDDLE) return cudaSuccess;   // lnL is assembled after the last pass
  const int64_t n = c.n_batches * RIFT_TC_NB;
  lnl_tc_finalize_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(tp, c, lnL_out);
  if (n_launch) ++*n_launch;
  return cudaGetLastError();
}
