// Fused lnL kernel, tensor-core variant with shift-sorted batches (steps a6-a7 of DESIGN.md section 1, mixed precision).
//
// Same contraction, operand split and epilogue as lnl_tc.cu, with one exchange removed: the samples of a chunk are bucketed
// by their relative shift d_1 = s_1 - s_0 (geometry.cu: tcs_key_kernel, tcs_scan_kernel), so that all 16 samples of a batch
// share d_1.  The detector-1 operand Q'_1 then does not have to be shifted per sample: it lives in SHARED memory in the
// K-major, unswizzled UMMA layout with contiguous 8-row groups, i.e. row r of plane c at byte 16 r, extended circularly by
// dmax_1 rows on both sides, and the UMMA of detector 1 simply starts its A operand at row d_1 + dmax_1 + 128 i and
// accumulates onto the detector-0 tile:
//     D_0[t, n] = sum_kappa Q'_0[t, kappa] B'_0[kappa, n] + sum_kappa Q'_1[(t + d_1) mod N_t, kappa] B'_1[kappa, n].
// Detectors k >= 2 keep the per-sample shared-memory exchange of lnl_tc.cu.  For three detectors this halves the
// tensor-memory loads, exchange stores and exchange reads of the epilogue, which bound lnl_tc.
//
// Batches are indexed in sorted order (TcChunk::seg_begin, perm); the number of batches is read from device memory.
#include <cuda_fp16.h>

#include "tc_common.cuh"

namespace {

constexpr int TC_THREADS = 384;       // 8 epilogue warps, producer, UMMA issuer, 2 idle warps completing the third warpgroup
constexpr int TC_STAGES = 3;
constexpr int NH = RIFT_TC_NB / 2;    // samples per epilogue warpgroup

struct TcsArgs {
  TcPlan tp;
  TcChunk ch;
  const uint32_t *qtc;           // [P][K][nt*128][acols] words of two fp16 (detector 1 unused here)
  const uint16_t *qs;            // [P][kp/8][as_rows][8] fp16: extended detector-1 operand
};

// PASS = RIFT_TC_PASS_* as in lnl_tc.cu: with the modes split into subsets, every pass but the last writes its window sums
// x[t, n] to global memory instead of reducing them, every pass but the first adds the sums of the pass before.
template <int NT, int PITCH, bool GUARD, int PASS>
__global__ void __launch_bounds__(TC_THREADS, 1) lnl_tcs_kernel(const TcsArgs args) {
  const TcPlan &tp = args.tp;
  const TcChunk &ch = args.ch;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar_full = reinterpret_cast<uint64_t *>(smem_raw);            // [TC_STAGES]  blob landed
  uint64_t *bar_empty = bar_full + TC_STAGES;                             // [TC_STAGES]  blob consumed by the epilogue
  uint64_t *bar_tfull = bar_empty + TC_STAGES;                            // accumulators ready
  uint64_t *bar_tempty = bar_tfull + 1;                                   // accumulators drained
  uint32_t *tmem_ptr_s = reinterpret_cast<uint32_t *>(smem_raw + 96);
  const int BW = tp.blob_words_s;
  float *blob_s = reinterpret_cast<float *>(smem_raw + 128);
  const int as_words = (tp.kp >> 3) * tp.as_rows * 4;                     // 32-bit words of the detector-1 operand
  uint32_t *as_s = reinterpret_cast<uint32_t *>(blob_s + TC_STAGES * BW);
  float *xb_s = reinterpret_cast<float *>(as_s + as_words);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K = tp.K, acols = tp.acols;
  const int hdr = K * tp.nch * 64 + K * 16 + 16;                           // batch header: d_1

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

  const int64_t n_sorted = ch.seg_begin[ch.n_lseg];
  const int64_t b_begin = (n_sorted * blockIdx.x) / gridDim.x;
  const int64_t b_end = (n_sorted * (blockIdx.x + 1)) / gridDim.x;
  const int64_t seg0 = ch.gb0 / ch.nbps;

  // Jobs = runs of sorted batches of one segment.  At a job boundary all warps meet, warps 0-3 put the A operands of
  // detectors 0 and >= 2 into tensor memory (tile slot 0 and k - 1) and all threads copy the extended detector-1 operand
  // into shared memory.
  auto for_each_job = [&](auto &&body) {
    uint32_t it = 0;
    int staged_point = -1;
    int ls = 0;
    for (int64_t b0 = b_begin; b0 < b_end;) {
      while (ch.seg_begin[ls + 1] <= b0) ++ls;
      const int64_t job_end = min(b_end, (int64_t)ch.seg_begin[ls + 1]);
      const int point = ch.ids[seg0 + ls];
      const uint32_t nb = (uint32_t)(job_end - b0);
      __syncthreads();
      if (point != staged_point) {
        if (warp < 4) {
          for (int k = 0; k < K; ++k) {
            if (k == 1) continue;
            const int ka = k ? k - 1 : 0;
            for (int i = 0; i < NT; ++i) {
              const int row = 128 * i + 32 * warp + lane;
              const float4 *src =
                  reinterpret_cast<const float4 *>(args.qtc + (((int64_t)point * K + k) * (NT * 128) + row) * acols);
              const uint32_t taddr = tmem_base + ((uint32_t)(32 * warp) << 16) + (uint32_t)((ka * NT + i) * acols);
              for (int c8 = 0; c8 < acols; c8 += 8) {
                const float4 a = __ldg(src + (c8 >> 2)), b = __ldg(src + (c8 >> 2) + 1);
                tc_st8(taddr + c8, a, b);
              }
            }
          }
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
        const uint4 *src = reinterpret_cast<const uint4 *>(args.qs) + (int64_t)point * (as_words >> 2);
        uint4 *dst = reinterpret_cast<uint4 *>(as_s);
        for (int i = threadIdx.x; i < (as_words >> 2); i += TC_THREADS) dst[i] = __ldg(src + i);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");       // generic-proxy writes -> UMMA operand reads
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

  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == 8) {
      // ===== producer: one bulk copy per batch blob =====
      for_each_job([&](int, int64_t b0, uint32_t nb, uint32_t it) {
      if (lane == 0) {
        for (uint32_t j = 0; j < nb; ++j) {
          const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
          mbar_wait_idle(bar_empty + stage, ph ^ 1u);
          const uint32_t bytes = (uint32_t)BW * 4u;
          mbar_expect_tx(bar_full + stage, bytes);
          bulk_g2s(blob_s + stage * BW, ch.blob + (b0 + j) * BW, bytes, bar_full + stage);
        }
      }
      __syncwarp();
      });
    } else if (warp == 9) {
      // ===== UMMA issuer =====  (K=16 steps outermost; per step: detector-0 tiles, detector-1 tiles onto the same
      // accumulators from the shifted shared-memory operand, then the exchanged detectors)
      const int n_steps = tp.kp >> 4;
      const uint32_t as_lbo = (uint32_t)tp.as_rows * 16u;                  // bytes between the 16-byte K chunks (planes)
      for_each_job([&](int, int64_t, uint32_t nb, uint32_t it) {
      for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t g = it + j, stage = g % TC_STAGES, ph = (g / TC_STAGES) & 1u;
        mbar_wait_idle(bar_full + stage, ph);
        mbar_wait_idle(bar_tempty, (g & 1u) ^ 1u);
        tc_fence_after();
        if (elect_one()) {
          const float *blob = blob_s + stage * BW;
          const int d1 = reinterpret_cast<const int32_t *>(blob)[hdr];
          const uint64_t desc0 = tc_smem_desc(smem_u32(blob), 256u, 128u);
          const uint64_t adesc0 = tc_smem_desc(smem_u32(as_s) + (uint32_t)(d1 + tp.dmax[1]) * 16u, as_lbo, 128u);
          for (int s = 0; s < n_steps; ++s) {
            const uint64_t descb0 = desc0 + (uint64_t)((s * 512) >> 4);
            const uint64_t descb1 = desc0 + (uint64_t)((tp.nch * 256 + s * 512) >> 4);
#pragma unroll
            for (int i = 0; i < NT; ++i)
              tc_mma_ts(tmem_base + (uint32_t)(tp.dcol0_s + i * RIFT_TC_NB), tmem_base + (uint32_t)(i * acols + 8 * s), descb0,
                        TC_IDESC, s > 0 ? 1u : 0u);
#pragma unroll
            for (int i = 0; i < NT; ++i)
              tc_mma_ss(tmem_base + (uint32_t)(tp.dcol0_s + i * RIFT_TC_NB),
                        adesc0 + (uint64_t)(((uint32_t)(2 * s) * as_lbo + (uint32_t)(128 * i) * 16u) >> 4), descb1, TC_IDESC, 1u);
            for (int k = 2; k < K; ++k) {
              const uint64_t desc = desc0 + (uint64_t)((k * tp.nch * 256 + s * 512) >> 4);
#pragma unroll
              for (int i = 0; i < NT; ++i) {
                const uint32_t d_t = tmem_base + (uint32_t)(tp.dcol0_s + ((k - 1) * NT + i) * RIFT_TC_NB);
                const uint32_t a_t = tmem_base + (uint32_t)(((k - 1) * NT + i) * acols + 8 * s);
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
    int H = 0;                                                              // halo of the exchanged detectors
    for (int k = 2; k < K; ++k) H = max(H, tp.dmax[k]);
    for_each_job([&](int point, int64_t b0, uint32_t nb, uint32_t it) {
      // ===== epilogue warpgroups =====
      const int wg = warp >> 2, q = warp & 3;
      const int T = 32 * q + lane;
      const uint32_t lane_addr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(tp.dcol0_s + NH * wg);
      const int n_t = tp.n_t;
      const float inv_scale = 1.0f / (ch.qscale[point] * (float)RIFT_TC_BSCALE);   // accumulators carry x / inv_scale
      const bool last_valid = 128 * (NT - 1) + T < n_t;                    // tiles 0..NT-2 are full, the last one ragged
      const int last_clamp = last_valid ? 0 : (n_t - 1) - (128 * (NT - 1) + T);   // row offset that keeps reads in range

      auto load_tiles = [&](int kd, float (&r)[NT][NH]) {
#pragma unroll
        for (int i = 0; i < NT; ++i) tc_ld8(lane_addr + (uint32_t)((kd * NT + i) * RIFT_TC_NB), r[i]);
      };
      auto wait_tiles = [&](float (&r)[NT][NH]) {
#pragma unroll
        for (int i = 0; i < NT; ++i) tc_wait_ld8(r[i]);
      };
      auto store_tiles = [&](int k, float *xb, const float (&r)[NT][NH]) {
        const int dm = tp.dmax[k];
        float *base = xb + (size_t)(k - 2) * NH * PITCH + T + H;
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

      // Phase A of batch g: P_k (k >= 2) -> exchange buffer, P_0 + P_1 (shifted) -> registers xd
      auto phase_a = [&](uint32_t g, float (&xd)[NT][NH]) {
        float *xb = xb_s + (size_t)((wg * 2 + (g & 1u)) * (K - 2)) * NH * PITCH;
        float ra[NT][NH];
        load_tiles(0, xd);
        for (int k = 2; k < K; ++k) {
          load_tiles(k - 1, ra);
          wait_tiles(ra);
          store_tiles(k, xb, ra);
        }
        wait_tiles(xd);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty);                            // the UMMAs of the next batch may overwrite D
      };
      // Phase B: shifted sum over the exchanged detectors
      auto phase_b = [&](uint32_t g, int64_t lb, float (&x)[NT][NH]) {
        float xp[NT][NH];
        if constexpr (PASS == RIFT_TC_PASS_MIDDLE || PASS == RIFT_TC_PASS_LAST) {   // in flight under the exchange reads
          const float *src = ch.xacc + ((size_t)(lb * RIFT_TC_NB + NH * wg)) * (NT * 128) + T;
#pragma unroll
          for (int n = 0; n < NH; ++n)
#pragma unroll
            for (int i = 0; i < NT; ++i) xp[i][n] = __ldcs(src + (size_t)n * (NT * 128) + 128 * i);
        }
        const float *blob = blob_s + (g % TC_STAGES) * BW;
        const float *xb = xb_s + (size_t)((wg * 2 + (g & 1u)) * (K - 2)) * NH * PITCH;
        const int32_t *dsh = reinterpret_cast<const int32_t *>(blob + K * tp.nch * 64) + NH * wg;
        for (int k = 2; k < K; ++k) {
          const int4 d0 = *reinterpret_cast<const int4 *>(dsh + k * 16), d1 = *reinterpret_cast<const int4 *>(dsh + k * 16 + 4);
          const int d[NH] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
          const float *base = xb + (size_t)(k - 2) * NH * PITCH + T + H;
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
      // per-warp (reference, sum) of the time marginal for the 8 samples of batch g (sorted batch index lb)
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
        const float *blob = blob_s + stage * BW;
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
          const float off = (mx == -INFINITY) ? 0.f : mx * cl2[n];       // reference in log2 units, rounded once
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

      // Software pipeline: the reduction of batch g and Phase A of batch g + 1 are issued from one basic block.
      float x[NT][NH];
      mbar_wait(bar_tfull, it & 1u);
      tc_fence_after();
      phase_a(it, x);
      for (uint32_t j = 0; j < nb; ++j) {
        const uint32_t g = it + j;
        if (K > 2) named_bar_sync(1 + wg, 128);                            // exchange rows of batch g are complete
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

// Combine the four lane-quarter partials of every sorted slot (fp64) and write lnL at the sample's natural position
__global__ void lnl_tcs_finalize_kernel(TcPlan tp, TcChunk ch, double *__restrict__ lnL_out) {
  const int64_t ws = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (ws >= (int64_t)ch.seg_begin[ch.n_lseg] * RIFT_TC_NB) return;
  const int32_t w = ch.perm[ws];
  if (w < 0) return;
  const int64_t gb = ch.gb0 + w / RIFT_TC_NB;
  const int64_t seg = gb / ch.nbps;
  const int64_t i = (gb % ch.nbps) * RIFT_TC_NB + (w % RIFT_TC_NB);
  const float4 *p = reinterpret_cast<const float4 *>(ch.part + ws * 4);
  const float4 p0 = p[0], p1 = p[1];
  const double m[4] = {p0.x, p0.z, p1.x, p1.z}, s[4] = {p0.y, p0.w, p1.y, p1.w};
  const double c = ch.scale_c[ws];
  double mm = -INFINITY;
  for (int a = 0; a < 4; ++a) mm = fmax(mm, m[a]);
  double sum = 0.0;
  for (int a = 0; a < 4; ++a)
    if (m[a] > -INFINITY) sum += s[a] * exp(c * (m[a] - mm));
  lnL_out[seg * ch.n_per_seg + i] = c * mm + log(sum) - log((double)tp.n_tau) - ch.quad[ws];
}

// Q [P][K][M][n_t] complex128, detector 1  ->  [P][kp/8][as_rows][8] fp16: row r holds time (r - dmax_1) mod n_t for
// r < n_t + 2 dmax_1 (zero beyond), contraction index kappa' = 8 plane + e over [Q_hi | Q_lo | Q_hi] as in convert_q_tc_kernel.
__global__ void convert_q_tcs_kernel(const double2 *__restrict__ src, uint16_t *__restrict__ dst, const float *__restrict__ scale,
                                     TcPlan tp, int sub, int64_t total) {
  const int ms = tp.m_sub, planes = tp.kp >> 3, dm = tp.dmax[1], a0 = sub * tp.m_sub;   // modes [a0, a0 + ms) of this subset
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const int e = (int)(idx & 7);
    const int64_t r64 = idx >> 3;
    const int r = (int)(r64 % tp.as_rows);
    const int c = (int)((r64 / tp.as_rows) % planes);
    const int64_t p = r64 / tp.as_rows / planes;
    const int kp_i = 8 * c + e;
    const int part = kp_i / (2 * ms), kap = kp_i % (2 * ms);
    const int a = a0 + (kap >> 1);
    uint16_t out = 0;
    if (r < tp.n_t + 2 * dm && part < 3 && a < tp.M) {
      int t = (r - dm) % tp.n_t;
      if (t < 0) t += tp.n_t;
      const double2 qv = src[((p * tp.K + 1) * tp.M + a) * tp.n_t + t];
      const double x = ((kap & 1) ? qv.y : qv.x) * (double)scale[p];
      const __half hi = __double2half(x);
      out = __half_as_ushort((part == 1) ? __double2half(x - (double)__half2float(hi)) : hi);
    }
    dst[idx] = out;
  }
}

template <int NT>
cudaError_t launch_nt(const TcsArgs &a, int pass, unsigned grid, size_t smem, cudaStream_t s) {
#define RIFT_TCS_CASE(P)                                                                                         \
  case P: {                                                                                                      \
    void (*kern)(TcsArgs) = nullptr;                                                                             \
    if (a.tp.n_tau < a.tp.n_t) {                                                                                 \
      if (pass != RIFT_TC_PASS_SINGLE) return cudaErrorInvalidValue;                                             \
      kern = lnl_tcs_kernel<NT, P, true, RIFT_TC_PASS_SINGLE>;                                                   \
    } else {                                                                                                     \
      kern = pass == RIFT_TC_PASS_SINGLE  ? lnl_tcs_kernel<NT, P, false, RIFT_TC_PASS_SINGLE>                    \
             : pass == RIFT_TC_PASS_FIRST ? lnl_tcs_kernel<NT, P, false, RIFT_TC_PASS_FIRST>                     \
             : pass == RIFT_TC_PASS_MIDDLE ? lnl_tcs_kernel<NT, P, false, RIFT_TC_PASS_MIDDLE>                   \
                                           : lnl_tcs_kernel<NT, P, false, RIFT_TC_PASS_LAST>;                    \
    }                                                                                                            \
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
    if (e != cudaSuccess) return e;                                                                              \
    kern<<<grid, TC_THREADS, smem, s>>>(a);                                                                      \
    return cudaGetLastError();                                                                                   \
  }
  switch (a.tp.pitch_s) {
    RIFT_TCS_CASE(256)
    RIFT_TCS_CASE(512)
    RIFT_TCS_CASE(640)
    RIFT_TCS_CASE(768)
    default: return cudaErrorInvalidValue;
  }
#undef RIFT_TCS_CASE
}

}  // namespace

size_t lnl_tcs_smem_bytes(const TcPlan &tp) {
  return 128 + (size_t)TC_STAGES * tp.blob_words_s * 4 + (size_t)(tp.kp >> 3) * tp.as_rows * 16 +
         (size_t)4 * (tp.K - 2) * NH * tp.pitch_s * 4;
}

cudaError_t launch_convert_q_tcs(const double *Q_c128, uint16_t *dst, const float *qscale, const TcPlan &tp,
                                 int32_t n_points, cudaStream_t s) {
  const int64_t total = (int64_t)n_points * (tp.kp >> 3) * tp.as_rows * 8;   // per mode subset
  if (total <= 0) return cudaSuccess;
  int64_t grid = (total + 255) / 256;
  if (grid > 148 * 32) grid = 148 * 32;
  for (int sub = 0; sub < tp.n_sub; ++sub)
    convert_q_tcs_kernel<<<(unsigned)grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), dst + (size_t)sub * total,
                                                        qscale, tp, sub, total);
  return cudaGetLastError();
}

cudaError_t launch_lnl_tcs(const TcPlan &tp, const uint32_t *qtc, const uint16_t *qs, const TcChunk &c, int pass,
                           double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (c.n_batches <= 0) return cudaSuccess;
  const size_t smem = lnl_tcs_smem_bytes(tp);
  TcsArgs a;
  a.tp = tp;
  a.ch = c;
  a.qtc = qtc;
  a.qs = qs;
  int64_t grid = n_sm;
  if (grid > c.n_batches) grid = c.n_batches;
  cudaError_t e;
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
  const int64_t n = c.cap_sorted * RIFT_TC_NB;
  lnl_tcs_finalize_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(tp, c, lnL_out);
  if (n_launch) ++*n_launch;
  return cudaGetLastError();
}
