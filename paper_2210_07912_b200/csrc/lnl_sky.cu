// Fused lnL kernel of the mixed mode for windows of any length: steps a6-a7 of DESIGN.md section 1 on sky-sorted batches.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// The samples of a chunk arrive bucketed by sky cell (sky_sort.cu): the 64 samples of a batch have relative shifts
// d_{n,k} = s_k - s_0 = b_k + r_{n,k} with one base b_k per detector and residuals 0 <= r < SKY_E.  Circular window
// (N_tau = N_t), detector-0 time: x_j = sum_k P_k[(j + b_k + r_{n,k}) mod N_t, n], P_k[t, n] = sum_kappa A_k[t, kappa] B_k[kappa, n].
// Time is tiled in blocks of 224 window entries (SKY_TBO = 256 - SKY_E - the 8-row rounding; 15 blocks on C4).
// Per (block, detector) a chunk of 256 consecutive operand rows starting at
// row  block start + b_k (rounded down to a multiple of 8: the remainder joins the residuals)  of the circularly extended fp16
// operand [Q_hi | Q_lo | Q_hi] -- stored as groups of 8 rows x K-major planes of 8 elements, so that a chunk is contiguous --
// arrives by ONE bulk copy into one of three ring slots; one elected thread contracts it with the coefficient operand
// [B_hi | B_hi | B_lo] of the batch (reading B8: fp16 pieces, products exact in the fp32 accumulator) by tcgen05.mma, both
// operands from shared memory, 2 row tiles of 128 x 64 samples x K = 16 per step, accumulators double-buffered in tensor
// memory so that the tensor core works on chunk i + 1 while the 16 warps drain chunk i: tcgen05.ld (thread = row, 16 samples),
// unshifted store into an exchange buffer [64 samples][256 rows] (lanes = consecutive rows: conflict-free), barrier, then
// every warp adds  P_k[j + r_{n,k}][n]  for its 4 samples n and the block's 224 window entries j = lane + 32 e into registers
// (again lanes = consecutive rows, whatever the shifts).  After the last detector the block joins the lane's running
// (max, sum) of 2^(c log2e (x - max)) per sample -- an on-line log-sum-exp, so the window never exists anywhere as a whole.
// Nothing but Q rows, 23 KB of coefficients per batch and one lnL per sample moves through L2 / HBM.
#include <cuda_fp16.h>

#include "tc_common.cuh"

namespace {

constexpr int SKY_WARPS = 16, SKY_THREADS = SKY_WARPS * 32, SKY_SLOTS = 3;
constexpr int SKY_NE = (SKY_TBO + 31) / 32;        // window entries per lane, sample and time block
constexpr int SKY_SPW = SKY_NB / SKY_WARPS;        // samples per warp in the reader role
constexpr float SKY_BSCALE = 8192.f;               // 2^13: scale of the coefficient operand (|F_k Y_lm| < 2) into the fp16 range
// instruction descriptor: D fp32, A/B fp16, both K-major, N = 64, M = 128
constexpr uint32_t SKY_IDESC = (1u << 4) | ((uint32_t)(SKY_NB >> 3) << 17) | ((128u >> 4) << 24);

struct SkySmem {                                   // byte offsets inside dynamic shared memory
  uint32_t bars, tmem, cl2, cval, qval, orig, resid, bk, bs, bs_det, xb, ring, slot_bytes, total;
};

__host__ __device__ inline SkySmem sky_smem(const SkyPlan &p) {
  SkySmem L;
  L.bars = 0;                                                          // full[3], tfull[2], tempty[2]
  L.tmem = 56;
  L.cl2 = 64;                                                          // float [64]
  L.cval = L.cl2 + SKY_NB * 4;                                         // double [64] c = D_ref / D
  L.qval = L.cval + SKY_NB * 8;                                        // double [64] q
  L.orig = L.qval + SKY_NB * 8;                                        // int [64] caller's sample (chunk-local), -1 = padding
  L.resid = L.orig + SKY_NB * 4;                                       // int [K][64] residual shifts
  L.bk = L.resid + (uint32_t)p.K * SKY_NB * 4;                         // int [8] base shifts, [8] = intrinsic point
  L.bs = (L.bk + 64 + 127u) & ~127u;                                   // fp16 [K][kp/8 planes][64 samples][8]
  L.bs_det = (uint32_t)(p.kp >> 3) * SKY_NB * 16;
  L.xb = (L.bs + (uint32_t)p.K * L.bs_det + 127u) & ~127u;             // float [64 samples][256 rows]
  L.ring = L.xb + SKY_TBR * SKY_NB * 4;
  L.slot_bytes = SKY_TBR * (uint32_t)p.ppp * 16;                       // one K piece: [32 groups of 8 rows][ppp planes][8 rows][8 fp16]
  L.total = L.ring + SKY_SLOTS * L.slot_bytes;
  return L;
}

struct SkyArgs {
  SkyPlan p;
  SkySmem L;
  const unsigned char *q;          // [P][K][n_pc pieces][rows_ext / 8][ppp planes][8 rows][8] fp16
  const float *qscale;             // [P] power-of-two scale of each point's Q
  Batch b;
  Workspace ws;                    // sorted slots: coef (fp32), scale_c, quad, shift, orig
  const int32_t *n_batches;        // device: batches of SKY_NB slots
  double *lnL_out;
};

// NPC, PPP: K pieces per chunk and planes per piece at compile time (0: read from the plan)
template <int NPC, int PPP>
__global__ void __launch_bounds__(SKY_THREADS, 1) lnl_sky_kernel(const SkyArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const SkyPlan &P = A.p;
  const SkySmem &L = A.L;
  const Batch &b = A.b;
  const Workspace &ws = A.ws;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + L.bars);
  uint64_t *tfull = full + SKY_SLOTS;                            // accumulators of a chunk ready (tcgen05.commit)
  uint64_t *tempty = tfull + 2;                                  // accumulator buffer drained by all 16 warps
  uint32_t *tmem_ptr_s = reinterpret_cast<uint32_t *>(smem_raw + L.tmem);
  float *cl2_s = reinterpret_cast<float *>(smem_raw + L.cl2);
  double *cval_s = reinterpret_cast<double *>(smem_raw + L.cval);
  double *qval_s = reinterpret_cast<double *>(smem_raw + L.qval);
  int *orig_s = reinterpret_cast<int *>(smem_raw + L.orig);
  int *resid_s = reinterpret_cast<int *>(smem_raw + L.resid);
  int *bk_s = reinterpret_cast<int *>(smem_raw + L.bk);
  unsigned char *bs = smem_raw + L.bs;
  float *xb = reinterpret_cast<float *>(smem_raw + L.xb);
  unsigned char *ring = smem_raw + L.ring;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_pc = NPC ? NPC : P.n_pc, ppp = PPP ? PPP : P.ppp;
  const int K = P.K, n_t = P.n_t, m2 = 2 * P.M, npl = n_pc * ppp;
  if (tid == 0) {
    for (int i = 0; i < SKY_SLOTS; ++i) mbar_init(full + i, 1);
    mbar_init(tfull, 1);
    mbar_init(tfull + 1, 1);
    mbar_init(tempty, SKY_WARPS);
    mbar_init(tempty + 1, SKY_WARPS);
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr_s)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr_s;

  // Four groups of 4 warps own the sample quarters 0-15 / ... / 48-63 of the batch (their columns of the accumulators, their
  // quarter of the exchange buffer: a warp drains lanes 32 (warp & 3) .. of its group's columns and reads back four of its
  // group's samples) and synchronise among themselves only: the drain, store and read phases of the groups interleave
  // (two groups of 8 warps: 353 ms on C4; four groups: 327 ms).
  // drain role: tensor-memory lanes 32 (warp & 3) .. + 31 (rows of a 128-row tile), columns 16 (warp >> 2) .. + 15 (samples)
  const int q4 = warp & 3, cg = warp >> 2, grp = warp >> 2;
  auto group_bar = [&]() { named_bar_sync(1 + grp, 4 * 32); };
  const uint32_t t_lane = ((uint32_t)(32 * q4)) << 16;
  float *xst = xb + (size_t)(16 * cg) * SKY_TBR + 32 * q4 + lane;        // + c * 256 (sample) + 128 mt (row tile)
  // reader role: samples SKY_SPW warp .. + 3, window entries lane + 32 e of the block
  const double ln_ntau = log((double)n_t);
  const int n_chunks = P.n_blocks * K;
  const uint32_t ring_u32 = smem_u32(ring), bs_u32 = smem_u32(bs);

  const int total_batches = *A.n_batches;
  const int bt_begin = (int)(((int64_t)total_batches * blockIdx.x) / gridDim.x);
  const int bt_end = (int)(((int64_t)total_batches * (blockIdx.x + 1)) / gridDim.x);
  uint32_t cnt = 0;                                              // chunks consumed so far (ring slot, buffers, phases)

  for (int bt = bt_begin; bt < bt_end; ++bt) {
    const int64_t slot0 = (int64_t)bt * SKY_NB;
    // ---- stage the batch
    if (tid < 8) bk_s[tid] = INT32_MAX;
    __syncthreads();                                             // previous batch fully consumed; bk reset
    if (tid < SKY_NB) {
      orig_s[tid] = ws.orig[slot0 + tid];
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
    // coefficient operand [B_hi | B_hi | B_lo]: K-major planes of 8 elements, [detector][plane][sample][8 fp16]
    for (int idx = tid; idx < SKY_NB * K * npl; idx += SKY_THREADS) {
      const int n = idx % SKY_NB, kc = idx / SKY_NB, c = kc % npl, k = kc / npl;
      const float *src = reinterpret_cast<const float *>(ws.coef) + (slot0 + n) * ws.coef_stride + k * m2;
      __align__(16) __half hv[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const int kap = 8 * c + e, region = kap / m2;
        __half h = __float2half_rn(0.f);
        if (region < 3) {
          const float v = src[kap - region * m2] * SKY_BSCALE;
          const __half hi = __float2half_rn(v);
          h = region < 2 ? hi : __float2half_rn(v - __half2float(hi));
        }
        hv[e] = h;
      }
      *reinterpret_cast<uint4 *>(bs + (size_t)k * L.bs_det + ((size_t)c * SKY_NB + n) * 16) = *reinterpret_cast<const uint4 *>(hv);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> UMMA operand reads
    __syncthreads();
    const int point = bk_s[8];
    if (tid < SKY_NB * K) {
      const int bkk = bk_s[tid / SKY_NB] == INT32_MAX ? 0 : bk_s[tid / SKY_NB];
      int r = my_d == INT32_MAX ? 0 : my_d - bkk;
      r = r < 0 ? 0 : (r > SKY_E - 1 ? SKY_E - 1 : r);           // out of range only for a sample with NaN angles
      resid_s[tid] = r + (bkk & 7);                              // the chunk starts at the 8-row group holding b_k
    }
    if (tid < SKY_NB) cl2_s[tid] = (float)(cval_s[tid] * 1.4426950408889634 / ((double)A.qscale[point] * SKY_BSCALE));
    const unsigned char *qpoint = A.q + (int64_t)point * P.point_stride;
    // ring entry e = (chunk e / n_pc = (block, detector), K piece e % n_pc): 32 groups of 8 rows x ppp planes, one bulk copy
    // into ring slot re % 3 (re = the entry's running number)
    auto issue_tma = [&](int e, uint32_t re) {
      const int i = e / n_pc, pc = e - i * n_pc;
      const int blk = i / K, k = i - blk * K;
      const int bk = bk_s[k] == INT32_MAX ? 0 : bk_s[k];
      const int64_t grp = (P.R0 + blk * SKY_TBO + (bk & ~7)) >> 3;          // R0, SKY_TBO are multiples of 8; floor for bk < 0
      const uint32_t slot = re % SKY_SLOTS;
      mbar_expect_tx(full + slot, L.slot_bytes);
      bulk_g2s(ring + slot * L.slot_bytes,
               qpoint + (((int64_t)k * n_pc + pc) * (P.rows_ext >> 3) + grp) * (int64_t)(ppp * 128), L.slot_bytes, full + slot);
    };
    // P_k tiles of chunk i into accumulator buffer c & 1: 2 row tiles x kp / 16 steps
    auto issue_mma = [&](int i, uint32_t c) {
      const int k = i % K;
      mbar_wait(tempty + (c & 1u), ((c >> 1) & 1u) ^ 1u);         // both groups have drained the chunk before last
      const uint32_t d0 = tmem_base + (c & 1u) * 128u;
      for (int pc = 0; pc < n_pc; ++pc) {
        const uint32_t re = c * (uint32_t)n_pc + (uint32_t)pc, slot = re % SKY_SLOTS;
        mbar_wait(full + slot, (re / SKY_SLOTS) & 1u);
        tc_fence_after();
        // A: planes of one 8-row group are 128 bytes apart (LBO), groups ppp * 128 bytes (SBO); B: [plane][sample][16 bytes]
        const uint64_t adesc = tc_smem_desc(ring_u32 + slot * L.slot_bytes, 128u, (uint32_t)ppp * 128u);
        const uint64_t bdesc = tc_smem_desc(bs_u32 + (uint32_t)k * L.bs_det + (uint32_t)(pc * ppp) * (SKY_NB * 16u), SKY_NB * 16u, 128u);
        for (int s = 0; 2 * s < ppp; ++s) {
          const uint64_t bd = bdesc + (uint64_t)((uint32_t)(2 * s) * (SKY_NB * 16u) >> 4);
          const uint64_t ad = adesc + (uint64_t)((uint32_t)(2 * s) * 128u >> 4);
          const uint32_t accum = (pc > 0 || s > 0) ? 1u : 0u;
          tc_mma_ss(d0, ad, bd, SKY_IDESC, accum);
          tc_mma_ss(d0 + SKY_NB, ad + (uint64_t)((16u * (uint32_t)ppp * 128u) >> 4), bd, SKY_IDESC, accum);
        }
      }
      tc_commit(tfull + (c & 1u));
    };
    const int n_entries = n_chunks * n_pc;
    if (warp == 0) {                                             // bulk copies and tensor-core instructions come from warp 0 here,
      if (elect_one()) {                                         // in the loop from two different warps
        for (int e = 0; e < SKY_SLOTS && e < n_entries; ++e) issue_tma(e, cnt * (uint32_t)n_pc + (uint32_t)e);
        issue_mma(0, cnt);
      }
      __syncwarp();
    }
    __syncthreads();

    // Padding slots sit at the end of a batch (the last batch of a sky cell holds 32 samples on average): a group whose
    // sample quarter is all padding keeps the barrier protocol of the chunks (tfull / tempty, the ring refills of warp 13)
    // and skips the drain, the exchange and the log-sum-exp, which leaves the shared-memory pipe to the other groups
    const bool live = orig_s[16 * grp] >= 0;
    float m_run[SKY_SPW], s_run[SKY_SPW], cl2n[SKY_SPW];
#pragma unroll
    for (int sp = 0; sp < SKY_SPW; ++sp) {
      m_run[sp] = -INFINITY;
      s_run[sp] = 0.f;
      cl2n[sp] = cl2_s[SKY_SPW * warp + sp];
    }
    for (int blk = 0; blk < P.n_blocks; ++blk) {
      float x[SKY_SPW][SKY_NE];
      for (int k = 0; k < K; ++k, ++cnt) {
        const int i = blk * K + k;
        // the tensor core starts on the next chunk (its accumulator buffer was drained before the barriers of chunk i - 1)
        if (warp == 0 && i + 1 < n_chunks) {
          if (elect_one()) issue_mma(i + 1, cnt + 1);
          __syncwarp();
        }
        // ---- drain chunk i: thread = row, 16 samples per row tile
        mbar_wait(tfull + (cnt & 1u), (cnt >> 1) & 1u);
        tc_fence_after();
        float acc[2][2][8];
        if (live) {
#pragma unroll
          for (int mt = 0; mt < 2; ++mt) {
            const uint32_t ta = tmem_base + t_lane + (cnt & 1u) * 128u + (uint32_t)(mt * SKY_NB + 16 * cg);
            tc_ld8(ta, acc[mt][0]);
            tc_ld8(ta + 8, acc[mt][1]);
          }
#pragma unroll
          for (int mt = 0; mt < 2; ++mt) {
            tc_wait_ld8(acc[mt][0]);
            tc_wait_ld8(acc[mt][1]);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty + (cnt & 1u));
        if (live) {
          group_bar();                                           // every reader of the group is done with the previous detector
#pragma unroll
          for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int c = 0; c < 8; ++c) xst[(8 * h + c) * SKY_TBR + 128 * mt] = acc[mt][h][c];
          group_bar();                                           // the group's rows of detector k are complete
        }
        tc_fence_after();
        if (warp == 13) {                                        // tfull of chunk i was observed: its ring slots are free
          if (elect_one())
            for (int pc = 0; pc < n_pc; ++pc) {
              const int e = i * n_pc + pc + SKY_SLOTS;
              if (e < n_entries) issue_tma(e, cnt * (uint32_t)n_pc + (uint32_t)(pc + SKY_SLOTS));
            }
          __syncwarp();
        }
        // ---- shifted read: x_j += P_k[j + r][n], lanes = consecutive rows
        if (!live) continue;
#pragma unroll
        for (int sp = 0; sp < SKY_SPW; ++sp) {
          const int n = SKY_SPW * warp + sp;
          const float *src = xb + n * SKY_TBR + resid_s[k * SKY_NB + n] + lane;
          if (k == 0) {
#pragma unroll
            for (int e = 0; e < SKY_NE; ++e) x[sp][e] = src[32 * e];
          } else {
#pragma unroll
            for (int e = 0; e < SKY_NE; ++e) x[sp][e] += src[32 * e];
          }
        }
      }
      // ---- the block joins the running log-sum-exp of this lane, per sample
      if (!live) continue;
      const int j0 = blk * SKY_TBO + lane;
      const int j_end = min(n_t, (blk + 1) * SKY_TBO);
#pragma unroll
      for (int sp = 0; sp < SKY_SPW; ++sp) {
        float bm = -INFINITY;
#pragma unroll
        for (int e = 0; e < SKY_NE; ++e)
          if (j0 + 32 * e < j_end) bm = fmaxf(bm, x[sp][e]);
        const float m_new = fmaxf(m_run[sp], bm);
        float s = m_run[sp] == -INFINITY ? 0.f : s_run[sp] * fast_exp2((m_run[sp] - m_new) * cl2n[sp]);
#pragma unroll
        for (int e = 0; e < SKY_NE; ++e)
          if (j0 + 32 * e < j_end) s += fast_exp2((x[sp][e] - m_new) * cl2n[sp]);
        s_run[sp] = s;
        m_run[sp] = m_new;
      }
    }
    // ---- per sample: combine the 32 lanes, write lnL
#pragma unroll
    for (int sp = 0; sp < SKY_SPW; ++sp) {
      const int n = SKY_SPW * warp + sp;
      const float m = warp_max(m_run[sp]);
      float s = m_run[sp] == -INFINITY ? 0.f : s_run[sp] * fast_exp2((m_run[sp] - m) * cl2n[sp]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (lane == 0 && orig_s[n] >= 0) {
        const double inv = 1.0 / ((double)A.qscale[point] * SKY_BSCALE);
        A.lnL_out[b.g0 + orig_s[n]] = cval_s[n] * ((double)m * inv) + log((double)s) - ln_ntau - qval_s[n];
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
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
  // dst: [point][detector][K piece][group = extended row / 8][plane of the piece][row % 8][kappa % 8]
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int e8 = (int)(i & 7), r8 = (int)((i >> 3) & 7);
    const int64_t gi = i >> 6;
    const int pl = (int)(gi % p.ppp);
    const int64_t gg = gi / p.ppp;
    const int r = (int)(gg % (p.rows_ext >> 3)) * 8 + r8;
    const int64_t pp = gg / (p.rows_ext >> 3);
    const int pc = (int)(pp % p.n_pc);
    const int64_t pk = pp / p.n_pc;                                        // point * K + detector
    const int kap = 8 * (pc * p.ppp + pl) + e8;
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
    dst[i] = h;
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
  void (*kern)(SkyArgs) = lnl_sky_kernel<0, 0>;
  if (p.n_pc == 1 && p.ppp == 8) kern = lnl_sky_kernel<1, 8>;        // 9-10 modes (C4)
  else if (p.n_pc == 2 && p.ppp == 8) kern = lnl_sky_kernel<2, 8>;   // 20-21 modes (C2)
  else if (p.n_pc == 1 && p.ppp == 4) kern = lnl_sky_kernel<1, 4>;   // 5 modes (C1, C3)
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)a.L.total);
  if (e != cudaSuccess) return e;
  int64_t grid = n_sm;
  if (grid > max_batches) grid = max_batches;
  if (grid < 1) grid = 1;
  kern<<<(unsigned)grid, SKY_THREADS, a.L.total, s>>>(a);
  if (n_launch) ++*n_launch;
  return cudaGetLastError();
}
