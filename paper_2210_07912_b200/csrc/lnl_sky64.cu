// Fused lnL kernel of the fp64 mode for windows of any length: steps a6-a7 of DESIGN.md section 1 on sky-sorted batches --
// the fp64 sibling of lnl_sky.cu (same bucketing, same time tiling, same exchange and on-line log-sum-exp), with the
// contraction on the FP64 tensor cores (mma.sync.m8n8k4.f64, as lnl_mma.cu) because tcgen05 has no fp64 kind.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// A sorted batch of 64 slots (relative shifts d_{n,k} = b_k + r_{n,k}, 0 <= r < SKY64_E) is processed as two half batches of 32
// samples.  Per (block of 224 window entries, detector) a chunk of 256 consecutive rows of the circularly extended operand
// A_k[t, 2m + {0,1}] = {Re, Im} Q_{k,m}[t] (fp64, rows of kappa_p doubles with kappa_p = 4 (mod 8): conflict-free fragment
// loads) arrives by one bulk copy into a ring slot.  The CTA is two independent groups of 8 warps, each with 16 samples of the
// half batch, its own exchange buffer and named barrier: a group contracts the chunk with the coefficients B_k[kappa, n] of its
// samples -- 4 row blocks of 8 x 2 sample tiles per warp --, stores the tiles unshifted into its exchange buffer
// [16 samples][258 rows] (lanes = rows; sample pairs 32 bytes apart modulo 128), and after a group barrier adds
// P_k[j + r_{n,k}][n] for 2 samples per warp and the block's window entries j = lane + 32 e into registers.  After the last
// detector the block joins the lane's running (float max, fp64 sum of 2^(c log2e (x - max))) per sample.  The groups drift apart
// by up to `slots` chunks, so the tensor phase of one runs under the exchange and exponential phases of the other; the group
// that finishes a chunk last refills its ring slot.
#include "rift_internal.h"
#include "tma_utils.cuh"
#include "exp2_poly.cuh"

namespace {

constexpr int S64_WARPS = 16, S64_THREADS = S64_WARPS * 32, S64_NB = 32, S64_SPW = S64_NB / S64_WARPS;
constexpr int S64_TBO = 224, S64_TBR = 256, S64_NE = S64_TBO / 32, S64_XP = S64_TBR + 2;

struct S64Smem {
  uint32_t bars, cval, qval, orig, resid, bk, cs, xb, ring, slot_bytes, total;
};

__host__ __device__ inline S64Smem s64_smem(const Sky64Plan &p) {
  S64Smem L;
  L.bars = 0;                                                          // full[slots] (8 B each), done[slots] ints at +32
  L.cval = 64;                                                         // double [64] c
  L.qval = L.cval + 64 * 8;                                            // double [64] q
  L.orig = L.qval + 64 * 8;                                            // int [64]
  L.resid = L.orig + 64 * 4;                                           // int [K][64]
  L.bk = L.resid + (uint32_t)p.K * 64 * 4;                             // int [8] base shifts, [8] = intrinsic point
  L.cs = (L.bk + 64 + 127u) & ~127u;                                   // double [K][KS][32][4]: B fragments of a half batch
  L.xb = (L.cs + (uint32_t)p.K * p.KS * S64_NB * 4 * 8 + 127u) & ~127u;  // double [32][258]
  L.ring = (L.xb + S64_NB * S64_XP * 8 + 127u) & ~127u;
  L.slot_bytes = S64_TBR * (uint32_t)p.kp * 8;
  L.total = L.ring + (uint32_t)p.slots * L.slot_bytes;
  return L;
}

struct S64Args {
  Sky64Plan p;
  S64Smem L;
  const unsigned char *q;          // [P][K][rows_ext][kp] doubles
  Batch b;
  Workspace ws;                    // sorted slots: coef (fp64), scale_c, quad, shift, orig
  const int32_t *n_batches;
  double *lnL_out;
};

__device__ __forceinline__ void dmma64(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

__device__ __forceinline__ void s64_bar(int id) { asm volatile("bar.sync %0, 256;" ::"r"(id) : "memory"); }

__global__ void __launch_bounds__(S64_THREADS, 1) lnl_sky64_kernel(const S64Args A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const Sky64Plan &P = A.p;
  const S64Smem &L = A.L;
  const Batch &b = A.b;
  const Workspace &ws = A.ws;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + L.bars);
  double *cval_s = reinterpret_cast<double *>(smem_raw + L.cval);
  double *qval_s = reinterpret_cast<double *>(smem_raw + L.qval);
  int *orig_s = reinterpret_cast<int *>(smem_raw + L.orig);
  int *resid_s = reinterpret_cast<int *>(smem_raw + L.resid);
  int *bk_s = reinterpret_cast<int *>(smem_raw + L.bk);
  double *cs = reinterpret_cast<double *>(smem_raw + L.cs);
  double *xb = reinterpret_cast<double *>(smem_raw + L.xb);
  unsigned char *ring = smem_raw + L.ring;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K = P.K, KS = P.KS, n_t = P.n_t, m2 = 2 * P.M, kp = P.kp, slots = P.slots;
  if (tid == 0)
    for (int i = 0; i < slots; ++i) mbar_init(full + i, 1);
  __syncthreads();

  // two groups of 8 warps: group grp takes samples 16 grp .. 16 grp + 15 of the half batch
  const int grp = warp >> 3, wg = warp & 7, gtid = tid & 255, bar_id = 1 + grp;
  int *done = reinterpret_cast<int *>(smem_raw + L.bars + 32);   // groups that have consumed the chunk in a ring slot
  if (tid < 8) done[tid] = 0;
  // MMA role: fragment coordinates; row blocks 4 wg .. 4 wg + 3 of the chunk; the group's two sample tiles
  const int g = lane >> 2, t4 = lane & 3;
  const uint32_t a_off = (uint32_t)(32 * wg + g) * (uint32_t)kp * 8u + (uint32_t)t4 * 8u;   // + 8 rb kp * 8 (row block rb) + 32 s
  // store role: rows 32 wg + g + 8 rb, samples 8 nt + 2 t4 (+ 1) of the group
  double *xbg = xb + grp * (S64_NB / 2) * S64_XP;
  double *xst = xbg + (2 * t4) * S64_XP + 32 * wg + g;
  const double ln_ntau = log((double)n_t);
  const int n_chunks = P.n_blocks * K;

  const int total_batches = *A.n_batches;
  const int bt_begin = (int)(((int64_t)total_batches * blockIdx.x) / gridDim.x);
  const int bt_end = (int)(((int64_t)total_batches * (blockIdx.x + 1)) / gridDim.x);
  uint32_t cnt = 0;                                              // chunks consumed so far (ring slot and phase)

  for (int bt = bt_begin; bt < bt_end; ++bt) {
    const int64_t slot0 = (int64_t)bt * SKY_NB;
    // ---- stage what both half batches share
    if (tid < 8) bk_s[tid] = INT32_MAX;
    __syncthreads();
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
    __syncthreads();
    const int point = bk_s[8];
    if (tid < SKY_NB * K) {
      const int bkk = bk_s[tid / SKY_NB] == INT32_MAX ? 0 : bk_s[tid / SKY_NB];
      int r = my_d == INT32_MAX ? 0 : my_d - bkk;
      resid_s[tid] = r < 0 ? 0 : (r > SKY64_E - 1 ? SKY64_E - 1 : r);   // out of range only for a sample with NaN angles
    }
    const unsigned char *qpoint = A.q + (int64_t)point * P.point_stride;
    auto issue = [&](int i, uint32_t c) {                        // chunk i = (block i / K, detector i % K) into ring slot c % slots
      const int blk = i / K, k = i - blk * K;
      const int bk = bk_s[k] == INT32_MAX ? 0 : bk_s[k];
      const int64_t row = (int64_t)k * P.rows_ext + P.R0 + blk * S64_TBO + bk;
      const uint32_t slot = c % (uint32_t)slots;
      mbar_expect_tx(full + slot, L.slot_bytes);
      for (uint32_t off = 0; off < L.slot_bytes; off += 32768u)
        bulk_g2s(ring + slot * L.slot_bytes + off, qpoint + row * (int64_t)(kp * 8) + off, min(32768u, L.slot_bytes - off),
                 full + slot);
    };

    for (int half = 0; half < 2; ++half) {
      // ---- coefficients of the half batch as B fragments cs[k][s][n][4] (zero beyond 2 M)
      __syncthreads();                                           // the previous half batch is done with cs, xb and the ring
      if (half == 1 && orig_s[32] < 0) break;                    // padding sits at the end of a batch: nothing in this half
      for (int idx = tid; idx < K * KS * S64_NB * 4; idx += S64_THREADS) {
        const int e = idx & 3, n = (idx >> 2) % S64_NB, ks = (idx >> 2) / S64_NB, s = ks % KS, k = ks / KS;
        const int kap = 4 * s + e;
        cs[idx] = kap < m2 ? reinterpret_cast<const double *>(ws.coef)[(slot0 + 32 * half + n) * ws.coef_stride + k * m2 + kap] : 0.0;
      }
      if (tid == 0)
        for (int i = 0; i < slots && i < n_chunks; ++i) issue(i, cnt + i);
      __syncthreads();

      // A group whose 16 samples are all padding only keeps the ring's bookkeeping: one thread counts the group's consumption
      // of every chunk once it has landed (and refills the slot if the other group was there first); the FP64 unit is the
      // other group's meanwhile
      if (orig_s[32 * half + 16 * grp] < 0) {
        if (gtid == 0)
          for (int i = 0; i < n_chunks; ++i) {
            const uint32_t c = cnt + (uint32_t)i, slot = c % (uint32_t)slots;
            mbar_wait(full + slot, (c / (uint32_t)slots) & 1u);
            __threadfence_block();
            if (atomicAdd(done + slot, 1) == 1) {
              done[slot] = 0;
              __threadfence_block();
              if (i + slots < n_chunks) issue(i + slots, c + (uint32_t)slots);
            }
          }
        cnt += (uint32_t)n_chunks;
        continue;
      }
      float m_run[S64_SPW];
      double s_run[S64_SPW], cl2n[S64_SPW];
#pragma unroll
      for (int sp = 0; sp < S64_SPW; ++sp) {
        m_run[sp] = -INFINITY;
        s_run[sp] = 0.0;
        cl2n[sp] = cval_s[32 * half + 16 * grp + S64_SPW * wg + sp] * 1.4426950408889634;
      }
      // Software pipeline over the chunks c = (block, detector): the tensor phase of chunk c + 1 is issued between the barrier
      // that completes the rows of chunk c and the shifted read of those rows, so that the read's shared-memory latency and
      // the block's exponentials run under the next chunk's DMMAs
      double acc[4][2][2];
      auto tensor_phase = [&](int k, uint32_t c) {               // P_k tiles of the chunk in ring slot c % slots
        const uint32_t slot = c % (uint32_t)slots;
        mbar_wait(full + slot, (c / (uint32_t)slots) & 1u);
#pragma unroll
        for (int rb = 0; rb < 4; ++rb)
#pragma unroll
          for (int nt = 0; nt < 2; ++nt) acc[rb][nt][0] = acc[rb][nt][1] = 0.0;
        const unsigned char *ap = ring + slot * L.slot_bytes + a_off;
        const double *bp = cs + (size_t)(k * KS) * S64_NB * 4 + (16 * grp + g) * 4 + t4;
#pragma unroll 1
        for (int s = 0; s < KS; ++s, ap += 32, bp += S64_NB * 4) {
          double av[4];
#pragma unroll
          for (int rb = 0; rb < 4; ++rb) av[rb] = *reinterpret_cast<const double *>(ap + rb * (8 * kp * 8));
          const double b0 = bp[0], b1 = bp[32];
#pragma unroll
          for (int rb = 0; rb < 4; ++rb) {
            dmma64(acc[rb][0], av[rb], b0);
            dmma64(acc[rb][1], av[rb], b1);
          }
        }
      };
      tensor_phase(0, cnt);
      double x[S64_SPW][S64_NE];
      for (int blk = 0; blk < P.n_blocks; ++blk) {
        for (int k = 0; k < K; ++k, ++cnt) {
          const int i = blk * K + k;
          s64_bar(bar_id);                                       // every reader of the group is done with the previous chunk's rows
#pragma unroll
          for (int rb = 0; rb < 4; ++rb)
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
              xst[(8 * nt) * S64_XP + 8 * rb] = acc[rb][nt][0];
              xst[(8 * nt + 1) * S64_XP + 8 * rb] = acc[rb][nt][1];
            }
          s64_bar(bar_id);                                       // the rows of chunk i are complete; the group has consumed it
          if (gtid == 0) {                                       // the group that consumes the chunk last refills its slot
            const uint32_t slot = cnt % (uint32_t)slots;
            __threadfence_block();
            if (atomicAdd(done + slot, 1) == 1) {
              done[slot] = 0;
              __threadfence_block();
              if (i + slots < n_chunks) issue(i + slots, cnt + (uint32_t)slots);
            }
          }
          if (i + 1 < n_chunks) tensor_phase(k + 1 < K ? k + 1 : 0, cnt + 1u);
          // ---- shifted read: x_j += P_k[j + r][n], lanes = consecutive rows
#pragma unroll
          for (int sp = 0; sp < S64_SPW; ++sp) {
            const int n = S64_SPW * wg + sp;
            const double *src = xbg + n * S64_XP + resid_s[k * SKY_NB + 32 * half + 16 * grp + n] + lane;
            if (k == 0) {
#pragma unroll
              for (int e = 0; e < S64_NE; ++e) x[sp][e] = src[32 * e];
            } else {
#pragma unroll
              for (int e = 0; e < S64_NE; ++e) x[sp][e] += src[32 * e];
            }
          }
        }
        // ---- the block joins the running log-sum-exp of this lane, per sample
        const int j0 = blk * S64_TBO + lane;
#pragma unroll
        for (int sp = 0; sp < S64_SPW; ++sp) {
          float bm = -INFINITY;
#pragma unroll
          for (int e = 0; e < S64_NE; ++e)
            if (j0 + 32 * e < n_t) bm = fmaxf(bm, __double2float_ru(x[sp][e]));
          const float m_new = fmaxf(m_run[sp], bm);
          const double mo = -(double)m_new * cl2n[sp];
          double s = m_run[sp] == -INFINITY ? 0.0 : s_run[sp] * poly_exp2(fma((double)m_run[sp], cl2n[sp], mo));
#pragma unroll
          for (int e = 0; e < S64_NE; ++e)
            if (j0 + 32 * e < n_t) s += poly_exp2(fma(x[sp][e], cl2n[sp], mo));
          s_run[sp] = s;
          m_run[sp] = m_new;
        }
      }
      // ---- per sample: combine the 32 lanes, write lnL
#pragma unroll
      for (int sp = 0; sp < S64_SPW; ++sp) {
        const int n = 32 * half + 16 * grp + S64_SPW * wg + sp;
        const float m = warp_max(m_run[sp]);
        double s = m_run[sp] == -INFINITY ? 0.0 : s_run[sp] * poly_exp2(((double)m_run[sp] - (double)m) * cl2n[sp]);
        s = warp_sum(s);
        if (lane == 0 && orig_s[n] >= 0) A.lnL_out[b.g0 + orig_s[n]] = cval_s[n] * (double)m + log(s) - ln_ntau - qval_s[n];
      }
    }
  }
}

__global__ void convert_q_sky64_kernel(const double2 *__restrict__ src, double *__restrict__ dst, Sky64Plan p, int64_t total) {
  // dst: [point][detector][extended row][kappa], kappa = 2 m + {Re, Im}, zero beyond 2 M; row e holds (e - R0) mod n_t
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int kap = (int)(i % p.kp);
    const int64_t ri = i / p.kp;
    const int r = (int)(ri % p.rows_ext);
    const int64_t pk = ri / p.rows_ext;
    int t = (r - p.R0) % p.n_t;
    if (t < 0) t += p.n_t;
    double v = 0.0;
    if (kap < 2 * p.M) {
      const double2 v2 = src[(pk * p.M + (kap >> 1)) * p.n_t + t];
      v = (kap & 1) ? v2.y : v2.x;
    }
    dst[i] = v;
  }
}

}  // namespace

size_t lnl_sky64_smem_bytes(const Sky64Plan &p) { return s64_smem(p).total; }

cudaError_t launch_convert_q_sky64(const double *Q_c128, void *dst, const Sky64Plan &p, int32_t n_points, cudaStream_t s) {
  const int64_t total = (int64_t)n_points * p.K * p.rows_ext * p.kp;
  convert_q_sky64_kernel<<<148 * 16, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), reinterpret_cast<double *>(dst), p,
                                                  total);
  return cudaGetLastError();
}

cudaError_t launch_lnl_sky64(const Sky64Plan &p, const void *q, const Batch &b, const Workspace &ws,
                             const int32_t *n_batches_dev, int64_t max_batches, double *lnL_out, int n_sm, cudaStream_t s,
                             int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  S64Args a;
  a.p = p;
  a.L = s64_smem(p);
  a.q = reinterpret_cast<const unsigned char *>(q);
  a.b = b;
  a.ws = ws;
  a.n_batches = n_batches_dev;
  a.lnL_out = lnL_out;
  cudaError_t e = cudaFuncSetAttribute(lnl_sky64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)a.L.total);
  if (e != cudaSuccess) return e;
  int64_t grid = n_sm;
  if (grid > max_batches) grid = max_batches;
  if (grid < 1) grid = 1;
  lnl_sky64_kernel<<<(unsigned)grid, S64_THREADS, a.L.total, s>>>(a);
  if (n_launch) ++*n_launch;
  return cudaGetLastError();
}
