// Fused lnL kernel of the fp64 mode on the FP64 tensor cores: steps a6-a7 of DESIGN.md section 1.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// "Contract in unshifted detector time, then shift": per detector k the window term is the real GEMM
//     P_k[t, n] = sum_kappa A_k[t, kappa] B_k[kappa, n],   A_k[t, 2m + {0,1}] = {Re, Im} Q_{k,m}[t],  B_k[2m + {0,1}, n] = {Re, Im}(F_k Y_m)_n
// over ALL stored rows t (M = time, N = samples of the batch, K = 2 x modes), issued as mma.sync.m8n8k4.f64 (DMMA, 256 FMA
// per instruction and warp: one Q value read from shared memory feeds 8 samples, one coefficient 8 rows -- the direct kernel
// reads a 16-byte Q value per 2 DFMA and cannot pass 25 % of the pipe).  The per-sample shift is applied when a tile of P_k
// leaves the registers: x[n][(t - off_{n,k}) mod N_t] (+)= P_k[t, n] in a per-batch window buffer in shared memory (the
// first detector stores, the others read-modify-write; within one detector every (t, n) owns its target, detectors are
// separated by a barrier).  The time marginal then runs over the finished windows with lanes over tau.
//
// Q operand: the handle keeps [P][K][M2][pitch] bytes, M2 = 2 ceil(M/2) mode rows per detector (zero rows pad an odd mode
// count), every row n_r = 8 ceil(N_t/8) complex128 (zero beyond N_t) followed by 64 pad bytes, so that the two mode rows of
// one k-step sit 64 bytes apart modulo 128 and an A fragment load (8 rows x 2 modes x 16 B) is conflict-free.  Small
// configurations keep the whole block of the intrinsic point resident in shared memory (one bulk copy per point); larger
// ones stream (detector, row range, k-step) chunks through a ring filled by a producer warp with cp.async.bulk on mbarriers.
#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

constexpr int MM_WARPS = 16;                       // warps per CTA: 16 consumers (resident) or 15 consumers + 1 producer (ring),
                                                   // so that every thread may hold 128 registers
constexpr int MM_RBW = 4;                          // row blocks (of 8 rows) per warp and row range: a range = 32 rows x consumers
constexpr int MM_MAX_SLOTS = 8;

__device__ __forceinline__ void mm_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
template <int CW>
__device__ __forceinline__ void mm_bar_consumers() { asm volatile("bar.sync 1, %0;" ::"n"(CW * 32) : "memory"); }

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

// 2^y for y <= 0 (NaN propagates): y = n + r, |r| <= 1/2, 2^r by a degree-8 polynomial (interpolation at Chebyshev nodes,
// relative error 1.1e-12), 2^n through the exponent field.  12 FP64-pipe operations with the argument FMA of the caller.
__device__ __forceinline__ double mm_exp2(double y) {
  y = fmax(y, -1000.0);
  const double t = y + 6755399441055744.0;                       // 1.5 * 2^52: the low word of t holds rint(y)
  const int n = __double2loint(t);
  const double r = y - (t - 6755399441055744.0);
  double p = 0x1.63d1363b4014fp-20;
  p = fma(p, r, 0x1.00dc4a5363675p-16);
  p = fma(p, r, 0x1.4308ac85a5afep-13);
  p = fma(p, r, 0x1.5d8745a727ee4p-10);
  p = fma(p, r, 0x1.3b2ab7181b784p-7);
  p = fma(p, r, 0x1.c6b08dd6fd239p-5);
  p = fma(p, r, 0x1.ebfbdff823cedp-3);
  p = fma(p, r, 0x1.62e42fef84cf0p-1);
  p = fma(p, r, 1.0);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}

struct MmaSmem {                                   // byte offsets inside dynamic shared memory
  uint32_t bars, coef, meta_c, meta_q, meta_off, part, xbuf, q, total;
};

__host__ __device__ inline MmaSmem mma_smem(const MmaPlan &p) {
  MmaSmem L;
  const uint32_t nb = 8u * p.nt;
  L.bars = 0;                                                          // full[8], empty[8], resident
  L.coef = 256;
  L.meta_c = L.coef + (uint32_t)p.K * p.KS * nb * 4 * 8;               // cs[K][KS][NB][4] doubles
  L.meta_q = L.meta_c + nb * 8;
  L.meta_off = L.meta_q + nb * 8;                                      // off[K][NB] int32
  L.part = (L.meta_off + (uint32_t)p.K * nb * 4 + 15u) & ~15u;         // part[NB][2] double2
  L.xbuf = L.part + nb * 2 * 16;
  L.q = (L.xbuf + nb * (uint32_t)p.xp * 8 + 127u) & ~127u;
  const uint32_t qbytes = p.stream ? (uint32_t)p.slots * 2u * ((uint32_t)p.tr * 16u + 64u)
                                   : (uint32_t)p.K * 2u * p.KS * (uint32_t)p.pitch_q;
  L.total = L.q + qbytes;
  return L;
}

struct MmaArgs {
  MmaPlan p;
  const unsigned char *q;          // [P][K][2 KS][pitch_q]
  Batch b;
  Workspace ws;
  double *lnL_out;
};

template <int NT, bool STREAM>
__global__ void __launch_bounds__(MM_WARPS * 32, 1) lnl_mma_kernel(const MmaArgs A) {
  constexpr int NB = 8 * NT;
  constexpr int CW = STREAM ? MM_WARPS - 1 : MM_WARPS;             // consumer warps
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const MmaPlan &P = A.p;
  const Batch &b = A.b;
  const Workspace &ws = A.ws;
  const MmaSmem L = mma_smem(P);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + L.bars);
  uint64_t *empty = full + MM_MAX_SLOTS;
  uint64_t *resbar = empty + MM_MAX_SLOTS;
  double *cs = reinterpret_cast<double *>(smem_raw + L.coef);
  double *mc = reinterpret_cast<double *>(smem_raw + L.meta_c);
  double *mq = reinterpret_cast<double *>(smem_raw + L.meta_q);
  int *moff = reinterpret_cast<int *>(smem_raw + L.meta_off);
  double2 *part = reinterpret_cast<double2 *>(smem_raw + L.part);
  double *xbuf = reinterpret_cast<double *>(smem_raw + L.xbuf);
  unsigned char *qs = smem_raw + L.q;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
  const int K = P.K, KS = P.KS, n_t = P.n_t, n_r = P.n_r, n_x = P.n_x, xp = P.xp, tr = P.tr;
  const int m2 = 2 * P.M, km2 = m2 * K;                               // doubles of coefficients per detector / sample
  const uint32_t slot_bytes = 2u * ((uint32_t)tr * 16u + 64u);
  const int n_ranges = (n_r + tr - 1) / tr;

  if (tid == 0) {
    for (int i = 0; i < MM_MAX_SLOTS; ++i) {
      mbar_init(full + i, 1);
      mbar_init(empty + i, CW);
    }
    mbar_init(resbar, 1);
  }
  for (int i = tid; i < K * KS * NB * 4; i += blockDim.x) cs[i] = 0.0;  // the pad entries of an odd mode count stay zero
  __syncthreads();

  const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x;
  const int64_t w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;

  // ---------------------------------------------------------------------------------------------- producer warp (ring)
  if (STREAM && warp == CW) {
    if (lane == 0) {
      uint32_t cnt = 0;
      for (int64_t w0 = w_begin; w0 < w_end;) {
        const int64_t seg = (b.g0 + w0) / b.n_per_seg;
        const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
        const unsigned char *qp = A.q + (int64_t)b.ids[seg] * P.point_stride;
        for (int64_t s0 = w0; s0 < run_end; s0 += NB)
          for (int k = 0; k < K; ++k)
            for (int r = 0; r < n_ranges; ++r) {
              const int r0 = r * tr;
              const uint32_t rows = (uint32_t)min(tr, n_r - r0);
              for (int s = 0; s < KS; ++s, ++cnt) {
                const uint32_t slot = cnt % (uint32_t)P.slots, ph = (cnt / (uint32_t)P.slots) & 1u;
                mbar_wait(empty + slot, ph ^ 1u);
                mbar_expect_tx(full + slot, 2u * rows * 16u);
                const unsigned char *src = qp + (size_t)(k * 2 * KS + 2 * s) * P.pitch_q + (size_t)r0 * 16;
                unsigned char *dst = qs + slot * slot_bytes;
                bulk_g2s(dst, src, rows * 16u, full + slot);
                bulk_g2s(dst + tr * 16 + 64, src + P.pitch_q, rows * 16u, full + slot);
              }
            }
        w0 = run_end;
      }
    }
    return;
  }

  // ---------------------------------------------------------------------------------------------- consumer warps
  const int lr = lane >> 2, lc = lane & 3;                       // fragment coordinates: row (A, C) / column group
  // byte offset of this lane's A element inside a k-step chunk whose mode rows are `mp` bytes apart
  const uint32_t mp = STREAM ? (uint32_t)tr * 16u + 64u : (uint32_t)P.pitch_q;
  const uint32_t a_lane = (uint32_t)(lc >> 1) * mp + (uint32_t)(lc & 1) * 8u;
  const double ln_ntau = log((double)P.n_tau);
  uint32_t cnt = 0, res_phase = 0;
  int staged_point = -1;

  for (int64_t w0 = w_begin; w0 < w_end;) {
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    if (!STREAM && point != staged_point) {
      mm_bar_consumers<CW>();                                        // every warp is done with the previous block
      if (tid == 0) stage_block(qs, A.q + (int64_t)point * P.point_stride, (uint32_t)P.point_stride, resbar);
      mbar_wait(resbar, res_phase);
      res_phase ^= 1u;
      staged_point = point;
    }

    for (int64_t s0 = w0; s0 < run_end; s0 += NB) {
      const int nvalid = (int)min((int64_t)NB, run_end - s0);
      // ---- stage the batch: coefficients as B fragments cs[k][s][n][4], c, q, target offsets
      for (int e = tid; e < NB * km2; e += CW * 32) {
        const int n = e / km2, j = e - n * km2, k = j / m2, kap = j - k * m2;
        const double v = n < nvalid ? reinterpret_cast<const double *>(ws.coef)[(s0 + n) * ws.coef_stride + j] : 0.0;
        cs[((k * KS + (kap >> 2)) * NB + n) * 4 + (kap & 3)] = v;
      }
      if (tid < NB) {
        mc[tid] = tid < nvalid ? ws.scale_c[s0 + tid] : 1.0;
        mq[tid] = tid < nvalid ? ws.quad[s0 + tid] : 0.0;
      }
      if (tid < NB * K) {
        const int k = tid / NB, n = tid - k * NB;
        int off = 0;
        if (n < nvalid) {
          const int sk = ws.shift[(s0 + n) * K + k];
          off = P.circular ? sk - ws.shift[(s0 + n) * K] : P.j0 + sk;
          if (off <= -n_t || off >= n_t) off = 0;                // only a sample with NaN angles (its lnL is NaN anyway)
        }
        moff[tid] = off;
      }
      mm_bar_consumers<CW>();

      for (int k = 0; k < K; ++k) {
        int off[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          off[nt][0] = moff[k * NB + 8 * nt + 2 * lc];
          off[nt][1] = moff[k * NB + 8 * nt + 2 * lc + 1];
        }
        for (int r = 0; r < n_ranges; ++r) {
          const int r0 = r * tr;
          const int rb0 = MM_RBW * warp;                          // first row block of this warp inside the range
          double acc[MM_RBW][NT][2];
#pragma unroll
          for (int i = 0; i < MM_RBW; ++i)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc[i][nt][0] = acc[i][nt][1] = 0.0;
          const bool active = r0 + 8 * rb0 < n_r;                 // this warp owns rows of the range
          for (int s = 0; s < KS; ++s, ++cnt) {
            const unsigned char *chunk;
            uint32_t slot = 0;
            if (STREAM) {
              slot = cnt % (uint32_t)P.slots;
              mbar_wait(full + slot, (cnt / (uint32_t)P.slots) & 1u);
              chunk = qs + slot * slot_bytes;
            } else {
              chunk = qs + (size_t)(k * 2 * KS + 2 * s) * P.pitch_q + (size_t)r0 * 16;
            }
            if (active) {
              double bf[NT];
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) bf[nt] = cs[((k * KS + s) * NB + 8 * nt + lr) * 4 + lc];
              double af[MM_RBW];
#pragma unroll
              for (int i = 0; i < MM_RBW; ++i) {
                const int row = 8 * (rb0 + i) + lr;               // rows past n_r of a short last range: clamp (masked below)
                const int rowc = r0 + row < n_r ? row : 0;
                af[i] = *reinterpret_cast<const double *>(chunk + a_lane + (uint32_t)rowc * 16u);
              }
#pragma unroll
              for (int i = 0; i < MM_RBW; ++i)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) dmma(acc[i][nt], af[i], bf[nt]);
            }
            if (STREAM) {
              __syncwarp();
              if (lane == 0) mm_arrive(empty + slot);
            }
          }
          if (active) {
            // ---- shifted write-out: x[n][(t - off) mod N_t] (+)= P_k[t, n]; all loads first, then all stores
            uint32_t idx[MM_RBW][NT][2];                              // element of xbuf, ~0 = masked
            double old[MM_RBW][NT][2];
#pragma unroll
            for (int i = 0; i < MM_RBW; ++i) {
              const int t = r0 + 8 * (rb0 + i) + lr;
#pragma unroll
              for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  int u = t - off[nt][e];
                  bool ok;
                  if (P.circular) {
                    u += u < 0 ? n_t : 0;
                    u -= u >= n_t ? n_t : 0;
                    ok = t < n_t;
                  } else {
                    ok = t < n_t && u >= 0 && u < n_x;
                  }
                  idx[i][nt][e] = ok ? (uint32_t)((8 * nt + 2 * lc + e) * xp + u) : 0xffffffffu;
                  old[i][nt][e] = 0.0;
                  if (k > 0 && ok) old[i][nt][e] = xbuf[idx[i][nt][e]];
                }
            }
#pragma unroll
            for (int i = 0; i < MM_RBW; ++i)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e)
                  if (idx[i][nt][e] != 0xffffffffu) xbuf[idx[i][nt][e]] = old[i][nt][e] + acc[i][nt][e];
          }
        }
        mm_bar_consumers<CW>();                                       // detector k is complete in every window
      }

      // ---- time marginal: portion (sample n, half h) of a window per warp, lanes over tau
      const int half = (n_x + 1) >> 1;
      for (int pi = warp; pi < 2 * NB; pi += CW) {
        const int n = pi >> 1, h = pi & 1;
        const double *xw = xbuf + n * xp;
        const int j_lo = h * half, j_hi = min(n_x, j_lo + half);
        double m = -INFINITY;
        for (int j = j_lo + lane; j < j_hi; j += 32) m = fmax(m, xw[j]);
        m = warp_max(m);
        const double cl2 = mc[n] * 1.4426950408889634;
        const double mo = -m * cl2;
        double sum = 0.0;
        for (int j = j_lo + lane; j < j_hi; j += 32) sum += mm_exp2(fma(xw[j], cl2, mo));
        sum = warp_sum(sum);
        if (lane == 0) part[pi] = make_double2(m, sum);
      }
      mm_bar_consumers<CW>();
      if (tid < nvalid) {
        const double c = mc[tid];
        const double2 p0 = part[2 * tid], p1 = part[2 * tid + 1];
        const double m = fmax(p0.x, p1.x);
        double sum = 0.0;
        if (p0.x > -INFINITY) sum += p0.y * exp(c * (p0.x - m));
        if (p1.x > -INFINITY) sum += p1.y * exp(c * (p1.x - m));
        A.lnL_out[b.g0 + s0 + tid] = c * m + log(sum) - ln_ntau - mq[tid];
      }
      // the next batch's staging overwrites cs / meta: the combine above read mc, mq, part
      mm_bar_consumers<CW>();
    }
    w0 = run_end;
  }
}

template <int NT, bool STREAM>
cudaError_t launch_t(const MmaArgs &a, int n_sm, cudaStream_t s) {
  constexpr int NB = 8 * NT;
  auto kern = lnl_mma_kernel<NT, STREAM>;
  const size_t smem = mma_smem(a.p).total;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int64_t grid = n_sm;
  const int64_t max_grid = (a.b.n + NB - 1) / NB;
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, MM_WARPS * 32, smem, s>>>(a);
  return cudaGetLastError();
}

// [rows][n_t] complex128 -> the operand layout described at the top: [P][K][M2][pitch] bytes
__global__ void convert_q_mma_kernel(const double2 *__restrict__ src, unsigned char *__restrict__ dst, int P, int K, int M,
                                     int M2, int n_t, int n_r, int pitch) {
  const int64_t per_row = pitch / 16;                                       // 16-byte units per row, pad included
  const int64_t total = (int64_t)P * K * M2 * per_row;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = i / per_row;
    const int t = (int)(i - row * per_row);
    const int m = (int)(row % M2);
    const int64_t pk = row / M2;
    double2 v = make_double2(0.0, 0.0);
    if (m < M && t < n_t) v = src[(pk * M + m) * n_t + t];
    (void)n_r;
    reinterpret_cast<double2 *>(dst)[i] = v;
  }
}

}  // namespace

size_t lnl_mma_smem_bytes(const MmaPlan &p) { return mma_smem(p).total; }

cudaError_t launch_convert_q_mma(const double *Q_c128, void *dst, const MmaPlan &p, int32_t n_points, cudaStream_t s) {
  const int64_t total = (int64_t)n_points * p.K * 2 * p.KS * (p.pitch_q / 16);
  int grid = (int)((total + 255) / 256);
  if (grid > 148 * 16) grid = 148 * 16;
  if (grid < 1) grid = 1;
  convert_q_mma_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), reinterpret_cast<unsigned char *>(dst),
                                            n_points, p.K, p.M, 2 * p.KS, p.n_t, p.n_r, p.pitch_q);
  return cudaGetLastError();
}

cudaError_t launch_lnl_mma(const MmaPlan &p, const void *q, const Batch &b, const Workspace &ws, double *lnL_out, int n_sm,
                           cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  MmaArgs a;
  a.p = p;
  a.q = reinterpret_cast<const unsigned char *>(q);
  a.b = b;
  a.ws = ws;
  a.lnL_out = lnL_out;
  if (n_launch) ++*n_launch;
  if (p.stream) {
    switch (p.nt) {
      case 1: return launch_t<1, true>(a, n_sm, s);
      case 2: return launch_t<2, true>(a, n_sm, s);
      default: return cudaErrorInvalidValue;
    }
  }
  switch (p.nt) {
    case 1: return launch_t<1, false>(a, n_sm, s);
    case 2: return launch_t<2, false>(a, n_sm, s);
    default: return cudaErrorInvalidValue;
  }
}
