// Fused lnL kernel, "direct" variant: steps a6-a7 of DESIGN.md section 1.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
// One warp per extrinsic sample, lanes over tau (j = lane + 32 i): the per-detector shift s_k is a warp-uniform
// address offset, so shared-memory reads of the staged Q window are contiguous across lanes and conflict-free.
// Each intrinsic point's Q block ([K*M][n_tp] complex) is staged in shared memory with cp.async.bulk (TMA 1-D)
// completing on an mbarrier; the time-axis max / sum are warp-shuffle reductions.  fp32 variant = reading A17.
#include "rift_internal.h"
#include "tma_utils.cuh"
#include "exp2_poly.cuh"

namespace {

constexpr int LNL_WARPS = 8;
constexpr int LNL_THREADS = LNL_WARPS * 32;
constexpr int SLOTS = 13;                       // 13 * 32 = 416 >= 411 tau samples per block
constexpr int BLOCK_T = SLOTS * 32;

template <typename Real> struct CplxOf;
template <> struct CplxOf<float> { typedef float2 type; };
template <> struct CplxOf<double> { typedef double2 type; };

// x[i] = sum_k sum_m Re(conj(B) Q)[(j0 + s_k + jb + lane + 32 i) mod N_t] for one block of 416 window entries of one sample
template <typename Real, bool QSMEM, bool EXT>
__device__ __forceinline__ void direct_block(const QStore &q, const typename CplxOf<Real>::type *Qp,
                                             const typename CplxOf<Real>::type *wcoef, const int32_t *shift, int K, int M,
                                             int j0, int jb, int lane, Real (&x)[SLOTS]) {
  typedef typename CplxOf<Real>::type CT;
#pragma unroll
  for (int i = 0; i < SLOTS; ++i) x[i] = (Real)0;
  for (int k = 0; k < K; ++k) {
    int base = (j0 + shift[k] + jb) % q.n_t;
    if (base < 0) base += q.n_t;
    int idx[SLOTS];
#pragma unroll
    for (int i = 0; i < SLOTS; ++i) {
      int t = base + lane + 32 * i;
      if (t >= q.n_t) t -= q.n_t;
      if (jb + lane + 32 * i >= q.n_tau) t = 0;       // masked slot, keep the address in range
      idx[i] = t;
    }
    if constexpr (EXT) {
      // extended rows (n_tp >= N_t + 416): the block never wraps, one address per mode row plus immediate offsets
      const CT *row = Qp + (size_t)(k * M) * q.n_tp + base + lane;
      for (int m = 0; m < M; ++m, row += q.n_tp) {
        const CT a = wcoef[k * M + m];
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) {
          const CT v = __ldg(row + 32 * i);
          x[i] = fma(a.x, v.x, x[i]);
          x[i] = fma(a.y, v.y, x[i]);
        }
      }
    } else {
      for (int m = 0; m < M; ++m) {
        const CT a = wcoef[k * M + m];
        const CT *row = Qp + (size_t)(k * M + m) * q.n_tp;
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) {
          const CT v = QSMEM ? row[idx[i]] : __ldg(row + idx[i]);
          x[i] = fma(a.x, v.x, x[i]);
          x[i] = fma(a.y, v.y, x[i]);
        }
      }
    }
  }
}

template <typename Real, bool QSMEM, bool EXT>
__global__ void __launch_bounds__(LNL_THREADS, 2)
lnl_direct_kernel(QStore q, Batch b, Workspace ws, int K, double *__restrict__ lnL_out) {
  typedef typename CplxOf<Real>::type CT;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
  CT *Qs = reinterpret_cast<CT *>(smem_raw + 128);
  const size_t q_bytes = QSMEM ? (size_t)q.point_stride_bytes : 0;
  CT *coef_s = reinterpret_cast<CT *>(smem_raw + 128 + q_bytes);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int km = q.km, M = km / K;
  CT *wcoef = coef_s + warp * km;

  // contiguous sample range of this CTA, processed as runs of equal segment
  const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x;
  const int64_t w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;

  if (QSMEM && threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();

  uint32_t phase = 0;
  int staged_point = -1;
  const int j0 = (q.n_t - q.n_tau) / 2;
  const double ln_ntau = log((double)q.n_tau);

  for (int64_t w0 = w_begin; w0 < w_end;) {
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    const CT *Qp;
    if (QSMEM) {
      if (point != staged_point) {
        __syncthreads();                                  // every warp is done with the previous window
        if (threadIdx.x == 0) {
          stage_block(Qs, reinterpret_cast<const unsigned char *>(q.data) + (int64_t)point * q.point_stride_bytes,
                      (uint32_t)q.point_stride_bytes, bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1u;
        staged_point = point;
      }
      Qp = Qs;
    } else {
      Qp = reinterpret_cast<const CT *>(reinterpret_cast<const unsigned char *>(q.data) +
                                        (int64_t)point * q.point_stride_bytes);
    }

    for (int64_t w = w0 + warp; w < run_end; w += LNL_WARPS) {   // w = workspace slot
      const double c = ws.scale_c[w];
      const double quad = ws.quad[w];
      __syncwarp();
      {
        const CT *src = reinterpret_cast<const CT *>(reinterpret_cast<const Real *>(ws.coef) + w * ws.coef_stride);
        for (int i = lane; i < km; i += 32) wcoef[i] = src[i];
      }
      __syncwarp();

      Real run_max = -INFINITY;
      double run_sum = 0.0;
      for (int jb = 0; jb < q.n_tau; jb += BLOCK_T) {
        Real x[SLOTS];
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) x[i] = (Real)0;
        for (int k = 0; k < K; ++k) {
          int base = (j0 + ws.shift[w * K + k] + jb) % q.n_t;
          if (base < 0) base += q.n_t;
          int idx[SLOTS];
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) {
            int t = base + lane + 32 * i;
            if (t >= q.n_t) t -= q.n_t;
            if (jb + lane + 32 * i >= q.n_tau) t = 0;       // masked slot, keep the address in range
            idx[i] = t;
          }
          if constexpr (EXT) {
            // extended rows (n_tp >= N_t + 416): the block never wraps, one address per mode row plus immediate offsets
            const CT *row = Qp + (size_t)(k * M) * q.n_tp + base + lane;
            for (int m = 0; m < M; ++m, row += q.n_tp) {
              const CT a = wcoef[k * M + m];
#pragma unroll
              for (int i = 0; i < SLOTS; ++i) {
                const CT v = __ldg(row + 32 * i);
                x[i] = fma(a.x, v.x, x[i]);
                x[i] = fma(a.y, v.y, x[i]);
              }
            }
          } else {
            for (int m = 0; m < M; ++m) {
              const CT a = wcoef[k * M + m];
              const CT *row = Qp + (size_t)(k * M + m) * q.n_tp;
#pragma unroll
              for (int i = 0; i < SLOTS; ++i) {
                const CT v = QSMEM ? row[idx[i]] : __ldg(row + idx[i]);
                x[i] = fma(a.x, v.x, x[i]);
                x[i] = fma(a.y, v.y, x[i]);
              }
            }
          }
        }
        Real bmax = -INFINITY;
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) {
          if (jb + lane + 32 * i >= q.n_tau) x[i] = -INFINITY;
          bmax = fmax(bmax, x[i]);
        }
        bmax = warp_max(bmax);
        double bsum;
        if (sizeof(Real) == 4) {
          const float cl2 = (float)c * 1.4426950408889634f;
          float s = 0.f;
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) s += x[i] == -INFINITY ? 0.f : fast_exp2(((float)x[i] - (float)bmax) * cl2);   // masked slot: 0 even when c = 0
          bsum = (double)s;
        } else {
          double s = 0.0;
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) s += x[i] == -INFINITY ? 0.0 : exp(c * ((double)x[i] - (double)bmax));
          bsum = s;
        }
        bsum = warp_sum(bsum);
        if (jb == 0) {                         // first block (the only one when N_tau <= 416)
          run_sum = bsum;
          run_max = bmax;
        } else if (bmax > run_max) {
          run_sum = run_sum * exp(c * ((double)run_max - (double)bmax)) + bsum;
          run_max = bmax;
        } else {
          run_sum += bsum * exp(c * ((double)bmax - (double)run_max));
        }
      }
      if (lane == 0) lnL_out[b.g0 + (ws.orig ? ws.orig[w] : w)] = c * (double)run_max + log(run_sum) - ln_ntau - quad;
    }
    w0 = run_end;
  }
}

// ---- NEXT-2: distance-marginalised variant (include/rift_ile.h: rift_ile_eval_batch_dmarg).
// The window sums x_j do not depend on the distance, so with c_i = D_ref/D_i over the nodes of a quadrature rule in ln D
//   lnL_dm = ln[(1/N_tau) sum_i W_i exp(-c_i^2 b) sum_j exp(c_i x_j)],   b = the U/V bracket of Eq. (D3) (ws.quad at c = 1).
// One warp per sample as in lnl_direct_kernel.  m = max_j x_j serves every node (c_i > 0); per chunk of 8 nodes each lane
// sums exp(c_i (x_j - m)) over its window entries, a transposed shuffle reduction leaves node n's sum on lanes 4n..4n+3, and
// lane 4n adds it to S_i in per-warp shared memory (windows longer than one block are contracted twice: once for m, once
// for the sums).  Finally R = max_i (ln W_i + c_i m - c_i^2 b) and lnL = R + ln sum_i exp(ln W_i + c_i m - c_i^2 b - R) S_i - ln N_tau.
struct DmargDev {
  int n_dist;                      // nodes, a multiple of 8
  const double *c, *lnw;           // device [n_dist]: D_ref / D_i, ln W_i
};

template <typename Real, typename Op>
__device__ __forceinline__ Real treduce8r(const Real (&v)[8], int lane, Op op) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  Real w4[4], w2[2];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const Real send = b4 ? v[j] : v[j + 4], keep = b4 ? v[j + 4] : v[j];
    w4[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 16));
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const Real send = b3 ? w4[j] : w4[j + 2], keep = b3 ? w4[j + 2] : w4[j];
    w2[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 8));
  }
  const Real send = b2 ? w2[0] : w2[1], keep = b2 ? w2[1] : w2[0];
  Real w = op(keep, __shfl_xor_sync(0xffffffffu, send, 4));
  w = op(w, __shfl_xor_sync(0xffffffffu, w, 2));
  w = op(w, __shfl_xor_sync(0xffffffffu, w, 1));
  return w;                        // lanes 4n .. 4n+3 hold the reduction of v[n]
}

template <typename Real, bool QSMEM, bool EXT>
__global__ void __launch_bounds__(LNL_THREADS, 2)   // two blocks per SM when two Q blocks fit: the fp64 node sums are latency-bound
lnl_direct_dm_kernel(QStore q, Batch b, Workspace ws, int K, DmargDev dm, double *__restrict__ lnL_out) {
  typedef typename CplxOf<Real>::type CT;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
  CT *Qs = reinterpret_cast<CT *>(smem_raw + 128);
  const size_t q_bytes = QSMEM ? (size_t)q.point_stride_bytes : 0;
  CT *coef_s = reinterpret_cast<CT *>(smem_raw + 128 + q_bytes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int km = q.km, M = km / K, nd = dm.n_dist;
  CT *wcoef = coef_s + warp * km;
  Real *cl2_s = reinterpret_cast<Real *>(coef_s + LNL_WARPS * km);          // [nd] c_i log2(e)
  Real *S_s = cl2_s + nd + (size_t)warp * nd;                               // [warps][nd] sums over the window

  const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x;
  const int64_t w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;
  if (QSMEM && threadIdx.x == 0) mbar_init(bar, 1);
  for (int i = threadIdx.x; i < nd; i += LNL_THREADS) cl2_s[i] = (Real)(dm.c[i] * 1.4426950408889634);
  __syncthreads();

  uint32_t phase = 0;
  int staged_point = -1;
  const int j0 = (q.n_t - q.n_tau) / 2;
  const double ln_ntau = log((double)q.n_tau);
  const bool single = q.n_tau <= BLOCK_T;

  for (int64_t w0 = w_begin; w0 < w_end;) {
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    const CT *Qp;
    if (QSMEM) {
      if (point != staged_point) {
        __syncthreads();
        if (threadIdx.x == 0)
          stage_block(Qs, reinterpret_cast<const unsigned char *>(q.data) + (int64_t)point * q.point_stride_bytes,
                      (uint32_t)q.point_stride_bytes, bar);
        mbar_wait(bar, phase);
        phase ^= 1u;
        staged_point = point;
      }
      Qp = Qs;
    } else {
      Qp = reinterpret_cast<const CT *>(reinterpret_cast<const unsigned char *>(q.data) + (int64_t)point * q.point_stride_bytes);
    }

    for (int64_t w = w0 + warp; w < run_end; w += LNL_WARPS) {
      const double bq = ws.quad[w];                                         // b (geometry ran at D = D_ref, c = 1)
      const bool bad = !(ws.scale_c[w] == ws.scale_c[w]);                   // NaN marks an invalid sample
      __syncwarp();
      {
        const CT *src = reinterpret_cast<const CT *>(reinterpret_cast<const Real *>(ws.coef) + w * ws.coef_stride);
        for (int i = lane; i < km; i += 32) wcoef[i] = src[i];
        for (int i = lane; i < nd; i += 32) S_s[i] = (Real)0;
      }
      __syncwarp();
      const int32_t *shift = ws.shift + w * K;
      Real x[SLOTS];
      Real m = -INFINITY;
      for (int jb = 0; jb < q.n_tau; jb += BLOCK_T) {                       // pass 1: the window maximum
        direct_block<Real, QSMEM, EXT>(q, Qp, wcoef, shift, K, M, j0, jb, lane, x);
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) {
          if (jb + lane + 32 * i >= q.n_tau) x[i] = -INFINITY;
          m = fmax(m, x[i]);
        }
      }
      m = warp_max(m);
      for (int jb = 0; jb < q.n_tau; jb += BLOCK_T) {                       // pass 2: sums per node
        if (!single) {
          direct_block<Real, QSMEM, EXT>(q, Qp, wcoef, shift, K, M, j0, jb, lane, x);
#pragma unroll
          for (int i = 0; i < SLOTS; ++i)
            if (jb + lane + 32 * i >= q.n_tau) x[i] = -INFINITY;
        }
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) x[i] -= m;                          // <= 0, -inf for masked slots
        for (int ch = 0; ch < nd; ch += 8) {
          Real cq[8], s[8];
#pragma unroll
          for (int n = 0; n < 8; ++n) {
            cq[n] = cl2_s[ch + n];
            s[n] = (Real)0;
          }
          if (sizeof(Real) == 4) {
            // a slot (32 consecutive window entries, one per lane) whose largest exponent over the chunk's nodes lies below -40
            // is skipped by the whole warp: every window sum is >= 1 (the maximum entry), so the dropped terms change it by
            // < N_tau 2^-40 relative.  Near nodes (large c) skip all slots but those around the peak: 1.4x on C1
            Real cmin = cq[0];
#pragma unroll
            for (int n = 1; n < 8; ++n) cmin = fmin(cmin, cq[n]);
#pragma unroll
            for (int i = 0; i < SLOTS; ++i) {
              if (!__any_sync(0xffffffffu, x[i] * cmin > (Real)-40)) continue;
#pragma unroll
              for (int n = 0; n < 8; ++n) s[n] += (Real)fast_exp2((float)x[i] * (float)cq[n]);
            }
          } else {
            // fp64: all terms are kept -- the same skip (tried at 2^-45) breaks the 13 x 8 independent polynomial chains into
            // groups of 8 and measured slower (119 against 97 ms on C1)
#pragma unroll
            for (int i = 0; i < SLOTS; ++i)
#pragma unroll
              for (int n = 0; n < 8; ++n)                          // a masked entry (-inf) becomes 2^-1000 p(r): a relative 1e-301
                s[n] += (Real)poly_exp2(fmax((double)x[i] * (double)cq[n], -1100.0));
          }
          const Real tot = treduce8r(s, lane, [](Real a, Real c) { return a + c; });
          if ((lane & 3) == 0) S_s[ch + (lane >> 2)] += tot;
        }
      }
      __syncwarp();
      // ---- sum over the nodes in fp64: e_i = ln W_i + c_i m - c_i^2 b
      double R = -INFINITY;
      for (int i = lane; i < nd; i += 32) {
        const double c = dm.c[i];
        R = fmax(R, dm.lnw[i] + c * (double)m - c * c * bq);
      }
      R = warp_max(R);
      double tot = 0.0;
      for (int i = lane; i < nd; i += 32) {
        const double c = dm.c[i];
        tot += exp(dm.lnw[i] + c * (double)m - c * c * bq - R) * (double)S_s[i];
      }
      tot = warp_sum(tot);
      if (lane == 0) lnL_out[b.g0 + w] = bad ? __longlong_as_double(0x7ff8000000000000ll) : R + log(tot) - ln_ntau;
    }
    w0 = run_end;
  }
}

template <typename Real, bool QSMEM, bool EXT = false>
cudaError_t launch_dm_t(const QStore &q, const Batch &b, const Workspace &ws, int K, const DmargDev &dm, double *lnL_out,
                        int n_sm, size_t smem, cudaStream_t s) {
  auto kern = lnl_direct_dm_kernel<Real, QSMEM, EXT>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, LNL_THREADS, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)n_sm * occ;
  const int64_t max_grid = (b.n + LNL_WARPS - 1) / LNL_WARPS;
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, LNL_THREADS, smem, s>>>(q, b, ws, K, dm, lnL_out);
  return cudaGetLastError();
}

template <typename Real, bool QSMEM, bool EXT = false>
cudaError_t launch_t(const QStore &q, const Batch &b, const Workspace &ws, int K, double *lnL_out, int n_sm,
                     size_t smem, cudaStream_t s) {
  auto kern = lnl_direct_kernel<Real, QSMEM, EXT>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, LNL_THREADS, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)n_sm * occ;
  const int64_t max_grid = (b.n + LNL_WARPS - 1) / LNL_WARPS;
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, LNL_THREADS, smem, s>>>(q, b, ws, K, lnL_out);
  return cudaGetLastError();
}

}  // namespace

size_t lnl_direct_smem_bytes(const QStore &q, bool fp32, bool q_in_smem) {
  const size_t csz = fp32 ? 8 : 16;
  return 128 + (q_in_smem ? (size_t)q.point_stride_bytes : 0) + (size_t)LNL_WARPS * q.km * csz;
}

cudaError_t launch_lnl_direct(const QStore &q, bool fp32, bool q_in_smem, bool q_ext, const Batch &b, const Workspace &ws,
                              int n_det, double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  const size_t smem = lnl_direct_smem_bytes(q, fp32, q_in_smem);
  if (n_launch) ++*n_launch;
  if (q_ext && !q_in_smem)
    return fp32 ? launch_t<float, false, true>(q, b, ws, n_det, lnL_out, n_sm, smem, s)
                : launch_t<double, false, true>(q, b, ws, n_det, lnL_out, n_sm, smem, s);
  if (fp32)
    return q_in_smem ? launch_t<float, true>(q, b, ws, n_det, lnL_out, n_sm, smem, s)
                     : launch_t<float, false>(q, b, ws, n_det, lnL_out, n_sm, smem, s);
  return q_in_smem ? launch_t<double, true>(q, b, ws, n_det, lnL_out, n_sm, smem, s)
                   : launch_t<double, false>(q, b, ws, n_det, lnL_out, n_sm, smem, s);
}

size_t lnl_direct_dm_smem_bytes(const QStore &q, bool fp32, bool q_in_smem, int n_dist) {
  return lnl_direct_smem_bytes(q, fp32, q_in_smem) + (size_t)(1 + LNL_WARPS) * n_dist * (fp32 ? 4 : 8);
}

cudaError_t launch_lnl_direct_dmarg(const QStore &q, bool fp32, bool q_in_smem, bool q_ext, const Batch &b,
                                    const Workspace &ws, int n_det, int n_dist, const double *c_nodes, const double *lnw_nodes,
                                    double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  const size_t smem = lnl_direct_dm_smem_bytes(q, fp32, q_in_smem, n_dist);
  DmargDev dm;
  dm.n_dist = n_dist;
  dm.c = c_nodes;
  dm.lnw = lnw_nodes;
  if (n_launch) ++*n_launch;
  if (q_ext && !q_in_smem)
    return fp32 ? launch_dm_t<float, false, true>(q, b, ws, n_det, dm, lnL_out, n_sm, smem, s)
                : launch_dm_t<double, false, true>(q, b, ws, n_det, dm, lnL_out, n_sm, smem, s);
  if (fp32)
    return q_in_smem ? launch_dm_t<float, true>(q, b, ws, n_det, dm, lnL_out, n_sm, smem, s)
                     : launch_dm_t<float, false>(q, b, ws, n_det, dm, lnL_out, n_sm, smem, s);
  return q_in_smem ? launch_dm_t<double, true>(q, b, ws, n_det, dm, lnL_out, n_sm, smem, s)
                   : launch_dm_t<double, false>(q, b, ws, n_det, dm, lnL_out, n_sm, smem, s);
}
