// Fused lnL kernel, "direct" variant: steps a6-a7 of DESIGN.md section 1.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
// One warp per extrinsic sample, lanes over tau (j = lane + 32 i): the per-detector shift s_k is a warp-uniform
// address offset, so shared-memory reads of the staged Q window are contiguous across lanes and conflict-free.
// Each intrinsic point's Q block ([K*M][n_tp] complex) is staged in shared memory with cp.async.bulk (TMA 1-D)
// completing on an mbarrier; the time-axis max / sum are warp-shuffle reductions.  fp32 variant = reading A17.
#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

constexpr int LNL_WARPS = 8;
constexpr int LNL_THREADS = LNL_WARPS * 32;
constexpr int SLOTS = 13;                       // 13 * 32 = 416 >= 411 tau samples per block
constexpr int BLOCK_T = SLOTS * 32;

template <typename Real> struct CplxOf;
template <> struct CplxOf<float> { typedef float2 type; };
template <> struct CplxOf<double> { typedef double2 type; };

template <typename Real, bool QSMEM, bool EXT>
__global__ void __launch_bounds__(LNL_THREADS)
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
          for (int i = 0; i < SLOTS; ++i) s += fast_exp2(((float)x[i] - (float)bmax) * cl2);
          bsum = (double)s;
        } else {
          double s = 0.0;
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) s += exp(c * ((double)x[i] - (double)bmax));
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
