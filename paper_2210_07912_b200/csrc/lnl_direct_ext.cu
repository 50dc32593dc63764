// Fused lnL kernel, "direct, extended window" variant: steps a6-a7 of DESIGN.md section 1.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
// One warp per extrinsic sample, lanes over tau (j = lane + 32 i).  Q of the intrinsic point is staged by 1-D TMA in
// the interleaved layout with a circular extension ([K*M][n_te] complex, n_te >= N_t + 416), so the (j0 + s_k + j) mod
// N_t of a 416-sample block is ONE warp-uniform base plus immediate offsets: per mode row 13 conflict-free LDS.64 and 26
// FMAs, with the next row's loads issued under the current row's FMAs.  The kernel is bound by shared-memory bandwidth
// (8 B per lane per 2 FMAs = 2 wavefronts per LDS.64): 25 % of the FP32 pipe at best.
#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

constexpr int E_WARPS = 8;
constexpr int E_THREADS = E_WARPS * 32;
constexpr int SLOTS = RIFT_EXT / 32;            // 13

__device__ __forceinline__ float2 lds_c(uint32_t addr, float) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ double2 lds_c(uint32_t addr, double) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
template <typename Real> struct C2;
template <> struct C2<float> { typedef float2 type; };
template <> struct C2<double> { typedef double2 type; };

template <typename Real, typename CT>
__device__ __forceinline__ void load_row(CT (&v)[SLOTS], uint32_t addr) {
#pragma unroll
  for (int i = 0; i < SLOTS; ++i) v[i] = lds_c(addr + (uint32_t)(i * 32 * sizeof(CT)), Real());
}
template <typename Real, typename CT>
__device__ __forceinline__ void fma_row(Real (&x)[SLOTS], const CT (&v)[SLOTS], CT a) {
#pragma unroll
  for (int i = 0; i < SLOTS; ++i) {
    x[i] = fma(a.x, v[i].x, x[i]);
    x[i] = fma(a.y, v[i].y, x[i]);
  }
}

template <typename Real>
__global__ void __launch_bounds__(E_THREADS, (sizeof(Real) == 4 ? 2 : 1))
lnl_direct_ext_kernel(QStore q, Batch b, Workspace ws, int K, double *__restrict__ lnL_out) {
  typedef typename C2<Real>::type CT;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
  CT *Qs = reinterpret_cast<CT *>(smem_raw + 128);
  CT *coef_s = reinterpret_cast<CT *>(smem_raw + 128 + q.point_stride_bytes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int km = q.km, M = km / K;
  CT *wcoef = coef_s + warp * (2 * km);           // [2][km], double-buffered
  const uint32_t wcoef_addr = smem_u32(wcoef);
  const uint32_t q_addr = smem_u32(Qs);
  uint32_t row_bytes = (uint32_t)(q.n_tp * sizeof(CT));
  asm volatile("" : "+r"(row_bytes));

  const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x;
  const int64_t w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  uint32_t phase = 0;
  int staged_point = -1;
  const int j0 = (q.n_t - q.n_tau) / 2;
  const double ln_ntau = log((double)q.n_tau);

  for (int64_t w0 = w_begin; w0 < w_end;) {
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    if (point != staged_point) {
      __syncthreads();                                    // every warp is done with the previous window
      if (threadIdx.x == 0)
        stage_block(Qs, reinterpret_cast<const unsigned char *>(q.data) + (int64_t)point * q.point_stride_bytes,
                    (uint32_t)q.point_stride_bytes, bar);
      mbar_wait(bar, phase);
      phase ^= 1u;
      staged_point = point;
    }

    // The NEXT sample's scalars are prefetched into registers and its coefficient vector into the other half of the
    // per-warp shared buffer (cp.async) while the current sample is evaluated.
    auto fetch_coef = [&](int64_t w, int buf) {
      const CT *src = reinterpret_cast<const CT *>(reinterpret_cast<const Real *>(ws.coef) + w * ws.coef_stride);
      for (int i = lane; i < km; i += 32) {
        const uint32_t dst = wcoef_addr + (uint32_t)((buf * km + i) * sizeof(CT));
        if (sizeof(CT) == 8)
          asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src + i) : "memory");
        else
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + i) : "memory");
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    };
    int buf = 0;
    int64_t w = w0 + warp;
    double n_c = 0.0, n_quad = 0.0;
    int n_shift = 0;
    if (w < run_end) {
      n_c = ws.scale_c[w];
      n_quad = ws.quad[w];
      n_shift = (lane < K) ? ws.shift[w * K + lane] : 0;
      fetch_coef(w, buf);
    }
    for (; w < run_end; w += E_WARPS, buf ^= 1) {                // w = workspace slot
      const double c = n_c, quad = n_quad;
      const int my_shift = n_shift;
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const int64_t wn = w + E_WARPS;
      if (wn < run_end) {
        n_c = ws.scale_c[wn];
        n_quad = ws.quad[wn];
        n_shift = (lane < K) ? ws.shift[wn * K + lane] : 0;
        fetch_coef(wn, buf ^ 1);
      }
      const uint32_t wc_addr = wcoef_addr + (uint32_t)(buf * km * sizeof(CT));

      Real run_max = -INFINITY;
      double run_sum = 0.0;
      for (int jb = 0; jb < q.n_tau; jb += RIFT_EXT) {
        Real x[SLOTS];
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) x[i] = (Real)0;
#pragma unroll 1
        for (int k = 0; k < K; ++k) {
          int base = (j0 + __shfl_sync(0xffffffffu, my_shift, k) + jb) % q.n_t;
          if (base < 0) base += q.n_t;
          uint32_t addr = q_addr + (uint32_t)((k * M) * q.n_tp + base + lane) * (uint32_t)sizeof(CT);
          uint32_t caddr = wc_addr + (uint32_t)(k * M * sizeof(CT));
          CT va[SLOTS], vb[SLOTS];
          load_row<Real>(va, addr);
#pragma unroll 1
          for (int m = 0; m < M; m += 2) {
            const CT a0 = lds_c(caddr, Real());
            if (m + 1 < M) load_row<Real>(vb, addr + row_bytes);
            fma_row<Real>(x, va, a0);
            if (m + 1 < M) {
              const CT a1 = lds_c(caddr + (uint32_t)sizeof(CT), Real());
              if (m + 2 < M) load_row<Real>(va, addr + 2 * row_bytes);
              fma_row<Real>(x, vb, a1);
            }
            addr += 2 * row_bytes;
            caddr += 2 * (uint32_t)sizeof(CT);
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
          const float off = (float)bmax * cl2;
          float s0 = 0.f, s1 = 0.f;
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) {
            const float e = x[i] == -INFINITY ? 0.f : fast_exp2(fmaf((float)x[i], cl2, -off));   // masked slot: 0 even when c = 0
            if (i & 1) s1 += e; else s0 += e;
          }
          bsum = (double)(s0 + s1);
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
      if (lane == 0) {
        // ln of the sum of exponentials (1 <= sum <= N_tau): logf is accurate to ~1e-6 absolute here (reading B5)
        const double ls = (sizeof(Real) == 4) ? (double)logf((float)run_sum) : log(run_sum);
        lnL_out[b.g0 + (ws.orig ? ws.orig[w] : w)] = c * (double)run_max + ls - ln_ntau - quad;
      }
    }
    w0 = run_end;
  }
}

template <typename Real>
cudaError_t launch_t(const QStore &q, const Batch &b, const Workspace &ws, int K, double *lnL_out, int n_sm,
                     size_t smem, cudaStream_t s) {
  auto kern = lnl_direct_ext_kernel<Real>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, E_THREADS, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)n_sm * occ;
  const int64_t max_grid = (b.n + E_WARPS - 1) / E_WARPS;
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, E_THREADS, smem, s>>>(q, b, ws, K, lnL_out);
  return cudaGetLastError();
}

}  // namespace

size_t lnl_direct_ext_smem_bytes(const QStore &q, bool fp32) {
  const size_t csz = fp32 ? 8 : 16;
  return 128 + (size_t)q.point_stride_bytes + (size_t)E_WARPS * 2 * q.km * csz;
}

cudaError_t launch_lnl_direct_ext(const QStore &q, bool fp32, const Batch &b, const Workspace &ws, int n_det,
                                  double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  const size_t smem = lnl_direct_ext_smem_bytes(q, fp32);
  if (n_launch) ++*n_launch;
  return fp32 ? launch_t<float>(q, b, ws, n_det, lnL_out, n_sm, smem, s)
              : launch_t<double>(q, b, ws, n_det, lnL_out, n_sm, smem, s);
}
