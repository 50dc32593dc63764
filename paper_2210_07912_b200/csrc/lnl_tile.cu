// Fused lnL kernel, register-tiled fp64 variant: steps a6-a7 of DESIGN.md section 1 for the fp64 mode.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// Same decomposition as the tensor-core kernel (lnl_tc.cu), with the contraction on the FP64 FMA pipe (there is no fp64
// tcgen05 path): per detector, P_k[t, n] = sum_lm (B.re Q.re + B.im Q.im)[t] in UNSHIFTED detector time as a register
// tile -- a thread owns 4 time rows (t = T + 128 i) x 8 samples, so every Q value read from shared memory feeds 8 samples
// and every coefficient (a warp-wide broadcast read) feeds 4 rows: 64 DFMA per 12 shared-memory loads instead of 2 DFMA
// per load in the direct kernel.  In circular mode (N_tau = N_t) x[t] = P_0[t] + sum_{k>=1} P_k[(t + s_k - s_0) mod N_t]; the
// per-sample shift is applied by a shared-memory exchange, one detector at a time (Xb[n][t + H] with wrap-around copies
// inside the halo, read back at t + d + H: consecutive lanes, conflict-free).  The time marginal is reduced per warp
// (32 lanes x 4 rows) to (max, sum) pairs; one lane per sample combines the four warps of the warpgroup and writes lnL.
//
// CTA = 2 independent warpgroups of 4 warps (8 samples per batch each) sharing the staged Q block of the intrinsic point
// (interleaved complex128 [K*M][n_tp], 1-D bulk copy on an mbarrier).
#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

constexpr int TL_THREADS = 256;
constexpr int TL_NS = 8;              // samples per warpgroup batch
constexpr int TL_ROWS = 4;            // time rows per thread (tiles of 128)

__device__ __forceinline__ void tl_bar(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }

// exp(z) for z <= 0 to ~1e-13 relative: z = (64 n + j) ln2/64 + r, |r| <= ln2/128, e^r by a degree-5 polynomial,
// 2^(j/64) from a 64-entry table, 2^n through the exponent field.  Flushes to 0 below z = -700.
__device__ __forceinline__ double tl_exp(double z, const double *__restrict__ tab) {
  if (!(z > -700.0)) return (z != z) ? z : 0.0;
  const double kf = rint(z * 92.332482616893656);                            // 64 / ln 2
  const int k = (int)kf;
  const double r = fma(kf, -2.9815858269852933e-12, fma(kf, -0.01083042469326756, z));   // ln2/64 = hi (32 bits) + lo
  const double p = fma(fma(fma(fma(fma(1.0 / 120.0, r, 1.0 / 24.0), r, 1.0 / 6.0), r, 0.5), r, 1.0), r, 1.0);
  const double t = tab[k & 63];
  const long long bits = __double_as_longlong(t * p) + ((long long)(k >> 6) << 52);
  return __longlong_as_double(bits);
}

struct TileArgs {
  QStore q;
  Batch b;
  Workspace ws;
  int K, H, pitch;
  int dmax[RIFT_MAX_DET];
  const double *exp_tab;            // [64] 2^(j/64)
  double *lnL_out;
};

// byte offsets inside dynamic shared memory (host and device agree through this one function)
struct TileSmem {
  size_t q, tab, wg0, wg_stride, coef, meta, xb, part, total;
};
__host__ __device__ inline TileSmem tile_smem(size_t q_bytes, int km, int K, int pitch) {
  TileSmem L;
  L.q = 128;
  L.tab = L.q + ((q_bytes + 127) & ~(size_t)127);
  L.wg0 = L.tab + 512;
  L.coef = 0;                                                    // [2][km][8] double2
  L.meta = L.coef + (size_t)2 * km * TL_NS * 16;                  // [2] { c[8], quad[8] double; dsh[RIFT_MAX_DET][8] int }
  L.xb = L.meta + (size_t)2 * (16 * 8 + RIFT_MAX_DET * TL_NS * 4);
  L.part = L.xb + (size_t)TL_NS * pitch * 8;                      // [4][8] double2
  L.wg_stride = (L.part + 4 * TL_NS * 16 + 127) & ~(size_t)127;
  L.total = L.wg0 + 2 * L.wg_stride;
  (void)K;
  return L;
}

// 8 doubles per thread reduced across the warp with "transposed" butterflies; lane l ends with value n = l >> 2
template <typename Op>
__device__ __forceinline__ double treduce8d(const double (&v)[8], int lane, Op op) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  double w4[4], w2[2];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const double send = b4 ? v[j] : v[j + 4], keep = b4 ? v[j + 4] : v[j];
    w4[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 16));
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const double send = b3 ? w4[j] : w4[j + 2], keep = b3 ? w4[j + 2] : w4[j];
    w2[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 8));
  }
  const double send = b2 ? w2[0] : w2[1], keep = b2 ? w2[1] : w2[0];
  double w = op(keep, __shfl_xor_sync(0xffffffffu, send, 4));
  w = op(w, __shfl_xor_sync(0xffffffffu, w, 2));
  w = op(w, __shfl_xor_sync(0xffffffffu, w, 1));
  return w;
}

constexpr int TL_CF_MAX = 4;         // coefficient elements a thread prefetches per batch: 8 km <= 128 * TL_CF_MAX

__global__ void __launch_bounds__(TL_THREADS, 1) lnl_tile_kernel(const TileArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const QStore &q = A.q;
  const Batch &b = A.b;
  const Workspace &ws = A.ws;
  const int K = A.K, km = q.km, M = km / K, n_t = q.n_t, H = A.H, pitch = A.pitch;
  const TileSmem L = tile_smem((size_t)q.point_stride_bytes, km, K, pitch);
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
  const double2 *Qs = reinterpret_cast<const double2 *>(smem_raw + L.q);
  double *tab = reinterpret_cast<double *>(smem_raw + L.tab);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wg = warp >> 2, qw = warp & 3, tw = threadIdx.x & 127;          // warpgroup, warp in it, thread in it
  unsigned char *wgs = smem_raw + L.wg0 + wg * L.wg_stride;
  double2 *coef_s = reinterpret_cast<double2 *>(wgs + L.coef);
  unsigned char *meta_s = wgs + L.meta;
  double *xb = reinterpret_cast<double *>(wgs + L.xb);
  double2 *part = reinterpret_cast<double2 *>(wgs + L.part);
  constexpr int META_BYTES = 16 * 8 + RIFT_MAX_DET * TL_NS * 4;

  if (threadIdx.x == 0) mbar_init(bar, 1);
  if (threadIdx.x < 64) tab[threadIdx.x] = A.exp_tab[threadIdx.x];
  __syncthreads();

  const int T = 32 * qw + lane;
  int trow[TL_ROWS];                                                        // rows of this thread, clamped for reads
  bool tvalid[TL_ROWS];
#pragma unroll
  for (int i = 0; i < TL_ROWS; ++i) {
    tvalid[i] = 128 * i + T < n_t;
    trow[i] = tvalid[i] ? 128 * i + T : n_t - 1;
  }
  const double ln_nt = log((double)n_t);

  const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x;
  const int64_t w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;
  uint32_t phase = 0;
  int staged_point = -1;

  for (int64_t w0 = w_begin; w0 < w_end;) {
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    if (point != staged_point) {
      __syncthreads();                                    // both warpgroups are done with the previous window
      if (threadIdx.x == 0)
        stage_block(smem_raw + L.q, reinterpret_cast<const unsigned char *>(q.data) + (int64_t)point * q.point_stride_bytes,
                    (uint32_t)q.point_stride_bytes, bar);
      mbar_wait(bar, phase);
      phase ^= 1u;
      staged_point = point;
    }

    // ---- prefetch of one batch's per-sample data into registers, commit to the shared buffers of parity `buf`
    double2 cf[TL_CF_MAX];
    double m_c = 0.0, m_q = 0.0;
    int m_d = 0, m_d0 = 0;
    auto fetch = [&](int64_t s0) {
      const int nvalid = (int)min((int64_t)TL_NS, run_end - s0);
#pragma unroll
      for (int e4 = 0; e4 < TL_CF_MAX; ++e4) {
        const int e = tw + 128 * e4;
        cf[e4] = make_double2(0.0, 0.0);
        if (e < TL_NS * km) {
          const int n = e / km, ka = e - n * km;
          if (n < nvalid)
            cf[e4] = *reinterpret_cast<const double2 *>(reinterpret_cast<const double *>(ws.coef) + (s0 + n) * ws.coef_stride + 2 * ka);
        }
      }
      m_c = 0.0, m_q = 0.0, m_d = 0, m_d0 = 0;
      if (tw < TL_NS && tw < nvalid) {
        m_c = ws.scale_c[s0 + tw];
        m_q = ws.quad[s0 + tw];
      }
      if (tw < TL_NS * K) {
        const int k = tw / TL_NS, n = tw - k * TL_NS;
        if (n < nvalid) {
          m_d = ws.shift[(s0 + n) * K + k];
          m_d0 = ws.shift[(s0 + n) * K];
        }
      }
    };
    auto commit = [&](int buf) {
      double2 *cs = coef_s + (size_t)buf * km * TL_NS;
#pragma unroll
      for (int e4 = 0; e4 < TL_CF_MAX; ++e4) {
        const int e = tw + 128 * e4;
        if (e < TL_NS * km) {
          const int n = e / km, ka = e - n * km;
          cs[ka * TL_NS + n] = cf[e4];
        }
      }
      double *mc = reinterpret_cast<double *>(meta_s + (size_t)buf * META_BYTES);
      int *md = reinterpret_cast<int *>(mc + 16);
      if (tw < TL_NS) {
        mc[tw] = m_c;
        mc[8 + tw] = m_q;
      }
      if (tw < TL_NS * K) md[tw] = m_d - m_d0;                              // [k][n], relative to detector 0
    };

    int buf = 0;
    int64_t s0 = w0 + (int64_t)wg * TL_NS;
    if (s0 < run_end) {
      fetch(s0);
      commit(0);
    }
    tl_bar(1 + wg);
    for (; s0 < run_end; s0 += 2 * TL_NS, buf ^= 1) {
      const int64_t s_next = s0 + 2 * TL_NS;
      if (s_next < run_end) fetch(s_next);                                  // in flight during this batch
      const double2 *cs = coef_s + (size_t)buf * km * TL_NS;
      const double *mc = reinterpret_cast<const double *>(meta_s + (size_t)buf * META_BYTES);
      const int *md = reinterpret_cast<const int *>(mc + 16);

      // register-tiled contraction of one detector: acc[i][n] += sum_a B.re Q.re + B.im Q.im
      auto gemm = [&](int k, double (&acc)[TL_ROWS][TL_NS]) {
        const double2 *qrow = Qs + (size_t)(k * M) * q.n_tp;
        const double2 *cv = cs + (k * M) * TL_NS;
#pragma unroll 1
        for (int a = 0; a < M; ++a, qrow += q.n_tp, cv += TL_NS) {
          double2 qv[TL_ROWS];
#pragma unroll
          for (int i = 0; i < TL_ROWS; ++i) qv[i] = qrow[trow[i]];
#pragma unroll
          for (int n = 0; n < TL_NS; ++n) {
            const double2 c2 = cv[n];
#pragma unroll
            for (int i = 0; i < TL_ROWS; ++i) acc[i][n] = fma(c2.y, qv[i].y, fma(c2.x, qv[i].x, acc[i][n]));
          }
        }
      };

      double x[TL_ROWS][TL_NS];
#pragma unroll
      for (int i = 0; i < TL_ROWS; ++i)
#pragma unroll
        for (int n = 0; n < TL_NS; ++n) x[i][n] = 0.0;
      gemm(0, x);
      for (int k = 1; k < K; ++k) {
        double p[TL_ROWS][TL_NS];
#pragma unroll
        for (int i = 0; i < TL_ROWS; ++i)
#pragma unroll
          for (int n = 0; n < TL_NS; ++n) p[i][n] = 0.0;
        gemm(k, p);
        tl_bar(1 + wg);                                                     // the exchange buffer is free
        const int dm = A.dmax[k];
#pragma unroll
        for (int i = 0; i < TL_ROWS; ++i) {
          const int t = 128 * i + T;
          if (tvalid[i]) {
            double *dst = xb + t + H;
#pragma unroll
            for (int n = 0; n < TL_NS; ++n) dst[n * pitch] = p[i][n];
            if (t < dm) {
#pragma unroll
              for (int n = 0; n < TL_NS; ++n) dst[n * pitch + n_t] = p[i][n];
            }
            if (t >= n_t - dm) {
#pragma unroll
              for (int n = 0; n < TL_NS; ++n) dst[n * pitch - n_t] = p[i][n];
            }
          }
        }
        tl_bar(1 + wg);                                                     // exchange rows complete
#pragma unroll
        for (int n = 0; n < TL_NS; ++n) {
          const double *src = xb + n * pitch + H + md[k * TL_NS + n];
#pragma unroll
          for (int i = 0; i < TL_ROWS; ++i) x[i][n] += src[trow[i]];
        }
      }

      // time marginal: per-warp (max, sum of exp) for the 8 samples
      double mloc[TL_NS];
#pragma unroll
      for (int n = 0; n < TL_NS; ++n) {
        double mm = -INFINITY;
#pragma unroll
        for (int i = 0; i < TL_ROWS; ++i) {
          if (!tvalid[i]) x[i][n] = -INFINITY;
          mm = fmax(mm, x[i][n]);
        }
        mloc[n] = mm;
      }
      const double mine = treduce8d(mloc, lane, [](double a, double c) { return fmax(a, c); });
      double sums[TL_NS];
#pragma unroll
      for (int n = 0; n < TL_NS; ++n) {
        const double mx = __shfl_sync(0xffffffffu, mine, n << 2);
        const double c = mc[n];
        double sacc = 0.0;
#pragma unroll
        for (int i = 0; i < TL_ROWS; ++i) sacc += (mx == -INFINITY) ? 0.0 : tl_exp(c * (x[i][n] - mx), tab);
        sums[n] = sacc;
      }
      const double ssum = treduce8d(sums, lane, [](double a, double c) { return a + c; });
      if ((lane & 3) == 0) part[qw * TL_NS + (lane >> 2)] = make_double2(mine, ssum);
      tl_bar(1 + wg);                                                       // partials of the four warps are visible
      if (qw == 0 && lane < TL_NS && s0 + lane < run_end) {
        const double c = mc[lane];
        double mm = -INFINITY;
#pragma unroll
        for (int w4 = 0; w4 < 4; ++w4) mm = fmax(mm, part[w4 * TL_NS + lane].x);
        double sum = 0.0;
#pragma unroll
        for (int w4 = 0; w4 < 4; ++w4) {
          const double2 pw = part[w4 * TL_NS + lane];
          if (pw.x > -INFINITY) sum += pw.y * exp(c * (pw.x - mm));
        }
        A.lnL_out[b.g0 + s0 + lane] = c * mm + log(sum) - ln_nt - mc[8 + lane];
      }
      if (s_next < run_end) commit(buf ^ 1);
      tl_bar(1 + wg);                                                       // next batch's data visible, partials consumed
    }
    w0 = run_end;
  }
}

}  // namespace

size_t lnl_tile_smem_bytes(const QStore &q, int K, int pitch) {
  return tile_smem((size_t)q.point_stride_bytes, q.km, K, pitch).total;
}

cudaError_t launch_lnl_tile(const QStore &q, const Batch &b, const Workspace &ws, int K, int H, int pitch, const int *dmax,
                            const double *exp_tab, double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  if (TL_NS * q.km > 128 * TL_CF_MAX) return cudaErrorInvalidValue;
  const size_t smem = lnl_tile_smem_bytes(q, K, pitch);
  cudaError_t e = cudaFuncSetAttribute(lnl_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  TileArgs a;
  a.q = q;
  a.b = b;
  a.ws = ws;
  a.K = K;
  a.H = H;
  a.pitch = pitch;
  for (int k = 0; k < RIFT_MAX_DET; ++k) a.dmax[k] = dmax[k];
  a.exp_tab = exp_tab;
  a.lnL_out = lnL_out;
  int64_t grid = n_sm;
  const int64_t max_grid = (b.n + 2 * TL_NS - 1) / (2 * TL_NS);
  if (grid > max_grid) grid = max_grid;
  lnl_tile_kernel<<<(unsigned)grid, TL_THREADS, smem, s>>>(a);
  if (n_launch) ++*n_launch;
  return cudaGetLastError();
}
