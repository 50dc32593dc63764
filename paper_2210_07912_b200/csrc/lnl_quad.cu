// Fused lnL kernel, "quad" variant: steps a6-a7 of DESIGN.md section 1 on samples sorted by their relative shift tuple
// d_k = s_k - s_0 (sort.cu), NQ consecutive sorted samples per warp.
//   a6  x_n[t'] = sum_k sum_lm ( B.re Q.re + B.im Q.im )[(t' + d_nk) mod N_t],  t' = j0 + s_n0 + j    (Eq. (D2))
//   a7  lnL_tm  = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                (App. D.2)
// Same structure as lnl_direct_ext (one warp, lanes over time, 13 slots, TMA-staged extended interleaved window,
// next row's loads under the current row's FMAs), but a warp carries NQ samples in registers.  Per detector the NQ
// relative shifts are compared (warp-uniform): if they are all equal, ONE set of shared-memory loads feeds NQ samples
// (13 LDS.64 : 26 NQ FMAs); if they are equal in pairs, one set per pair; otherwise one set per sample.  Detector 0 is
// always shared (d_0 = 0) and, in sorted order, so is nearly always detector 1.  This divides the shared-memory traffic
// that bounds lnl_direct_ext by ~2.5 on C1 while keeping the control flow regular (no variable-size groups).
#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

#include <cstdlib>

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
template <> struct C2<float> { typedef float2 type; static constexpr int NQ = 4; };
template <> struct C2<double> { typedef double2 type; static constexpr int NQ = 2; };

template <typename Real, int SLOTS, typename CT>
__device__ __forceinline__ void load_row(CT (&v)[SLOTS], uint32_t addr) {
#pragma unroll
  for (int i = 0; i < SLOTS; ++i) v[i] = lds_c(addr + (uint32_t)(i * 32 * sizeof(CT)), Real());
}

// Mode rows of one detector for members [C0, C0+NB) of the quad, all reading the window at the same base address.
// caddr: shared address of member C0's coefficient of this detector's first mode; members are cstride bytes apart.
// Software pipeline, two mode rows per trip: the window values of the next row and the coefficients of the next trip
// are loaded while the FMAs of the current row issue.
template <typename Real, int SLOTS, int NQ, int C0, int NB>
__device__ __forceinline__ void rows_shared(Real (&x)[SLOTS][NQ], uint32_t addr, uint32_t row_bytes, uint32_t caddr,
                                            uint32_t cstride, int M) {
  typedef typename C2<Real>::type CT;
  CT va[SLOTS], vb[SLOTS], ca[NB], cb[NB];
  load_row<Real, SLOTS>(va, addr);
#pragma unroll
  for (int j = 0; j < NB; ++j) ca[j] = lds_c(caddr + (uint32_t)(j * cstride), Real());
#pragma unroll 1
  for (int m = 0; m < M; m += 2) {
    const bool has_b = m + 1 < M, has_next = m + 2 < M;
    if (has_b) {
      load_row<Real, SLOTS>(vb, addr + row_bytes);
#pragma unroll
      for (int j = 0; j < NB; ++j) cb[j] = lds_c(caddr + (uint32_t)(j * cstride + sizeof(CT)), Real());
    }
#pragma unroll
    for (int j = 0; j < NB; ++j)
#pragma unroll
      for (int i = 0; i < SLOTS; ++i) {
        x[i][C0 + j] = fma(ca[j].x, va[i].x, x[i][C0 + j]);
        x[i][C0 + j] = fma(ca[j].y, va[i].y, x[i][C0 + j]);
      }
    if (has_next) {
      load_row<Real, SLOTS>(va, addr + 2 * row_bytes);
#pragma unroll
      for (int j = 0; j < NB; ++j) ca[j] = lds_c(caddr + (uint32_t)(j * cstride + 2 * sizeof(CT)), Real());
    }
    if (has_b) {
#pragma unroll
      for (int j = 0; j < NB; ++j)
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) {
          x[i][C0 + j] = fma(cb[j].x, vb[i].x, x[i][C0 + j]);
          x[i][C0 + j] = fma(cb[j].y, vb[i].y, x[i][C0 + j]);
        }
    }
    addr += 2 * row_bytes;
    caddr += 2 * (uint32_t)sizeof(CT);
  }
}

struct MaxOp {
  template <typename T> __device__ __forceinline__ T operator()(T a, T b) const { return fmax(a, b); }
};
struct SumOp {
  template <typename T> __device__ __forceinline__ T operator()(T a, T b) const { return a + b; }
};
// Reduce N per-lane values across the warp: every lane ends with the reduction of member (lane >> (5 - log2 N)) & (N-1).
template <int N, typename T, typename Op>
__device__ __forceinline__ T transpose_reduce(T (&v)[N], int lane, Op op) {
  int bit = 16;
#pragma unroll
  for (int n = N; n > 1; n >>= 1) {
    const bool hi = (lane & bit) != 0;
#pragma unroll
    for (int i = 0; i < n / 2; ++i) {
      const T send = hi ? v[i] : v[i + n / 2];
      const T keep = hi ? v[i + n / 2] : v[i];
      v[i] = op(keep, __shfl_xor_sync(0xffffffffu, send, bit));
    }
    bit >>= 1;
  }
#pragma unroll
  for (; bit > 0; bit >>= 1) v[0] = op(v[0], __shfl_xor_sync(0xffffffffu, v[0], bit));
  return v[0];
}
template <int N> struct MemberShift { static constexpr int value = MemberShift<N / 2>::value - 1; };
template <> struct MemberShift<1> { static constexpr int value = 5; };

__device__ __forceinline__ float exp_rel(float x, float a, float am) { return fast_exp2(fmaf(x, a, -am)); }
__device__ __forceinline__ double exp_rel(double x, double a, double am) { return exp(fma(x, a, -am)); }

template <typename Real, int SLOTS, int Q_WARPS, int MINB>
__global__ void __launch_bounds__(Q_WARPS * 32, MINB)
lnl_quad_kernel(QStore q, Batch b, Workspace ws, int K, double *__restrict__ lnL_out) {
  typedef typename C2<Real>::type CT;
  constexpr int BLOCK = SLOTS * 32;
  constexpr int NQ = C2<Real>::NQ;
  constexpr int MSH = MemberShift<NQ>::value;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
  CT *Qs = reinterpret_cast<CT *>(smem_raw + 128);
  CT *coef_s = reinterpret_cast<CT *>(smem_raw + 128 + q.point_stride_bytes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int km = q.km, M = km / K;
  CT *wcoef = coef_s + warp * (2 * NQ * km);             // [2][NQ][km], double-buffered
  const uint32_t wcoef_addr = smem_u32(wcoef);
  const uint32_t cstride = (uint32_t)(km * sizeof(CT));
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
  const bool circular = (q.n_tau == q.n_t);
  const unsigned span = (unsigned)q.n_tau;
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

    // Per-warp loop over quads (NQ consecutive workspace slots).  The NEXT quad's metadata is prefetched into registers
    // and its coefficient vectors into the other half of the per-warp shared buffer (cp.async) while the current quad is
    // evaluated, so no global-memory latency sits on the critical path.
    struct Meta {
      int dval;                 // lane j*K + k: relative shift of member j, detector k, reduced to [0, n_t)
      double c, quad;           // lanes < nv
      int lo;
      long long out;
    };
    auto fetch_meta = [&](int64_t w, Meta &mt) {
      const int nv = (int)min((int64_t)NQ, run_end - w);
      mt.dval = 0;
      if (lane < NQ * K) {
        const int j = lane / K, k = lane - j * K;
        const int64_t p = w + (j < nv ? j : 0);     // missing members copy member 0 (zero coefficients, no output)
        int d = ws.shift[p * K + k] - ws.shift[p * K];
        d %= q.n_t;
        mt.dval = d < 0 ? d + q.n_t : d;
      }
      mt.c = 0.0;
      mt.quad = 0.0;
      mt.lo = 0;
      mt.out = -1;
      if (lane < nv) {
        const int64_t p = w + lane;
        mt.c = ws.scale_c[p];
        mt.quad = ws.quad[p];
        mt.lo = circular ? 0 : j0 + ws.shift[p * K];
        mt.out = (long long)(b.g0 + (ws.orig ? ws.orig[p] : p));
      }
    };
    auto fetch_coef = [&](int64_t w, int buf) {
      const int nv = (int)min((int64_t)NQ, run_end - w);
      for (int i = lane; i < NQ * km; i += 32) {
        const int j = i / km, r = i - j * km;
        const int jj = j < nv ? j : 0;
        const CT *src = reinterpret_cast<const CT *>(reinterpret_cast<const Real *>(ws.coef) + (w + jj) * ws.coef_stride) + r;
        const uint32_t dst = wcoef_addr + (uint32_t)((buf * NQ * km + i) * sizeof(CT));
        const int src_bytes = j < nv ? (int)sizeof(CT) : 0;          // 0 => zero fill
        if (sizeof(CT) == 8)
          asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
        else
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    };

    int buf = 0;
    int64_t w = w0 + NQ * warp;
    Meta nxt;
    if (w < run_end) {
      fetch_meta(w, nxt);
      fetch_coef(w, buf);
    }
    for (; w < run_end; w += NQ * Q_WARPS, buf ^= 1) {
      const int dval = nxt.dval;
      const double my_c = nxt.c, my_quad = nxt.quad;
      const int my_lo = nxt.lo;
      const long long my_out = nxt.out;
      const Real my_a = (sizeof(Real) == 4) ? (Real)(my_c * 1.4426950408889634) : (Real)my_c;
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const int64_t wn = w + NQ * Q_WARPS;
      if (wn < run_end) {
        fetch_meta(wn, nxt);
        fetch_coef(wn, buf ^ 1);
      }
      const uint32_t wc_addr = wcoef_addr + (uint32_t)(buf * NQ * km * sizeof(CT));

      Real m_run[NQ], s_run[NQ];
      Real m_own = -INFINITY;
#pragma unroll
      for (int j = 0; j < NQ; ++j) {
        m_run[j] = -INFINITY;
        s_run[j] = 0;
      }
      for (int tb = 0; tb < q.n_t; tb += BLOCK) {
        Real x[SLOTS][NQ];
#pragma unroll
        for (int i = 0; i < SLOTS; ++i)
#pragma unroll
          for (int j = 0; j < NQ; ++j) x[i][j] = 0;
#pragma unroll 1
        for (int k = 0; k < K; ++k) {
          int dj[NQ];
          uint32_t addr[NQ];
#pragma unroll
          for (int j = 0; j < NQ; ++j) {
            dj[j] = __shfl_sync(0xffffffffu, dval, j * K + k);
            int base = tb + dj[j];
            base -= (base >= q.n_t) ? q.n_t : 0;
            addr[j] = q_addr + (uint32_t)((k * M) * q.n_tp + base + lane) * (uint32_t)sizeof(CT);
          }
          const uint32_t caddr = wc_addr + (uint32_t)(k * M * sizeof(CT));
          if (NQ == 4) {
            if (dj[0] == dj[1] && dj[1] == dj[NQ - 2] && dj[NQ - 2] == dj[NQ - 1]) {
              rows_shared<Real, SLOTS, NQ, 0, NQ>(x, addr[0], row_bytes, caddr, cstride, M);
            } else if (dj[0] == dj[1] && dj[NQ - 2] == dj[NQ - 1]) {
              rows_shared<Real, SLOTS, NQ, 0, 2>(x, addr[0], row_bytes, caddr, cstride, M);
              rows_shared<Real, SLOTS, NQ, NQ - 2, 2>(x, addr[NQ - 2], row_bytes, caddr + (NQ - 2) * cstride, cstride, M);
            } else {
              rows_shared<Real, SLOTS, NQ, 0, 1>(x, addr[0], row_bytes, caddr, cstride, M);
              rows_shared<Real, SLOTS, NQ, 1, 1>(x, addr[1], row_bytes, caddr + cstride, cstride, M);
              rows_shared<Real, SLOTS, NQ, NQ - 2, 1>(x, addr[NQ - 2], row_bytes, caddr + (NQ - 2) * cstride, cstride, M);
              rows_shared<Real, SLOTS, NQ, NQ - 1, 1>(x, addr[NQ - 1], row_bytes, caddr + (NQ - 1) * cstride, cstride, M);
            }
          } else {
            if (dj[0] == dj[NQ - 1]) {
              rows_shared<Real, SLOTS, NQ, 0, NQ>(x, addr[0], row_bytes, caddr, cstride, M);
            } else {
              rows_shared<Real, SLOTS, NQ, 0, 1>(x, addr[0], row_bytes, caddr, cstride, M);
              rows_shared<Real, SLOTS, NQ, NQ - 1, 1>(x, addr[NQ - 1], row_bytes, caddr + (NQ - 1) * cstride, cstride, M);
            }
          }
        }
        // ---- block epilogue: mask, per-member max (transposed shuffle reduction), exponentials
        const int tl = tb + lane;
        Real lmax[NQ];
#pragma unroll
        for (int j = 0; j < NQ; ++j) {
          const int lo = __shfl_sync(0xffffffffu, my_lo, j);
          Real mx = -INFINITY;
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) {
            const int t = tl + 32 * i;
            const bool ok = (t < q.n_t) && ((unsigned)(t - lo) < span);
            x[i][j] = ok ? x[i][j] : (Real)-INFINITY;
            mx = fmax(mx, x[i][j]);
          }
          lmax[j] = mx;
        }
        const Real mb_own = transpose_reduce<NQ>(lmax, lane, MaxOp());
        m_own = fmax(m_own, mb_own);
#pragma unroll
        for (int j = 0; j < NQ; ++j) {
          const Real mb = __shfl_sync(0xffffffffu, mb_own, j << MSH);
          const Real a = __shfl_sync(0xffffffffu, my_a, j);
          const Real mnew = fmax(m_run[j], mb);
          const Real mref = (mnew == (Real)-INFINITY) ? (Real)0 : mnew;
          const Real am = a * mref;
          Real s0 = (m_run[j] == (Real)-INFINITY) ? (Real)0 : s_run[j] * exp_rel(m_run[j], a, am);
          Real s1 = 0;
#pragma unroll
          for (int i = 0; i < SLOTS; ++i) {
            const Real e = exp_rel(x[i][j], a, am);
            if (i & 1) s1 += e; else s0 += e;
          }
          m_run[j] = mnew;
          s_run[j] = s0 + s1;
        }
      }
      // ---- sums across lanes in fp64 (reading A17); lane (jm << MSH) assembles member jm in fp64
      double sd[NQ];
#pragma unroll
      for (int j = 0; j < NQ; ++j) sd[j] = (double)s_run[j];
      const double tot = transpose_reduce<NQ>(sd, lane, SumOp());
      const int jm = (lane >> MSH) & (NQ - 1);
      const double cm = __shfl_sync(0xffffffffu, my_c, jm);
      const double qm = __shfl_sync(0xffffffffu, my_quad, jm);
      const long long om = __shfl_sync(0xffffffffu, my_out, jm);
      if (lane == (jm << MSH) && om >= 0) lnL_out[om] = cm * (double)m_own + log(tot) - ln_ntau - qm;
    }
    w0 = run_end;
  }
}

template <typename Real, int SLOTS, int Q_WARPS, int MINB>
cudaError_t launch_t(const QStore &q, const Batch &b, const Workspace &ws, int K, double *lnL_out, int n_sm,
                     cudaStream_t s) {
  auto kern = lnl_quad_kernel<Real, SLOTS, Q_WARPS, MINB>;
  constexpr int threads = Q_WARPS * 32;
  const size_t smem = 128 + (size_t)q.point_stride_bytes + (size_t)Q_WARPS * 2 * C2<Real>::NQ * q.km * sizeof(typename C2<Real>::type);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)n_sm * occ;
  const int64_t max_grid = (b.n + 4 * Q_WARPS - 1) / (4 * Q_WARPS);
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, threads, smem, s>>>(q, b, ws, K, lnL_out);
  return cudaGetLastError();
}

int quad_cfg_id() {
  static int id = -1;
  if (id < 0) {
    const char *e = getenv("RIFT_QUAD_CFG");
    id = e ? atoi(e) : 0;
  }
  return id;
}

}  // namespace

size_t lnl_quad_smem_bytes(const QStore &q, bool fp32) {
  const size_t csz = fp32 ? 8 : 16;
  const int nq = fp32 ? C2<float>::NQ : C2<double>::NQ;
  return 128 + (size_t)q.point_stride_bytes + (size_t)12 * 2 * nq * q.km * csz;     // sized for the widest CTA (12 warps)
}

cudaError_t launch_lnl_quad(const QStore &q, bool fp32, const Batch &b, const Workspace &ws, int n_det,
                            double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  if (n_launch) ++*n_launch;
  if (!fp32) return launch_t<double, 7, 8, 1>(q, b, ws, n_det, lnL_out, n_sm, s);
  switch (quad_cfg_id()) {
    case 1: return launch_t<float, 13, 8, 1>(q, b, ws, n_det, lnL_out, n_sm, s);
    case 2: return launch_t<float, 13, 10, 1>(q, b, ws, n_det, lnL_out, n_sm, s);
    default: return launch_t<float, 7, 8, 2>(q, b, ws, n_det, lnL_out, n_sm, s);
  }
}
