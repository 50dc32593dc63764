// Fused lnL kernel, "grouped" variant: steps a6-a7 of DESIGN.md section 1 on samples sorted by their relative shift
// tuple d_k = s_k - s_0 (sort.cu).
//   a6  x_n[t'] = sum_k sum_c B_n[k][c] Q_k[c][(t' + d_k) mod N_t],  t' = j0 + s_n0 + j   (Eq. (D2))
//   a7  lnL_tm  = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                   (App. D.2)
// A warp slides a window of 32 sorted samples, splits it into groups of up to BMAX samples with identical tuples
// (ballot / shuffle), and evaluates one group at a time: lanes run over time (t' = lane + 32 i), registers over the
// group members, so each shared-memory load of Q (conflict-free, contiguous across lanes) feeds up to BMAX FMAs.
// Q of the intrinsic point is staged by 1-D TMA in the planar, circularly extended layout (QStore) so that slot
// addresses are immediates.  The time-axis logsumexp is a transposed warp-shuffle reduction; final assembly in fp64.
// The code is kept small on purpose: one instruction stream per member-pair count, no per-size epilogues (an earlier
// version with eight fully unrolled variants spent most of its time in instruction-cache misses).
#include <cstdlib>

#include "rift_internal.h"
#include "tma_utils.cuh"

namespace {

// BMAX members per group (register columns), SLOTS time slots per lane and block, WARPS per CTA, MINB CTAs per SM.
template <typename Real_, int BMAX_, int SLOTS_, int WARPS_, int MINB_> struct GCfg {
  typedef Real_ Real;
  static constexpr int BMAX = BMAX_, SLOTS = SLOTS_, WARPS = WARPS_, MINB = MINB_;
};

__device__ __forceinline__ float lds_real(uint32_t addr, float) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ double lds_real(uint32_t addr, double) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}

// exp(c * (x - m)) with the per-member constants a = c*log2(e) (fp32) or c (fp64), am = a * m
__device__ __forceinline__ float exp_rel(float x, float a, float am) { return fast_exp2(fmaf(x, a, -am)); }
__device__ __forceinline__ double exp_rel(double x, double a, double am) { return exp(fma(x, a, -am)); }
__device__ __forceinline__ float exp_scale_of(double c, float) { return (float)(c * 1.4426950408889634); }
__device__ __forceinline__ double exp_scale_of(double c, double) { return c; }
// ln of the sum of exponentials (1 <= tot <= n_tau): fp32 logf is accurate to ~1e-6 absolute here, far inside the
// mixed-mode tolerance; fp64 mode uses the double routine
__device__ __forceinline__ double log_of(double v, float) { return (double)logf((float)v); }
__device__ __forceinline__ double log_of(double v, double) { return log(v); }

template <int SLOTS, typename Real>
__device__ __forceinline__ void load_q(Real (&q)[SLOTS], uint32_t addr) {
#pragma unroll
  for (int i = 0; i < SLOTS; ++i) q[i] = lds_real(addr + (uint32_t)(i * 32 * sizeof(Real)), Real());
}
// coefficients of the first N members of one row (N even), broadcast vector loads pinned in program order
template <int N> __device__ __forceinline__ void load_cf(float (&cf)[N], uint32_t addr) {
#pragma unroll
  for (int j = 0; j + 4 <= N; j += 4)
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(cf[j]), "=f"(cf[j + 1]), "=f"(cf[j + 2]), "=f"(cf[j + 3]) : "r"(addr + 4 * j));
  if (N % 4)
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(cf[N - 2]), "=f"(cf[N - 1]) : "r"(addr + 4 * (N - 2)));
}
template <int N> __device__ __forceinline__ void load_cf(double (&cf)[N], uint32_t addr) {
#pragma unroll
  for (int j = 0; j < N; j += 2)
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(cf[j]), "=d"(cf[j + 1]) : "r"(addr + 8 * j));
}
template <int SLOTS, int BMAX, int N, typename Real>
__device__ __forceinline__ void fma_rows(Real (&x)[SLOTS][BMAX], const Real (&q)[SLOTS], const Real (&cf)[N]) {
#pragma unroll
  for (int j = 0; j < N; ++j)
#pragma unroll
    for (int i = 0; i < SLOTS; ++i) x[i][j] = fma(q[i], cf[j], x[i][j]);
}

// The 2M rows (Re, Im of each mode) of one detector for the first 2*NPAIR members: branch-free, software pipelined
// (the Q values and coefficients of the next rows are loaded while the FMAs of the current ones issue).  The last trip
// prefetches two rows past the detector's block; those loads stay inside the shared allocation (padded) and are unused.
template <typename Real, int BMAX, int SLOTS, int NPAIR>
__device__ __forceinline__ void detector_rows(Real (&x)[SLOTS][BMAX], uint32_t addr, uint32_t row_bytes,
                                              uint32_t cf_addr, int M2) {
  constexpr int N = 2 * NPAIR;
  constexpr uint32_t CF_ROW = BMAX * sizeof(Real);
  Real qa[SLOTS], qb[SLOTS], cfa[N], cfb[N];
  load_q<SLOTS>(qa, addr);
  load_q<SLOTS>(qb, addr + row_bytes);
  load_cf<N>(cfa, cf_addr);
#pragma unroll 1
  for (int c = 0; c < M2; c += 2) {
    load_cf<N>(cfb, cf_addr + CF_ROW);
    fma_rows<SLOTS, BMAX, N>(x, qa, cfa);
    load_q<SLOTS>(qa, addr + 2 * row_bytes);
    load_cf<N>(cfa, cf_addr + 2 * CF_ROW);
    fma_rows<SLOTS, BMAX, N>(x, qb, cfb);
    load_q<SLOTS>(qb, addr + 3 * row_bytes);
    addr += 2 * row_bytes;
    cf_addr += 2 * CF_ROW;
  }
}

struct MaxOp {
  template <typename T> __device__ __forceinline__ T operator()(T a, T b) const { return fmax(a, b); }
};
struct SumOp {
  template <typename T> __device__ __forceinline__ T operator()(T a, T b) const { return a + b; }
};

// Reduce N per-lane values across the warp in N-1 + log2(32/N) shuffles (instead of 5N): each halving step sends the
// half a lane does not keep.  Returns, in every lane, the reduction of member (lane >> (5 - log2 N)) & (N-1).
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

struct GroupCtx {
  uint32_t q_addr;                 // shared address of the staged Q block
  int n_t, n_tp, K, M2;            // M2 = 2*M rows per detector
  unsigned span;                   // a time sample t' of a member is valid iff (unsigned)(t' - lo) < span
  int circular;
  double ln_ntau;
};

// per-warp shared scratch of one group
template <typename Real, int BMAX> struct alignas(16) GroupScalars {
  double c[BMAX], quad[BMAX];
  long long out[BMAX];
  Real a[BMAX];                    // exp scale: c*log2(e) (fp32) or c (fp64)
  int lo[BMAX];                    // first valid t' of the member's tau window (0 in circular mode)
  int d[RIFT_MAX_DET];             // the group's relative shifts reduced to [0, n_t); d[0] = 0
};

// One group of nb <= BMAX members (warp-uniform nb).  Unused member columns have zero coefficients.
template <typename Real, int BMAX, int SLOTS>
__device__ __forceinline__ void eval_group(const GroupCtx &g, int nb, const Real *wc,
                                           const GroupScalars<Real, BMAX> *gs, double *__restrict__ lnL_out, int lane) {
  constexpr int BLOCK = SLOTS * 32;
  constexpr int MSH = MemberShift<BMAX>::value;
  Real m_run[BMAX], s_run[BMAX];       // m_run: warp-uniform running max per member; s_run: per-lane sum relative to it
  Real m_own = -INFINITY;              // running max of the member this lane will finalise
#pragma unroll
  for (int j = 0; j < BMAX; ++j) {
    m_run[j] = -INFINITY;
    s_run[j] = 0;
  }
  const int npair = (nb + 1) >> 1;
  uint32_t row_bytes = (uint32_t)(g.n_tp * sizeof(Real));
  asm volatile("" : "+r"(row_bytes));               // keep it in a register (not re-read from the constant bank)
  const uint32_t wc_addr = smem_u32(wc);

  for (int tb = 0; tb < g.n_t; tb += BLOCK) {
    Real x[SLOTS][BMAX];
#pragma unroll
    for (int i = 0; i < SLOTS; ++i)
#pragma unroll
      for (int j = 0; j < BMAX; ++j) x[i][j] = 0;
#pragma unroll 1
    for (int k = 0; k < g.K; ++k) {
      int base = tb + gs->d[k];             // d[k] in [0, n_t), 0 <= tb < n_t
      base -= (base >= g.n_t) ? g.n_t : 0;
      const uint32_t addr = g.q_addr + (uint32_t)((k * g.M2) * g.n_tp + base + lane) * (uint32_t)sizeof(Real);
      const uint32_t cf_addr = wc_addr + (uint32_t)((k * g.M2) * BMAX * sizeof(Real));
      if (BMAX == 8) {
        switch (npair) {
          case 1: detector_rows<Real, BMAX, SLOTS, 1>(x, addr, row_bytes, cf_addr, g.M2); break;
          case 2: detector_rows<Real, BMAX, SLOTS, 2>(x, addr, row_bytes, cf_addr, g.M2); break;
          case 3: detector_rows<Real, BMAX, SLOTS, (BMAX >= 6 ? 3 : 1)>(x, addr, row_bytes, cf_addr, g.M2); break;
          default: detector_rows<Real, BMAX, SLOTS, (BMAX >= 8 ? 4 : 1)>(x, addr, row_bytes, cf_addr, g.M2); break;
        }
      } else {
        if (npair == 1) detector_rows<Real, BMAX, SLOTS, 1>(x, addr, row_bytes, cf_addr, g.M2);
        else detector_rows<Real, BMAX, SLOTS, (BMAX >= 4 ? 2 : 1)>(x, addr, row_bytes, cf_addr, g.M2);
      }
    }

    // ---- block epilogue: mask invalid time samples, per-member max
    const int tl = tb + lane;
    Real lmax[BMAX];
    if (g.circular && tb + BLOCK <= g.n_t) {            // every slot of the block is a valid time sample
#pragma unroll
      for (int j = 0; j < BMAX; ++j) {
        Real mx = x[0][j];
#pragma unroll
        for (int i = 1; i < SLOTS; ++i) mx = fmax(mx, x[i][j]);
        lmax[j] = mx;
      }
    } else {
#pragma unroll
      for (int j = 0; j < BMAX; ++j) {
        const int lo = gs->lo[j];
        Real mx = -INFINITY;
#pragma unroll
        for (int i = 0; i < SLOTS; ++i) {
          const bool ok = (unsigned)(tl + 32 * i - lo) < g.span;
          x[i][j] = ok ? x[i][j] : (Real)-INFINITY;
          mx = fmax(mx, x[i][j]);
        }
        lmax[j] = mx;
      }
    }
    const Real mb_own = transpose_reduce<BMAX>(lmax, lane, MaxOp());
    m_own = fmax(m_own, mb_own);
    Real mball[BMAX];
#pragma unroll
    for (int j = 0; j < BMAX; ++j) mball[j] = __shfl_sync(0xffffffffu, mb_own, j << MSH);
#pragma unroll
    for (int pr = 0; pr < BMAX / 2; ++pr) {
      if (pr < npair) {                     // two members per (uniform) branch, their chains interleave
        Real a[2], am[2], s0[2], s1[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int j = 2 * pr + u;
          a[u] = gs->a[j];
          const Real mnew = fmax(m_run[j], mball[j]);
          const Real mref = (mnew == (Real)-INFINITY) ? (Real)0 : mnew;
          am[u] = a[u] * mref;
          s0[u] = (m_run[j] == (Real)-INFINITY) ? (Real)0 : s_run[j] * exp_rel(m_run[j], a[u], am[u]);
          s1[u] = 0;
          m_run[j] = mnew;
        }
#pragma unroll
        for (int i = 0; i < SLOTS; ++i)
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const Real e = exp_rel(x[i][2 * pr + u], a[u], am[u]);
            if (i & 1) s1[u] += e; else s0[u] += e;
          }
#pragma unroll
        for (int u = 0; u < 2; ++u) s_run[2 * pr + u] = s0[u] + s1[u];
      }
    }
  }
  // ---- cross-lane sums in fp64 (reading A17), then one lane per member assembles lnL in fp64
  double sd[BMAX];
#pragma unroll
  for (int j = 0; j < BMAX; ++j) sd[j] = (double)s_run[j];
  const double tot = transpose_reduce<BMAX>(sd, lane, SumOp());
  const int jm = (lane >> MSH) & (BMAX - 1);
  if (jm < nb && lane == (jm << MSH))
    lnL_out[gs->out[jm]] = gs->c[jm] * (double)m_own + log_of(tot, Real()) - g.ln_ntau - gs->quad[jm];
}

template <typename Cfg>
__global__ void __launch_bounds__(Cfg::WARPS * 32, Cfg::MINB)
lnl_grouped_kernel(QStore q, Batch b, Workspace ws, int K, double *__restrict__ lnL_out) {
  typedef typename Cfg::Real Real;
  constexpr int BMAX = Cfg::BMAX;
  constexpr int SLOTS = Cfg::SLOTS;
  constexpr int G_WARPS = Cfg::WARPS;
  typedef GroupScalars<Real, BMAX> GS;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
  Real *Qs = reinterpret_cast<Real *>(smem_raw + 128);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int km2 = 2 * q.km;
  GS *gs = reinterpret_cast<GS *>(smem_raw + 128 + q.point_stride_bytes) + warp;
  Real *wc = reinterpret_cast<Real *>(smem_raw + 128 + q.point_stride_bytes + G_WARPS * sizeof(GS)) +
             (size_t)warp * km2 * BMAX;

  GroupCtx g;
  g.q_addr = smem_u32(Qs);
  g.n_t = q.n_t;
  g.n_tp = q.n_tp;
  g.K = K;
  g.M2 = km2 / K;
  g.circular = (q.n_tau == q.n_t);
  g.span = (unsigned)q.n_tau;
  g.ln_ntau = log((double)q.n_tau);
  const int j0 = (q.n_t - q.n_tau) / 2;

  const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x;
  const int64_t w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  uint32_t phase = 0;
  int staged_point = -1;

  for (int64_t w0 = w_begin; w0 < w_end;) {
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    if (point != staged_point) {
      __syncthreads();
      if (threadIdx.x == 0)
        stage_block(Qs, reinterpret_cast<const unsigned char *>(q.data) + (int64_t)point * q.point_stride_bytes,
                    (uint32_t)q.point_stride_bytes, bar);
      mbar_wait(bar, phase);
      phase ^= 1u;
      staged_point = point;
    }

    // each warp walks a contiguous part of the run with a sliding 32-sample window; a group cut by the window end
    // is deferred to the next window so that groups are split only at the part boundaries
    const int64_t part = (run_end - w0 + G_WARPS - 1) / G_WARPS;
    const int64_t r_begin = w0 + warp * part;
    const int64_t r_end = min(run_end, r_begin + part);
    for (int64_t ws0 = r_begin; ws0 < r_end;) {
      const int64_t p = ws0 + lane;
      const bool valid = p < r_end;
      // relative shifts packed 16 bits each: key1 holds d_1..d_4, key2 d_5..d_7 (exact for |d| < 32768)
      unsigned long long key1 = 0, key2 = 0;
      int s0 = 0;
      if (valid) {
        s0 = ws.shift[p * K];
        for (int k = 1; k < K; ++k) {
          const unsigned long long u = (unsigned long long)((ws.shift[p * K + k] - s0) & 0xffff);
          if (k <= 4) key1 |= u << (16 * (k - 1)); else key2 |= u << (16 * (k - 5));
        }
      }
      unsigned remaining = __ballot_sync(0xffffffffu, valid);
      const bool more = ws0 + 32 < r_end;
      int advance = 32;
      while (remaining) {
        const int leader = __ffs(remaining) - 1;
        const unsigned long long l1 = __shfl_sync(0xffffffffu, key1, leader);
        const unsigned long long l2 = __shfl_sync(0xffffffffu, key2, leader);
        const bool eq = ((remaining >> lane) & 1u) && key1 == l1 && key2 == l2;
        unsigned grp = __ballot_sync(0xffffffffu, eq);
        // a group that is exactly the contiguous tail of a full window continues in the next window: defer it
        if (more && leader > 0 && grp == (0xffffffffu << leader)) {
          advance = leader;
          break;
        }
        const int nb = min(__popc(grp), BMAX);
        // my member lane (lanes j < nb): the j-th set bit of grp
        int ml = 0;
        {
          unsigned t = grp;
          for (int j = 0; j < BMAX; ++j) {
            const int l = t ? __ffs(t) - 1 : 0;
            if (j == (lane % BMAX)) ml = l;
            if (j == nb - 1) remaining &= ~(grp ^ (t & (t - 1)));      // clear the first nb members
            t &= t - 1;
          }
        }
        __syncwarp();
        // stage the members' coefficient vectors transposed: wc[r * BMAX + j] = coef[member j][r]
        {
          const int j = lane % BMAX, rr = lane / BMAX;          // 32 / BMAX rows per pass
          const Real *src = reinterpret_cast<const Real *>(ws.coef) + (ws0 + ml) * ws.coef_stride;
#pragma unroll 4
          for (int r = rr; r < km2; r += 32 / BMAX) wc[r * BMAX + j] = (j < nb) ? src[r] : (Real)0;
        }
        if (lane < BMAX) {
          const int64_t pm = ws0 + ml;
          const bool on = lane < nb;
          const double c = on ? ws.scale_c[pm] : 0.0;
          gs->c[lane] = c;
          gs->a[lane] = exp_scale_of(c, Real());
          gs->quad[lane] = on ? ws.quad[pm] : 0.0;
          gs->lo[lane] = (on && !g.circular) ? j0 + ws.shift[pm * K] : 0;
          gs->out[lane] = on ? (long long)(b.g0 + (ws.orig ? ws.orig[pm] : pm)) : 0;
        }
        if (lane < K) {                                          // the group's shifts, reduced to [0, n_t)
          int dk = 0;
          if (lane >= 1) {
            const unsigned long long kk = lane <= 4 ? l1 >> (16 * (lane - 1)) : l2 >> (16 * (lane - 5));
            dk = (int)(short)(kk & 0xffff) % q.n_t;
            if (dk < 0) dk += q.n_t;
          }
          gs->d[lane] = dk;
        }
        __syncwarp();
        eval_group<Real, BMAX, SLOTS>(g, nb, wc, gs, lnL_out, lane);
      }
      ws0 += advance;
    }
    w0 = run_end;
  }
}

template <typename Cfg>
size_t smem_bytes_t(const QStore &q) {
  typedef typename Cfg::Real Real;
  // + two rows of padding: the pipelined loads of the last trip run two rows past the block (unused values)
  return 128 + (size_t)q.point_stride_bytes + Cfg::WARPS * sizeof(GroupScalars<Real, Cfg::BMAX>) +
         (size_t)Cfg::WARPS * 2 * q.km * Cfg::BMAX * sizeof(Real) + 2 * (size_t)q.n_tp * sizeof(Real) + 256;
}

template <typename Cfg>
cudaError_t launch_t(const QStore &q, const Batch &b, const Workspace &ws, int K, double *lnL_out, int n_sm,
                     cudaStream_t s) {
  auto kern = lnl_grouped_kernel<Cfg>;
  const size_t smem = smem_bytes_t<Cfg>(q);
  const int threads = Cfg::WARPS * 32;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)n_sm * occ;
  const int64_t max_grid = (b.n + threads - 1) / threads;
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, threads, smem, s>>>(q, b, ws, K, lnL_out);
  return cudaGetLastError();
}

typedef GCfg<float, 8, 7, 8, 2> CfgF_A;       // 7 slots, 2 CTAs/SM
typedef GCfg<float, 8, 13, 11, 1> CfgF_B;     // 13 slots, 11 warps, 1 CTA/SM
typedef GCfg<float, 8, 13, 8, 1> CfgF_C;      // 13 slots, 8 warps
typedef GCfg<double, 4, 7, 8, 2> CfgD_A;

int grouped_cfg_id() {
  static int id = -1;
  if (id < 0) {
    const char *e = getenv("RIFT_GROUPED_CFG");
    id = e ? atoi(e) : 0;
  }
  return id;
}

}  // namespace

size_t lnl_grouped_smem_bytes(const QStore &q, bool fp32) {
  if (!fp32) return smem_bytes_t<CfgD_A>(q);
  switch (grouped_cfg_id()) {
    case 1: return smem_bytes_t<CfgF_B>(q);
    case 2: return smem_bytes_t<CfgF_C>(q);
    default: return smem_bytes_t<CfgF_A>(q);
  }
}

cudaError_t launch_lnl_grouped(const QStore &q, bool fp32, const Batch &b, const Workspace &ws, int n_det,
                               double *lnL_out, int n_sm, cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  if (n_launch) ++*n_launch;
  if (!fp32) return launch_t<CfgD_A>(q, b, ws, n_det, lnL_out, n_sm, s);
  switch (grouped_cfg_id()) {
    case 1: return launch_t<CfgF_B>(q, b, ws, n_det, lnL_out, n_sm, s);
    case 2: return launch_t<CfgF_C>(q, b, ws, n_det, lnL_out, n_sm, s);
    default: return launch_t<CfgF_A>(q, b, ws, n_det, lnL_out, n_sm, s);
  }
}
