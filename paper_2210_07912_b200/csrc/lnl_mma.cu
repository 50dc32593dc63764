// Fused lnL kernel of the fp64 mode on the FP64 tensor cores: steps a6-a7 of DESIGN.md section 1.
//   a6  x_j = sum_k sum_lm ( B.re Q.re + B.im Q.im ),  B = F_k Y_lm,  Q = Q_{k,lm}[(j0 + s_k + j) mod N_t]   (Eq. (D2))
//   a7  lnL_tm = c x_max + ln sum_j exp(c (x_j - x_max)) - ln N_tau - q                                   (App. D.2)
//
// "Contract in unshifted detector time, then shift": per detector k the window term is the real GEMM
//     P_k[t, n] = sum_kappa A_k[t, kappa] B_k[kappa, n],   A_k[t, 2m + {0,1}] = {Re, Im} Q_{k,m}[t],  B_k[2m + {0,1}, n] = {Re, Im}(F_k Y_m)_n
// over ALL stored rows t (M = time, N = the samples of a batch, K = 2 x modes), issued as mma.sync.m8n8k4.f64 (DMMA, 256
// FMA per instruction and warp: one Q value read from shared memory feeds 8 samples, one coefficient 8 rows -- the direct
// kernel reads a 16-byte Q value per 2 DFMA and cannot pass 25 % of the pipe).  The per-sample shift is applied when the
// tiles leave the registers: the window X[j][n] of the batch lives in shared memory (rows of NBG samples, pitch NBG * 8 + 8
// bytes) and the thread holding P_k[t][n] adds it to row j = (t - off_{n,k}) mod N_t -- a plain store for the first detector,
// a read-modify-write for the others, one group barrier per detector in between (an element is touched by one thread per
// detector).  The row of tile i of a thread is row_0 + 8 GW i, so the wrap of a circular window is one threshold per sample
// and detector (tiles below it use one base address, the others a second one, N_t rows apart) and the addresses are a base
// register plus immediates; rows >= N_t of the operand are zero and add nothing wherever they land.  The tensor phase of
// detector k + 1 is issued before the barrier that closes detector k.  The time marginal then reads the window back, one
// sample and NE entries per thread: a float maximum (any reference >= max - eps serves the log-sum-exp) and the sum of
// 2^(c log2e (x - m)) with a polynomial exponential, both reduced across warps in shared memory.
//
// Q operand: the handle keeps [P][K][M2][pitch] bytes, M2 = 2 ceil(M/2) mode rows per detector (zero rows pad an odd mode
// count), every row n_r = 8 ceil(N_t/8) complex128 (zero beyond N_t) followed by 64 pad bytes, so that the two mode rows of
// one k-step sit 64 bytes apart modulo 128 and an A fragment load (8 rows x 2 modes x 16 B) is conflict-free.  Small
// configurations keep the whole block of the intrinsic point resident in shared memory (one bulk copy per point); larger
// ones stream (detector, k-step) chunks through a ring filled by a producer warp with cp.async.bulk on mbarriers.
#include <type_traits>

#include "rift_internal.h"
#include "tma_utils.cuh"
#include "exp2_poly.cuh"

namespace {

constexpr int MM_MAX_SLOTS = 8;

// Two shapes of the CTA.  Resident Q block: two or three independent groups of 8 warps (three when three windows fit beside the Q
// block: 24 warps of 80 registers; measured +4 % on C1 / C3 over two groups of 128 registers), each with its own batch of 8 samples (one
// 8-column tile), exchange buffer and named barrier, so that the tensor phase of one group runs under the exchange and
// exponential phases of the other.  Streamed Q: a bulk-copy producer warp feeds a ring of (detector, k-step) chunks to either two
// groups of 7 warps with batches of 8 samples each (windows up to 448 rows: both groups take every chunk, each for its own batch,
// and drift apart by up to the ring's depth, so that one group's scatter and exponentials run under the other's tensor phase;
// C2: 45.3 -> 43.7 ms per 8 points) or one group of 15 warps with batches of 16 samples (two tiles per A fragment).
template <bool STREAM, int NG = 2>
struct MmaShape {
  static constexpr int NT = (STREAM && NG == 1) ? 2 : 1;   // 8-sample tiles per batch of a group
  static constexpr int NBG = 8 * NT;               // samples per batch of a group
  static constexpr int GROUPS = NG;                // resident: 2 or 3 groups (3: 24 warps of 80 registers, when three windows fit);
                                                   // streamed: 1 group of 15 warps x 16 samples, or 2 groups of 7 warps x 8 samples that
                                                   // consume the same ring chunk and drift apart by up to the ring's depth
  static constexpr int WARPS = STREAM ? 16 : 8 * NG;
  static constexpr int GW = STREAM ? (NG == 1 ? 15 : 7) : 8;   // warps per group
  static constexpr int RBW = (STREAM && NG == 1) ? 4 : 8;   // row blocks (of 8 rows) per warp: wg + GW i
  static constexpr int GTHR = GW * 32;
  static constexpr int XP = 64 * NT;               // bytes per window row (8-byte slots, swizzled: x_slot)
  static constexpr int RS = 8 * GW;                // rows between two tiles of a thread
  static constexpr int RPW = NT == 2 ? 2 : 4;      // window entries a warp reads per element index e
  static constexpr int JS = RPW * GW;              // ... a group
};

__device__ __forceinline__ void mm_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ double ld_shared_f64(uint32_t a) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void st_shared_f64(uint32_t a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void mm_bar(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

// 8-byte slot of sample n inside window row r.  Shared memory serves a 64-bit access half a warp at a time: for a scatter
// instruction that is 4 consecutive rows (any start row, one per sample) of the 4 samples 2 lc + h.  The slot keeps the pair
// index lc and swaps the rest with the row, so that those 16 accesses land on 16 different bank pairs whatever the shifts
// are; a reader's half-warp takes whole rows.  The slot depends on r mod 4 only: rows 8 apart share it, so tile i of a
// thread is base + immediate.
template <int NT>
__device__ __forceinline__ uint32_t x_slot(int r, int n) {
  if (NT == 1) return (uint32_t)(n ^ ((r >> 1) & 1));            // bank pair 8 (r & 1) + 2 lc + (h ^ bit 1 of r)
  const int lc = (n >> 1) & 3, rest = ((n >> 3) << 1) | (n & 1);  // n = 8 nt + 2 lc + h
  return (uint32_t)(4 * lc + (rest ^ (r & 3)));                   // bank pair = slot
}
template <int NT>
__device__ __forceinline__ uint32_t x_addr(uint32_t xb, int r, int n) {
  return xb + (uint32_t)(r * (64 * NT)) + 8u * x_slot<NT>(r, n);
}

struct MmaSmem {                                   // byte offsets inside dynamic shared memory
  uint32_t bars, grp, grp_stride, coef_bytes, meta, meta_bytes, wmax, psum, xb, q, total;   // coef .. xb: inside a group block
};

__host__ __device__ inline MmaSmem mma_smem(const MmaPlan &p) {
  MmaSmem L;
  const uint32_t nbg = (p.stream && p.groups == 1) ? 16u : 8u, groups = (uint32_t)p.groups, rb = nbg * 8u;
  L.bars = 0;                                                          // full[8], empty[8], resident
  L.grp = 256;
  L.coef_bytes = (uint32_t)p.K * p.KS * nbg * 4 * 8;                   // cs[K][KS][NBG][4] doubles, two buffers at offset 0
  L.meta = 2 * L.coef_bytes;
  L.meta_bytes = 2 * nbg * 8 + (uint32_t)p.K * nbg * 4;                // c[NBG], q[NBG] doubles, off[K][NBG] int32, two buffers
  L.wmax = (L.meta + 2 * L.meta_bytes + 15u) & ~15u;                   // wmax[2][NBG][16] float
  L.psum = L.wmax + 2 * nbg * 16 * 4;                                  // psum[2][NBG][16] double
  L.xb = (L.psum + 2 * nbg * 16 * 8 + 127u) & ~127u;                   // window rows
  L.grp_stride = (L.xb + (uint32_t)p.xb_rows * rb + 127u) & ~127u;
  L.q = L.grp + groups * L.grp_stride;
  const uint32_t qbytes = p.stream ? (uint32_t)p.slots * 2u * (uint32_t)p.pitch_q
                                   : (uint32_t)p.K * 2u * p.KS * (uint32_t)p.pitch_q;
  L.total = L.q + qbytes;
  return L;
}

__device__ __forceinline__ float mf_of(const float *wmax, int n, bool wide) {          // maximum of a sample's per-warp slots
  float m = -INFINITY;
  for (int w = 0; w < (wide ? 16 : 8); ++w) m = fmaxf(m, wmax[n * 16 + w]);
  return m;
}

struct MmaArgs {
  MmaPlan p;
  MmaSmem L;                       // computed on the host: the kernel reads the offsets from the constant bank
  const unsigned char *q;          // [P][K][2 KS][pitch_q]
  Batch b;
  Workspace ws;
  double *lnL_out;
  double ln_ntau;
};

template <bool STREAM, int NE, int PFN, int NG>
__global__ void __launch_bounds__(MmaShape<STREAM, NG>::WARPS * 32, 1) lnl_mma_kernel(const MmaArgs A) {
  typedef MmaShape<STREAM, NG> S;
  constexpr int NT = S::NT, NBG = S::NBG, GW = S::GW, RBW = S::RBW, GTHR = S::GTHR, XP = S::XP, RS = S::RS, JS = S::JS;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const MmaPlan &P = A.p;
  const Batch &b = A.b;
  const Workspace &ws = A.ws;
  const MmaSmem &L = A.L;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + L.bars);
  uint64_t *empty = full + MM_MAX_SLOTS;
  uint64_t *resbar = empty + MM_MAX_SLOTS;
  unsigned char *qs = smem_raw + L.q;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K = P.K, KS = P.KS, n_t = P.n_t, n_r = P.n_r, n_x = P.n_x, H = P.H;
  const int m2 = 2 * P.M, km2 = m2 * K;                               // doubles of coefficients per detector / sample
  const uint32_t slot_bytes = 2u * (uint32_t)P.pitch_q;               // one k-step: two consecutive mode rows

  if (threadIdx.x == 0) {
    for (int i = 0; i < MM_MAX_SLOTS; ++i) {
      mbar_init(full + i, 1);
      mbar_init(empty + i, S::GROUPS * GW);
    }
    mbar_init(resbar, 1);
  }
  for (uint32_t i = threadIdx.x; i < S::GROUPS * L.grp_stride / 8; i += blockDim.x)   // coefficient pads 0, wmax / psum below
    reinterpret_cast<double *>(smem_raw + L.grp)[i] = 0.0;
  __syncthreads();


  // ---------------------------------------------------------------------------------------------- producer warp (ring)
  if (STREAM && warp >= S::GROUPS * GW) {                        // the producer warp; a spare warp (two groups of 7) leaves
    if (warp > S::GROUPS * GW) return;
    if (lane == 0) {
      const int64_t w_begin = (b.n * blockIdx.x) / gridDim.x, w_end = (b.n * (blockIdx.x + 1)) / gridDim.x;
      uint32_t slot = 0, ph = 0;                                 // ring position: slot and the parity of its use count
      for (int64_t w0 = w_begin; w0 < w_end;) {
        const int64_t seg = (b.g0 + w0) / b.n_per_seg;
        const int64_t run_end = min(w_end, (seg + 1) * b.n_per_seg - b.g0);
        const unsigned char *qp = A.q + (int64_t)b.ids[seg] * P.point_stride;
        for (int64_t s0 = w0; s0 < run_end; s0 += S::GROUPS * NBG)   // one pass over the chunks per batch of every group
          for (int k = 0; k < K; ++k)
            for (int s = 0; s < KS; ++s) {
              mbar_wait(empty + slot, ph ^ 1u);
              mbar_expect_tx(full + slot, slot_bytes);
              bulk_g2s(qs + slot * slot_bytes, qp + (size_t)(k * 2 * KS + 2 * s) * P.pitch_q, slot_bytes, full + slot);
              if (++slot == (uint32_t)P.slots) slot = 0, ph ^= 1u;
            }
        w0 = run_end;
      }
    }
    return;
  }

  // ---------------------------------------------------------------------------------------------- consumer groups
  const int g = warp / GW, wg = warp - g * GW, gtid = threadIdx.x - g * GTHR;
  const int bar_id = 1 + g;
  unsigned char *grp = smem_raw + L.grp + g * L.grp_stride;
  const uint32_t grp_u32 = smem_u32(grp), xb_u32 = grp_u32 + L.xb;
  for (int i = gtid; i < 2 * NBG * 16; i += GTHR) reinterpret_cast<float *>(grp + L.wmax)[i] = -INFINITY;   // absent warps
  // MMA role: fragment coordinates; row blocks wg + GW i are GW * 128 bytes apart: one base register plus immediates
  const int lr = lane >> 2, lc = lane & 3;
  const uint32_t a_base = (uint32_t)(lc >> 1) * (uint32_t)P.pitch_q + (uint32_t)(lc & 1) * 8u + (uint32_t)(8 * wg + lr) * 16u;
  const int nrb = 8 * wg < n_r ? (n_r - 8 * wg + 8 * GW - 1) / (8 * GW) : 0;   // valid row blocks of this warp (<= RBW)
  // scatter role: the thread holds P_k[t0 + RS i][8 nt + 2 lc + {0, 1}]; window row of stored row t and offset off:
  // t - off (+- n_t on a circular window), + H on a guard-band window (off >= 0 there, nothing wraps: wrap_rows 0)
  const int t0 = 8 * wg + lr;
  const bool last_ok = t0 + RS * (nrb - 1) < n_t;                // a zero row past n_t would wrap onto another thread's element
  const int wrap_rows = P.circular ? n_t : 0, row_bias = P.circular ? 0 : H;
  // window-reader role: sample n, window entries j = jb + JS e, e < nv
  const int n_mine = lane & (NBG - 1);                             // half a warp reads whole rows
  const int jj = lane / NBG, jb = S::RPW * wg + jj;
  const uint32_t rd_base = x_addr<NT>(xb_u32, jb + row_bias, n_mine);   // JS % 8 == 0: entry e is rd_base + e JS XP
  const int nv = min(NE, max(0, (n_x - jb + JS - 1) / JS));

  // coefficient items of this thread: element id = gtid + GTHR i of the [NBG][2 K M] block of a batch goes to the other
  // shared-memory buffer with an 8-byte cp.async (zero-filled for the slots past the end of a run).  PFN > 0: the (source,
  // destination) offsets of the <= PFN items wait in registers; PFN == 0 (many items): recomputed per batch
  constexpr int PFR = PFN > 0 ? PFN : 1;
  int pf_src[PFR], pf_dst[PFR];                                  // offset in the workspace row block; cs index | n << 24
#pragma unroll
  for (int i = 0; i < PFN; ++i) {
    const int id = gtid + GTHR * i;
    pf_src[i] = -1;
    pf_dst[i] = 0;
    if (id < NBG * km2) {
      const int n = id / km2, j = id - n * km2, k = j / m2, kap = j - k * m2;
      pf_src[i] = n * (int)ws.coef_stride + j;
      pf_dst[i] = (((k * KS + (kap >> 2)) * NBG + n) * 4 + (kap & 3)) | (n << 24);
    }
  }
  int pf_off = 0;
  auto cp8 = [](uint32_t dst, const void *src, bool ok) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(ok ? 8 : 0) : "memory");
  };
  auto prefetch = [&](int s0, int run_end, int dst_buf) {
    const int nvalid = min(NBG, run_end - s0);
    const double *src = reinterpret_cast<const double *>(ws.coef) + (int64_t)s0 * ws.coef_stride;
    const uint32_t cs_base = grp_u32 + dst_buf * L.coef_bytes;
#pragma unroll
    for (int i = 0; i < PFN; ++i)
      if (pf_src[i] >= 0) {
        const bool ok = (pf_dst[i] >> 24) < nvalid;
        cp8(cs_base + 8u * (uint32_t)(pf_dst[i] & 0xffffff), src + (ok ? pf_src[i] : 0), ok);
      }
    if (PFN == 0) {
      for (int id = gtid; id < NBG * km2; id += GTHR) {
        const int n = id / km2, j = id - n * km2, k = j / m2, kap = j - k * m2;
        cp8(cs_base + 8u * (uint32_t)(((k * KS + (kap >> 2)) * NBG + n) * 4 + (kap & 3)),
            src + (n < nvalid ? n : 0) * ws.coef_stride + j, n < nvalid);
      }
    }
    if (gtid < 2 * NBG) {                                        // c[NBG], q[NBG]
      const int n = gtid & (NBG - 1);
      const double *mp = (gtid < NBG ? ws.scale_c : ws.quad) + s0 + (n < nvalid ? n : 0);
      cp8(grp_u32 + L.meta + dst_buf * L.meta_bytes + 8u * gtid, mp, n < nvalid);
    }
    pf_off = 0;
    if (gtid < NBG * K) {
      const int k = gtid / NBG, n = gtid - k * NBG;
      if (n < nvalid) {
        const int sk = ws.shift[(int64_t)(s0 + n) * K + k];
        int off = P.circular ? sk - ws.shift[(int64_t)(s0 + n) * K] : P.j0 + sk;
        // out of range only for a sample with NaN angles (its lnL is NaN anyway)
        if (off > H) off = H;
        if (off < (P.circular ? -H : 0)) off = 0;
        pf_off = off;
      }
    }
  };
  auto commit = [&](int buf) {
    asm volatile("cp.async.wait_all;" ::: "memory");
    if (gtid < NBG * K) reinterpret_cast<int *>(grp + L.meta + buf * L.meta_bytes + 2 * NBG * 8)[gtid] = pf_off;
  };

  const int w_begin = (int)((b.n * blockIdx.x) / gridDim.x), w_end = (int)((b.n * (blockIdx.x + 1)) / gridDim.x);
  uint32_t ring_slot = 0, ring_ph = 0, res_phase = 0;            // ring position of the consumers (as the producer's)
  int staged_point = -1, fin_w = 0;
  for (int w0 = w_begin; w0 < w_end;) {                          // runs of one segment: every group takes every other batch
    const int64_t seg = (b.g0 + w0) / b.n_per_seg;
    const int run_end = (int)min((int64_t)w_end, (seg + 1) * b.n_per_seg - b.g0);
    const int point = b.ids[seg];
    if (!STREAM && point != staged_point) {                      // both groups are past the previous run
      if (threadIdx.x == 0) stage_block(qs, A.q + (int64_t)point * P.point_stride, (uint32_t)P.point_stride, resbar);
      mbar_wait(resbar, res_phase);
      res_phase ^= 1u;
      staged_point = point;
    }
    int s0 = w0 + g * NBG;
    int buf = 0;
    if (s0 < run_end) {
      prefetch(s0, run_end, 0);
      commit(0);
    }
    mm_bar(bar_id, GTHR);
    for (; s0 < run_end; s0 += S::GROUPS * NBG, buf ^= 1) {
      const int s_next = s0 + S::GROUPS * NBG;
      if (s_next < run_end) prefetch(s_next, run_end, buf ^ 1);  // copies in flight during this batch
      const double *cs = reinterpret_cast<const double *>(grp + buf * L.coef_bytes);
      const unsigned char *meta = grp + L.meta + buf * L.meta_bytes;
      const int *moff = reinterpret_cast<const int *>(meta + 2 * NBG * 8);

      // ---- detectors: tensor phase, then the tiles go to their window rows (store for k = 0, read-modify-write after)
      auto detector = [&](int k, auto nrb_c) {
        constexpr int NRB = decltype(nrb_c)::value;              // row blocks of this warp; 0: none (ring bookkeeping only)
        double acc[NRB > 0 ? NRB : 1][NT][2];
        const unsigned char *chunk = qs + (size_t)(k * 2 * KS) * P.pitch_q;                        // resident layout
        const double *bs = cs + (size_t)(k * KS) * NBG * 4 + lr * 4 + lc;
        auto kstep = [&](auto first_c) {                           // the first k-step of a detector clears the accumulators
          const uint32_t slot = ring_slot;
          if (STREAM) {
            mbar_wait(full + slot, ring_ph);
            chunk = qs + slot * slot_bytes;
            if (++ring_slot == (uint32_t)P.slots) ring_slot = 0, ring_ph ^= 1u;
          }
          if (NRB > 0) {
            double bf[NT], af[NRB > 0 ? NRB : 1];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) bf[nt] = bs[32 * nt];
#pragma unroll
            for (int i = 0; i < NRB; ++i) af[i] = *reinterpret_cast<const double *>(chunk + a_base + i * (GW * 128));
#pragma unroll
            for (int i = 0; i < NRB; ++i)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) {
                // (a first step written as D = A B + 0 with no read of D raced with the stores of the detector before:
                // the accumulators are cleared by ordinary moves instead)
                if (decltype(first_c)::value) acc[i][nt][0] = acc[i][nt][1] = 0.0;
                dmma(acc[i][nt], af[i], bf[nt]);
              }
          }
          if (STREAM) {
            __syncwarp();
            if (lane == 0) mm_arrive(empty + slot);
          }
          bs += NBG * 4, chunk += slot_bytes;
        };
        kstep(std::true_type());
#pragma unroll 1
        for (int s = 1; s < KS; ++s) kstep(std::false_type());
        if (k > 0) mm_bar(bar_id, GTHR);                         // detector k - 1 is in the window (k = 0: the batch before is read)
        if (NRB > 0) {
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            uint32_t adr[2][NRB > 0 ? NRB : 1];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const int n = 8 * nt + 2 * lc + h, off = moff[k * NBG + n];
              // k = 0: off = 0 (circular) or the guard-band offset, no wrap.  k > 0: tiles i < thr use row r_lo + RS i, the
              // others n_t rows less: off >= 0 wraps the first rows up, off < 0 the last rows down
              const int num = (off >= 0 ? off : n_t + off) - t0;
              const int thr = k == 0 ? NRB : (max(num, 0) + RS - 1) / RS;
              const int r_lo = t0 + row_bias - off + (k > 0 && off >= 0 ? wrap_rows : 0);
              const uint32_t b_lo = x_addr<NT>(xb_u32, r_lo, n), b_hi = x_addr<NT>(xb_u32, r_lo - wrap_rows, n);
#pragma unroll
              for (int i = 0; i < NRB; ++i) adr[h][i] = (i < thr ? b_lo : b_hi) + i * (RS * XP);
            }
            if (k == 0) {
#pragma unroll
              for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int i = 0; i < NRB; ++i) st_shared_f64(adr[h][i], acc[i][nt][h]);
            } else {                                             // all loads of the tile column first: one latency, not NRB
              double v[2][NRB > 0 ? NRB : 1];
#pragma unroll
              for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int i = 0; i < NRB; ++i) v[h][i] = ld_shared_f64(adr[h][i]);
#pragma unroll
              for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int i = 0; i < NRB; ++i)
                  if (i < NRB - 1 || last_ok) st_shared_f64(adr[h][i], v[h][i] + acc[i][nt][h]);
            }
          }
        }
      };
      for (int k = 0; k < K; ++k) {
        switch (nrb) {
          case 0: detector(k, std::integral_constant<int, 0>()); break;
          case 1: detector(k, std::integral_constant<int, 1>()); break;
          case 2: detector(k, std::integral_constant<int, 2>()); break;
          case 3: detector(k, std::integral_constant<int, 3>()); break;
          case 4: detector(k, std::integral_constant<int, 4>()); break;
          case 5: detector(k, std::integral_constant<int, (RBW > 4 ? 5 : 0)>()); break;
          case 6: detector(k, std::integral_constant<int, (RBW > 4 ? 6 : 0)>()); break;
          case 7: detector(k, std::integral_constant<int, (RBW > 4 ? 7 : 0)>()); break;
          default: detector(k, std::integral_constant<int, (RBW > 4 ? 8 : 0)>()); break;
        }
      }
      mm_bar(bar_id, GTHR);                                      // the window is complete

      // ---- time marginal: NE window entries of one sample per thread
      double x[NE];
#pragma unroll
      for (int e = 0; e < NE; ++e)
        x[e] = ld_shared_f64(JS % 8 == 0 ? rd_base + e * (JS * XP) : x_addr<NT>(xb_u32, jb + row_bias + JS * e, n_mine));
      float mf = -INFINITY;
#pragma unroll
      for (int e = 0; e < NE; ++e) mf = fmaxf(mf, e < nv ? __double2float_ru(x[e]) : -INFINITY);
      if (NT == 1) mf = fmaxf(mf, __shfl_xor_sync(0xffffffffu, mf, 8));
      mf = fmaxf(mf, __shfl_xor_sync(0xffffffffu, mf, 16));
      float *wmax = reinterpret_cast<float *>(grp + L.wmax) + buf * NBG * 16;
      if (jj == 0) wmax[n_mine * 16 + wg] = mf;
      mm_bar(bar_id, GTHR);
      {
        const float4 *wm = reinterpret_cast<const float4 *>(wmax + n_mine * 16);
        const float4 a0 = wm[0], a1 = wm[1];
        mf = fmaxf(fmaxf(fmaxf(a0.x, a0.y), fmaxf(a0.z, a0.w)), fmaxf(fmaxf(a1.x, a1.y), fmaxf(a1.z, a1.w)));
        if (GW > 8) {
          const float4 a2 = wm[2], a3 = wm[3];
          mf = fmaxf(mf, fmaxf(fmaxf(fmaxf(a2.x, a2.y), fmaxf(a2.z, a2.w)), fmaxf(fmaxf(a3.x, a3.y), fmaxf(a3.z, a3.w))));
        }
      }
      const double cl2 = reinterpret_cast<const double *>(meta)[n_mine] * 1.4426950408889634;
      const double mo = -(double)mf * cl2;
      double sum = 0.0;
#pragma unroll
      for (int e = 0; e < NE; ++e) {                             // no branch: the NE polynomial chains interleave
        const double pe = poly_exp2(fma(x[e], cl2, mo));
        sum += e < nv ? pe : 0.0;
      }
      if (NT == 1) sum += __shfl_xor_sync(0xffffffffu, sum, 8);
      sum += __shfl_xor_sync(0xffffffffu, sum, 16);
      double *psum = reinterpret_cast<double *>(grp + L.psum) + buf * NBG * 16;
      if (jj == 0) psum[n_mine * 16 + wg] = sum;
      // the warp that writes this batch's lnL (they take turns) reads c and q before the next batch's copies may land
      const bool fin = wg == fin_w && lane < min(NBG, run_end - s0);
      double fc = 0.0, fq = 0.0;
      if (fin) {
        fc = reinterpret_cast<const double *>(meta)[lane];
        fq = reinterpret_cast<const double *>(meta)[NBG + lane];
      }
      if (s_next < run_end) commit(buf ^ 1);                     // the other coefficient buffer was last read a batch ago
      mm_bar(bar_id, GTHR);
      if (fin) {
        double sacc = 0.0;
#pragma unroll
        for (int w = 0; w < (GW > 8 ? 16 : 8); ++w) sacc += psum[lane * 16 + w];
        A.lnL_out[b.g0 + s0 + lane] = fc * (double)mf_of(wmax, lane, GW > 8) + log(sacc) - A.ln_ntau - fq;
      }
      fin_w = fin_w + 1 == GW ? 0 : fin_w + 1;
    }
    if (STREAM && S::GROUPS > 1) {
      // a group without a batch in the last pass of the run still takes the pass's chunks off the ring
      const int n_b = (run_end - w0 + NBG - 1) / NBG, passes = (n_b + S::GROUPS - 1) / S::GROUPS;
      const int mine = n_b > g ? (n_b - g + S::GROUPS - 1) / S::GROUPS : 0;
      for (int pass = mine; pass < passes; ++pass)
        for (int c = 0; c < K * KS; ++c) {
          mbar_wait(full + ring_slot, ring_ph);
          __syncwarp();
          if (lane == 0) mm_arrive(empty + ring_slot);
          if (++ring_slot == (uint32_t)P.slots) ring_slot = 0, ring_ph ^= 1u;
        }
    }
    if (!STREAM) mm_bar(8, S::WARPS * 32);                       // all groups leave the run (and its Q block) together
    else mm_bar(bar_id, GTHR);
    w0 = run_end;
  }
}

template <bool STREAM, int NE, int PFN, int NG>
cudaError_t launch_t(const MmaArgs &a, int n_sm, cudaStream_t s) {
  auto kern = lnl_mma_kernel<STREAM, NE, PFN, NG>;
  const size_t smem = a.L.total;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int64_t grid = n_sm;
  const int64_t max_grid = (a.b.n + 15) / 16;
  if (grid > max_grid) grid = max_grid;
  kern<<<(unsigned)grid, MmaShape<STREAM, NG>::WARPS * 32, smem, s>>>(a);
  return cudaGetLastError();
}

template <bool STREAM, int PFN, int NG>
cudaError_t launch_ne(const MmaArgs &a, int n_sm, cudaStream_t s) {
  switch (a.p.ne) {
    case 4: return launch_t<STREAM, 4, PFN, NG>(a, n_sm, s);
    case 8: return launch_t<STREAM, 8, PFN, NG>(a, n_sm, s);
    case 13: return launch_t<STREAM, 13, PFN, NG>(a, n_sm, s);
    case 14: return launch_t<STREAM, 14, PFN, NG>(a, n_sm, s);
    case 16: return launch_t<STREAM, 16, PFN, NG>(a, n_sm, s);
    default: return cudaErrorInvalidValue;
  }
}

// [rows][n_t] complex128 -> the operand layout described at the top: [P][K][M2][pitch] bytes
__global__ void convert_q_mma_kernel(const double2 *__restrict__ src, unsigned char *__restrict__ dst, int P, int K, int M,
                                     int M2, int n_t, int pitch) {
  const int64_t per_row = pitch / 16;                                       // 16-byte units per row, pad included
  const int64_t total = (int64_t)P * K * M2 * per_row;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = i / per_row;
    const int t = (int)(i - row * per_row);
    const int m = (int)(row % M2);
    const int64_t pk = row / M2;
    double2 v = make_double2(0.0, 0.0);
    if (m < M && t < n_t) v = src[(pk * M + m) * n_t + t];
    reinterpret_cast<double2 *>(dst)[i] = v;
  }
}

}  // namespace

// Completes a plan whose K, M, n_t, n_tau, H (circular halo) and stream / slots are set; returns false when the window is too
// long for the 16 register entries per thread or the row blocks of the CTA.
bool lnl_mma_finish_plan(MmaPlan &p) {
  const bool wide = p.stream && p.groups == 1;          // one group of 15 warps with batches of 16 samples
  const int gw = p.stream ? (wide ? 15 : 7) : 8, nbg = wide ? 16 : 8, rbw = wide ? 4 : 8, js = (wide ? 2 : 4) * gw;
  p.KS = (p.M + 1) / 2;
  p.n_r = (p.n_t + 7) & ~7;
  p.circular = p.n_tau == p.n_t ? 1 : 0;
  p.n_x = p.n_tau;
  p.j0 = (p.n_t - p.n_tau) / 2;
  if (!p.circular) p.H = p.n_t - p.n_tau;                 // guard band: 0 <= off = j0 + s_k <= 2 j0
  p.pitch_q = p.n_r * 16 + 64;
  p.point_stride = (int64_t)p.K * 2 * p.KS * p.pitch_q;
  const int need = (p.n_x + js - 1) / js;
  static const int nes[] = {4, 8, 13, 14, 16};
  p.ne = 0;
  for (int v : nes)
    if (v >= need) {
      p.ne = v;
      break;
    }
  const int items = (nbg * 2 * p.K * p.M + gw * 32 - 1) / (gw * 32);
  p.pfn = (!p.stream && items <= 2) ? 2 : 0;
  p.xb_rows = (p.ne * js > p.n_r ? p.ne * js : p.n_r) + (p.circular ? 0 : p.H) + 8;   // window rows (+ guard-band bias)
  return p.ne != 0 && p.n_r <= 8 * rbw * gw && p.H < p.n_t && p.K * nbg <= gw * 32 &&
         (p.stream || p.point_stride < (1ll << 20));
}

size_t lnl_mma_smem_bytes(const MmaPlan &p) { return mma_smem(p).total; }

cudaError_t launch_convert_q_mma(const double *Q_c128, void *dst, const MmaPlan &p, int32_t n_points, cudaStream_t s) {
  const int64_t total = (int64_t)n_points * p.K * 2 * p.KS * (p.pitch_q / 16);
  int grid = (int)((total + 255) / 256);
  if (grid > 148 * 16) grid = 148 * 16;
  if (grid < 1) grid = 1;
  convert_q_mma_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<const double2 *>(Q_c128), reinterpret_cast<unsigned char *>(dst),
                                            n_points, p.K, p.M, 2 * p.KS, p.n_t, p.pitch_q);
  return cudaGetLastError();
}

cudaError_t launch_lnl_mma(const MmaPlan &p, const void *q, const Batch &b, const Workspace &ws, double *lnL_out, int n_sm,
                           cudaStream_t s, int *n_launch) {
  if (b.n <= 0) return cudaSuccess;
  if (b.n > 0x7fffffff) return cudaErrorInvalidValue;             // slots of a chunk are 32-bit inside the kernel
  MmaArgs a;
  a.p = p;
  a.L = mma_smem(p);
  a.q = reinterpret_cast<const unsigned char *>(q);
  a.b = b;
  a.ws = ws;
  a.lnL_out = lnL_out;
  a.ln_ntau = log((double)p.n_tau);
  if (n_launch) ++*n_launch;
  if (p.stream) return p.groups == 2 ? launch_ne<true, 0, 2>(a, n_sm, s) : launch_ne<true, 0, 1>(a, n_sm, s);
  if (p.groups == 3) return p.pfn == 2 ? launch_ne<false, 2, 3>(a, n_sm, s) : launch_ne<false, 0, 3>(a, n_sm, s);
  return p.pfn == 2 ? launch_ne<false, 2, 2>(a, n_sm, s) : launch_ne<false, 0, 2>(a, n_sm, s);
}
