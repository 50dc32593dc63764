// Internal declarations shared by the CUDA translation units of librift_ile.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <cmath>

#include "rift_ile.h"

#define RIFT_MAX_TERMS 8         // terms of the Wigner-d sum of one mode (l <= 8  =>  <= l-1 = 7)
#define RIFT_C_LIGHT 299792458.0

struct ModeEntry {               // one (l,m): -2Y_lm(th,ph) = e^{i m ph} sum_t coef[t] cos(th/2)^pc[t] sin(th/2)^ps[t]
  int32_t l, m, n_terms, pad;
  double coef[RIFT_MAX_TERMS];
  int32_t pc[RIFT_MAX_TERMS];
  int32_t ps[RIFT_MAX_TERMS];
};

struct DetGeom {                 // passed by value to the geometry kernel
  int32_t n_det, n_modes, l_max, pad;
  double gmst, delta_t, d_ref;
  double loc[RIFT_MAX_DET][3];
  double resp[RIFT_MAX_DET][9];
};

// A chunk = contiguous range [g0, g0 + n) of the caller's flattened sample index g = seg * n_per_seg + i.
struct Batch {
  int64_t n_per_seg;
  int64_t g0;
  int64_t n;
  const int32_t *ids;            // device [n_seg]: intrinsic point of each segment
};

// Per-sample workspace written by the geometry kernel for one chunk (slot = g - g0)
struct Workspace {
  void *coef;                    // [n][coef_stride] Real, the first 2*K*M hold complex B_{k,lm} = F_k * Y_lm (step a5)
  int64_t coef_stride;           // Reals per sample: 2*K*M rounded up to a 16-byte multiple
  double *scale_c;               // [n] c = D_ref / D (NaN marks an invalid sample)
  double *quad;                  // [n] q, the U/V term of Eq. (D3)
  int32_t *shift;                // [n][K]
  int32_t *orig;                 // [n] chunk-local index of the caller's sample held in this slot (NULL = identity)
};

// Device copy of Q.  Interleaved layout (direct kernel): [P][K*M][n_tp] complex<Real>, n_tp = n_t rounded up to even.
// Extended layout (direct_ext): every row is followed by a circular repeat of its first RIFT_EXT samples (so base + j
// never needs a wrap), zero padded.
struct QStore {
  const void *data;
  int32_t n_t, n_tp, n_tau, km;
  int64_t point_stride_bytes;
};
#define RIFT_EXT 416             // 13 slots x 32 lanes: one time block of the fused kernels

// Tensor-core path (lnl_tc.cu): plan of one handle.  Samples are processed in batches of RIFT_TC_NB consecutive samples
// of one segment; the geometry kernel writes one "blob" per batch: the B operand of the UMMA in its canonical K-major
// shared-memory layout, [K][nch][16 samples][8 fp16] (per detector the contraction index runs over [B_hi | B_hi | B_lo],
// kp = 6M rounded up to 16 elements, in 16-byte chunks of 8), then the relative shifts d_k = s_k - s_0 as int32 [K][16],
// then c*log2(e) / (operand scales) as float [16].
#define RIFT_TC_NB 16
#define RIFT_TC_BSCALE 8192.0    // 2^13: scale of the coefficient operand (|F_k Y_lm| < 2) into the fp16 range
struct TcPlan {
  int32_t ok;                    // 1 if this handle can run the tensor-core kernel
  int32_t K, M, n_t, nt;         // nt = ceil(n_t / 128) row tiles
  int32_t n_sub, m_sub;          // mode subsets (passes) and modes per subset; kp, nch, acols refer to ONE subset
  int32_t n_tau, j0;             // marginalisation samples and first window index (n_t - n_tau) / 2; n_tau == n_t: circular
  int32_t kp, nch, acols;        // contraction length (fp16 elements), 16-byte chunks per detector, TMEM columns of one A tile
  int32_t H, pitch;              // halo = max_k dmax[k]; exchange-row pitch in floats
  int32_t blob_words, dcol0;     // 32-bit words per batch blob; first accumulator column in TMEM
  int32_t dmax[RIFT_MAX_DET];    // bound on |s_k - s_0|
  // sorted variant (lnl_tcs.cu): batches hold samples of ONE relative shift d_1 = s_1 - s_0, so that detector 1 is contracted
  // from a shared-memory A operand whose rows start at d_1 and accumulates straight onto detector 0; detectors >= 2 keep
  // the exchange.  n_bkt = 2 dmax[1] + 1 shift buckets per segment; as_rows = rows of the extended detector-1 operand
  // (row r = time r - dmax[1], wrapped), [kp/8 planes][as_rows][8 fp16]; blob_words_s = blob_words + 4 (batch header: d_1).
  int32_t srt_ok, n_bkt, as_rows, pitch_s, blob_words_s, dcol0_s;
};
struct TcChunk {                 // a chunk = global batches [gb0, gb0 + n_batches), batch gb = seg * nbps + b
  int64_t n_per_seg, nbps, gb0, n_batches;
  const int32_t *ids;
  const float *qscale;           // [P] power-of-two scale applied to Q of each point in the A operand
  float *blob;                   // [n_batches][blob_words]
  double *scale_c, *quad;        // [n_batches * 16]
  float2 *part;                  // [n_batches * 16][4]: per lane-quarter (reference, sum)
  float *xacc;                   // [n_batches * 16][nt * 128]: window sums carried between mode-subset passes (or NULL)
  // sorted variant: key == NULL means natural order.  Natural slot w = (local batch) * 16 + n; sorted slots are assigned
  // per (local segment, shift bucket) in arrival order, every bucket padded to whole batches.
  int32_t *key;                  // [n_batches * 16] bucket index (lseg * n_bkt + d_1 + dmax[1]) of a natural slot, -1 = padding
  int32_t *pos;                  // [n_batches * 16] position of a natural slot inside its bucket
  int32_t *count, *base;         // [n_lseg * n_bkt] samples per bucket, first sorted batch of the bucket
  int32_t *seg_begin;            // [n_lseg + 1] first sorted batch of each local segment; seg_begin[n_lseg] = sorted batches
  int32_t *perm;                 // [cap_sorted * 16] natural slot of a sorted slot, -1 = padding
  int32_t n_lseg;                // segments touched by this chunk
  int64_t cap_sorted;            // capacity in sorted batches (n_batches + n_lseg * n_bkt)
};
// Mode-subset passes of lnl_tc (configurations whose A operand does not fit tensor memory whole, e.g. 21 modes): the modes are
// split into n_sub subsets of m_sub; pass s contracts subset s and adds the window sums of the passes before it.
enum { RIFT_TC_PASS_SINGLE = 0, RIFT_TC_PASS_FIRST = 1, RIFT_TC_PASS_MIDDLE = 2, RIFT_TC_PASS_LAST = 3 };

// Pair program of the quadratic term a4 for mode sets of more than 8 modes (geometry.cu).  With Y_a = d_a(iota) z^{m_a},
// z = e^{-i phi}, the products conj(Y_a) Y_b = d_a d_b z^{m_b - m_a} and Y_a Y_b = d_a d_b z^{m_a + m_b} share their phase among all
// mode pairs of equal exponent n, so  Y^dag U_k Y = sum_n Re( z^n S^U_{k,n} ),  Y^T V_k Y = sum_n z^n S^V_{k,n}  with
// S_{k,n} = sum_{pairs of exponent n} (d_a d_b) W_{k,ab}:  one real weight and 2 K FMAs per (pair, matrix) instead of two complex
// products and 6 K FMAs.  An entry is one pair a <= b of one matrix; W is U_ab (or conj U_ab when m_b < m_a, exponent
// |m_b - m_a|) resp. V_ab, times 2 off the diagonal (U Hermitian, V symmetric).  Bins are runs of entries of one (matrix,
// exponent), ordered U: n = 0, 1, ...; V: n = 0, 1, ..., then n = -1, -2, ... so that z^n is carried by one complex
// multiplication per bin.
#define RIFT_QP_MAX_ENT 1024     // mode pairs of both matrices: M (M + 1) <= 1024, i.e. up to 31 modes
#define RIFT_QP_AMP_STRIDE 1024u  // bytes between d_a and d_{a+1} in a thread's amplitude column (128 threads x 8 bytes)
#define RIFT_QP_MAX_BINS 52      // (2 n_max + 1) + n_max + 1 + ... <= 50 for l <= 8
struct QuadProg {                // passed to the kernels as a __grid_constant__ parameter: the tables are read from the constant bank
  int32_t n_entries, n_bins;
  const uint32_t *ent_full;      // device [n_entries]: a | b << 8 | matrix << 16 (0 U, 1 V) | conj << 17 (used to build uv)
  const double2 *uv;             // device [P][n_entries][K]: W of every entry and detector; NULL = no program
  uint2 ent[RIFT_QP_MAX_ENT];                // byte offsets of d_a and d_b in a thread's amplitude column (a * RIFT_QP_AMP_STRIDE)
  uint16_t bin_begin[RIFT_QP_MAX_BINS + 1];  // entries of bin i: [bin_begin[i], bin_begin[i + 1])
  uint8_t bin_kind[RIFT_QP_MAX_BINS];        // matrix | z step << 1  (0 z^0, 1 *= z, 2 conj z, 3 *= conj z)
};

// FP64 tensor-core path (lnl_mma.cu): plan of one handle.  Batches of 16 samples; the Q operand is [P][K][2 KS][pitch_q] bytes
// (see lnl_mma.cu), resident in shared memory (stream == 0) or streamed one (detector, k-step) chunk at a time through
// `slots` ring slots; the exchange buffer holds xb_rows rows of 16 doubles; a thread keeps `ne` window entries in registers.
struct MmaPlan {
  int32_t ok;
  int32_t K, M, KS;              // KS = ceil(M / 2) k-steps of 4 real contraction elements (2 modes) per detector
  int32_t n_t, n_r, n_tau, n_x;  // stored rows, rows padded to 8, marginalisation samples, window entries
  int32_t j0, circular;
  int32_t H;                     // circular: bound on |s_k - s_0| (halo rows); guard band: n_t - n_tau
  int32_t ne, pfn, xb_rows, stream, slots;
  int32_t groups;                // resident shape: independent 8-warp groups per CTA (2 or 3)
  int32_t pitch_q;               // bytes per mode row: n_r * 16 + 64
  int64_t point_stride;          // bytes per intrinsic point
};

// Sky-sorted, time-tiled tensor-core path (sky_sort.cu, lnl_sky.cu): mixed precision, windows of any length.
#define SKY_NB 64                // samples per batch (eight 8-column tiles)
#define SKY_E 24                 // mixed mode (lnl_sky): residual shifts of a batch lie in [0, SKY_E)
#define SKY64_E 32               // fp64 mode (lnl_sky64): its chunks start at any row, so 224 + 32 = 256 rows
#define SKY_TBO 224              // window entries per time block (a multiple of 8)
#define SKY_TBR 256              // Q rows per (time block, detector) chunk >= SKY_TBO + SKY_E + 7
#define SKY_MAX_RINGS 512
struct SkyCells {                // sky cells of the bucketing pass (sky_sort.cu)
  double delta;                  // ring width (rad)
  int32_t n_rings, n_cells;
  int32_t ring_off[SKY_MAX_RINGS + 1];   // first cell of each declination ring
};
struct SkyPlan {
  int32_t ok;
  int32_t K, M, n_t;
  int32_t kp, rowb;              // fp16 elements per operand row [Q_hi | Q_lo | Q_hi] (padded), bytes per row
  int32_t n_pc, ppp;             // the row is cut into n_pc K pieces of ppp planes of 8 elements (ppp even, <= 8): kp = 8 n_pc ppp
  int32_t R0, rows_ext;          // extended row of original row 0; rows per (point, detector): row e holds (e - R0) mod n_t
  int32_t n_blocks;              // time blocks of SKY_TBO window entries
  int64_t point_stride;          // bytes per intrinsic point: K * rows_ext * rowb
};

struct Sky64Plan {               // fp64 sibling (lnl_sky64.cu): operand rows of kp doubles (kp = 4 mod 8), KS = kp / 4 k-steps
  int32_t ok;
  int32_t K, M, n_t, kp, KS;
  int32_t R0, rows_ext, n_blocks, slots;   // blocks of 224 window entries; ring slots of 256 rows
  int64_t point_stride;          // bytes per intrinsic point: K * rows_ext * kp * 8
};

// geometry.cu
cudaError_t launch_geometry_tc(const DetGeom &g, const ModeEntry *modes, const TcPlan &tp, const TcChunk &c,
                               const double *const params[6], const double *U, const double *V, const QuadProg &qp,
                               int32_t *shift_out, cudaStream_t s);
cudaError_t launch_geometry(const DetGeom &g, const ModeEntry *modes, const Batch &b, const double *const params[6],
                            const double *U, const double *V, const QuadProg &qp, bool coef_fp32, const Workspace &ws,
                            int32_t *shift_out, double *dbg_F, double *dbg_Y, const int32_t *perm, cudaStream_t s);
cudaError_t launch_build_quad_uv(const QuadProg &qp, const double *U, const double *V, int32_t P, int32_t K, int32_t M,
                                 double2 *uv_out, cudaStream_t s);
// sky_frame.cu
cudaError_t launch_rho_guess(const QStore &q, bool q_fp32, const double *U, int32_t P, int32_t K, int32_t M, double *out,
                             cudaStream_t s);
// lnl_direct.cu
size_t lnl_direct_smem_bytes(const QStore &q, bool fp32, bool q_in_smem);
cudaError_t launch_lnl_direct(const QStore &q, bool fp32, bool q_in_smem, bool q_ext, const Batch &b, const Workspace &ws,
                              int n_det, double *lnL_out, int n_sm, cudaStream_t s, int *n_launch);
size_t lnl_direct_dm_smem_bytes(const QStore &q, bool fp32, bool q_in_smem, int n_dist);
cudaError_t launch_lnl_direct_dmarg(const QStore &q, bool fp32, bool q_in_smem, bool q_ext, const Batch &b,
                                    const Workspace &ws, int n_det, int n_dist, const double *c_nodes, const double *lnw_nodes,
                                    double *lnL_out, int n_sm, cudaStream_t s, int *n_launch);   // NEXT-2, distance marginal
// lnl_direct_ext.cu (interleaved layout with a circular extension of RIFT_EXT samples per row)
size_t lnl_direct_ext_smem_bytes(const QStore &q, bool fp32);
cudaError_t launch_lnl_direct_ext(const QStore &q, bool fp32, const Batch &b, const Workspace &ws, int n_det,
                                  double *lnL_out, int n_sm, cudaStream_t s, int *n_launch);
cudaError_t launch_convert_q_ext(const double *Q_c128, void *dst, int64_t rows, int32_t n_t, int32_t n_te, bool to_fp32,
                                 cudaStream_t s);
// lnl_tc.cu (tcgen05 / TMEM contraction, shift applied through a shared-memory exchange)
size_t lnl_tc_smem_bytes(const TcPlan &tp);
int lnl_tc_pitch(int n_t, int halo);   // exchange-row pitch (floats) the kernel is instantiated for, 0 = none fits
cudaError_t launch_convert_q_tc(const double *Q_c128, uint32_t *dst, float *qscale, const TcPlan &tp, int32_t n_points,
                                cudaStream_t s);   // dst: [n_sub][P][K][nt*128][acols]
cudaError_t launch_lnl_tc(const TcPlan &tp, const uint32_t *qtc, const TcChunk &c, int pass, double *lnL_out, int n_sm,
                          cudaStream_t s, int *n_launch);
// lnl_tcs.cu (sorted variant: detector 1 fused into detector 0 by the tensor core; geometry.cu holds the bucket kernels)
size_t lnl_tcs_smem_bytes(const TcPlan &tp);
cudaError_t launch_convert_q_tcs(const double *Q_c128, uint16_t *dst, const float *qscale, const TcPlan &tp,
                                 int32_t n_points, cudaStream_t s);   // dst: [n_sub][P][kp/8][as_rows][8] fp16, detector 1
cudaError_t launch_tcs_buckets(const DetGeom &g, const TcPlan &tp, const TcChunk &c, const double *const params[6],
                               cudaStream_t s, int *n_launch);        // key, pos, count, base, seg_begin, perm
cudaError_t launch_lnl_tcs(const TcPlan &tp, const uint32_t *qtc, const uint16_t *qs, const TcChunk &c, int pass,
                           double *lnL_out, int n_sm, cudaStream_t s, int *n_launch);
// lnl_mma.cu (fp64 mode: DMMA contraction in unshifted detector time, shift applied into a shared-memory window buffer)
bool lnl_mma_finish_plan(MmaPlan &p);
size_t lnl_mma_smem_bytes(const MmaPlan &p);
cudaError_t launch_convert_q_mma(const double *Q_c128, void *dst, const MmaPlan &p, int32_t n_points, cudaStream_t s);
cudaError_t launch_lnl_mma(const MmaPlan &p, const void *q, const Batch &b, const Workspace &ws, double *lnL_out, int n_sm,
                           cudaStream_t s, int *n_launch);
// sky_sort.cu / lnl_sky.cu
bool sky_make_cells(double dmax_samples, int e_max, SkyCells &c);
cudaError_t launch_sky_sort(const SkyCells &cells, double gmst, const Batch &b, const double *const params[6], int n_lseg,
                            int32_t *key, int32_t *pos, int32_t *count, int32_t *base, int32_t *perm, int64_t cap_slots,
                            int32_t *n_batches, cudaStream_t s, int *n_launch);
size_t lnl_sky_smem_bytes(const SkyPlan &p);
cudaError_t launch_convert_q_sky(const double *Q_c128, void *dst, float *qscale, const SkyPlan &p, int32_t n_points,
                                 cudaStream_t s);
cudaError_t launch_lnl_sky(const SkyPlan &p, const void *q, const float *qscale, const Batch &b, const Workspace &ws,
                           const int32_t *n_batches_dev, int64_t max_batches, double *lnL_out, int n_sm, cudaStream_t s,
                           int *n_launch);
size_t lnl_sky64_smem_bytes(const Sky64Plan &p);
cudaError_t launch_convert_q_sky64(const double *Q_c128, void *dst, const Sky64Plan &p, int32_t n_points, cudaStream_t s);
cudaError_t launch_lnl_sky64(const Sky64Plan &p, const void *q, const Batch &b, const Workspace &ws,
                             const int32_t *n_batches_dev, int64_t max_batches, double *lnL_out, int n_sm, cudaStream_t s,
                             int *n_launch);
// precompute.cu (NEXT-3: Q, U, V from frequency series)
cudaError_t launch_precompute(int32_t P, int32_t K, int32_t M, int32_t n_freq, const void *h, const void *d, const double *w,
                              const double *f, int equal_spacing, double df, int32_t n_t, double delta_t, void *Q, void *U,
                              void *V, cudaStream_t s);
// reduce.cu
struct ReduceState {             // device, per segment
  double m, s1, s2;
  int64_t n;
};
cudaError_t launch_reduce(int32_t n_seg, int64_t n_per_seg, const double *lnL, const double *ln_w,
                          const double *const params[6], const double lo[6], const double hi[6], int32_t n_bins,
                          int merge, ReduceState *state, double *state_hist, double *partial, int32_t blocks_per_seg,
                          double *out_scalars /*[4][n_seg]*/, double *out_hist, cudaStream_t s, int *n_launch);
size_t reduce_partial_doubles(int32_t n_seg, int32_t blocks_per_seg, int32_t n_bins);
int32_t reduce_blocks_per_seg(int64_t n_per_seg, int32_t n_seg);
// convert.cu
cudaError_t launch_convert_q(const double *Q_c128, void *dst, int64_t rows, int32_t n_t, int32_t n_tp, bool to_fp32,
                             cudaStream_t s);
cudaError_t launch_fill_f64(double *dst, int64_t n, double value, cudaStream_t s);
cudaError_t run_fma_peak(int mode, int iters, double *tflops, cudaStream_t s);   // 0 fp32, 1 fp64, 2 fp32 register tile
