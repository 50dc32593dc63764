// C ABI of librift_ile.so (include/rift_ile.h): handle management, argument validation, chunking, launches.
// Host logic only -- every step of the hot path runs in the kernels of geometry.cu, lnl_*.cu and reduce.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "rift_internal.h"

struct rift_ile {
  int device = 0, n_sm = 0;
  int P = 0, K = 0, M = 0, n_t = 0, n_tp = 0, n_tau = 0;
  int precision = 0, q_storage = 0;
  DetGeom geom{};
  ModeEntry *d_modes = nullptr;
  void *d_Q = nullptr;
  double *d_U = nullptr, *d_V = nullptr;
  QuadProg qp{};                   // pair program of the quadratic term (M > 8), device tables owned by the handle
  QStore qs{};
  void *d_Qe = nullptr;            // interleaved, circularly extended copy for the direct_ext kernel (NULL if too big)
  QStore qse{};
  void *d_Qg = nullptr;            // the same extended layout for configurations whose Q block does NOT fit shared memory:
  QStore qsg{};                    // lnl_direct reads it from global memory with one address per mode row (no wrap arithmetic)
  MmaPlan mma{};                   // fp64 tensor-core path (lnl_mma.cu); mma.ok == 0 when the configuration does not fit
  void *d_Qm = nullptr;            // its Q operand: [P][K][2 KS][pitch_q] bytes
  SkyPlan sky{};                   // sky-sorted, time-tiled tensor-core path (lnl_sky.cu); sky.ok == 0: does not apply
  Sky64Plan sky64{};               // its fp64 sibling (lnl_sky64.cu)
  void *d_Qsky64 = nullptr;        // [P][K][rows_ext][kp] doubles
  SkyCells sky_cells{};
  void *d_Qsky = nullptr;          // its Q operand: [P][K][rows_ext][kp] fp16
  float *d_qscale_sky = nullptr;   // [P]
  int32_t *sky_buf = nullptr;      // key, pos, count, base, perm, n_batches of a chunk
  int64_t sky_buf_cap = 0;
  int32_t *sky_orig = nullptr;     // [slots] chunk-local sample of a sorted slot
  int64_t sky_orig_cap = 0;
  TcPlan tc{};                     // tensor-core path (lnl_tc.cu); tc.ok == 0 when the configuration does not fit
  uint32_t *d_Qtc = nullptr;       // A operand: [P][K][nt*128][acols] words of two fp16
  float *d_qscale = nullptr;       // [P] power-of-two scale of each point's Q in the A operand
  float *tc_blob = nullptr;        // per-chunk workspace of the tensor-core path
  double *tc_c = nullptr, *tc_quad = nullptr;
  float2 *tc_part = nullptr;
  float *tc_xacc = nullptr;        // window sums carried between mode-subset passes (n_sub > 1)
  int64_t tc_cap = 0;              // batches the workspace holds
  uint16_t *d_Qs = nullptr;        // sorted variant (lnl_tcs.cu): extended detector-1 operand [P][kp/8][as_rows][8] fp16
  int32_t *tcs_key = nullptr, *tcs_perm = nullptr, *tcs_bkt = nullptr;   // natural-slot keys, sorted-slot permutation, bucket tables
  int64_t tcs_key_cap = 0, tcs_perm_cap = 0, tcs_bkt_cap = 0;
  // options (rift_ile_set_option)
  int64_t opt_tc_chunk_mib = 4096; // per-chunk workspace of the tensor-core kernels
  int opt_tc_sort = 1;             // AUTO may pick the shift-sorted tensor-core kernel
  int opt_quad_prog = 1;           // pair program of the quadratic term when M > 8
  const double2 *qp_uv_saved = nullptr;   // the program's W table while the option is off
  // per-chunk workspace
  int64_t ws_cap = 0;
  Workspace ws{};
  int32_t *d_ids = nullptr;
  std::vector<int32_t> ids_last;   // host copy of the ids d_ids holds, and the stream that uploaded them: an unchanged id list
  cudaStream_t ids_stream = nullptr;   // is not copied again, so a steady-state eval_batch is kernel launches only (graph capture)
  int64_t ids_cap = 0;
  // reduce state
  ReduceState *d_state = nullptr;
  double *d_state_hist = nullptr;
  int state_nseg = 0, state_nbins = -1;
  double *d_partial = nullptr;
  size_t partial_cap = 0;
  double *d_out = nullptr, *h_out = nullptr;
  size_t out_cap = 0;
  // host-buffer path (rift_ile_eval_batch_host): device staging [7][host_cap] (six parameters, ln weight) + lnL[host_cap],
  // an upload and a read-back stream, and the events that chain the slices
  double *d_hp = nullptr, *d_hl = nullptr;
  int64_t host_cap = 0, host_n = 0;
  bool host_has_w = false;
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  std::vector<cudaEvent_t> host_ev;
  // distance marginalisation (rift_ile_eval_batch_dmarg): quadrature nodes c_i = D_ref/D_i, ln W_i; a distance column = D_ref
  double *d_dm_nodes = nullptr, *d_dm_dist = nullptr;
  int dm_n = 0;
  double dm_dmin = 0, dm_dmax = 0;
  int64_t dm_dist_cap = 0;
  // bookkeeping
  int kernel_variant = RIFT_KERNEL_AUTO;
  const char *kernel_name = "none";
  int64_t launches = 0;
  char err[512] = {0};
  // optional per-kernel event timing (rift_ile_profile)
  bool profiling = false;
  struct Span { cudaEvent_t a, b; int kind; };
  std::vector<Span> spans;
};

namespace {

struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

int fail(rift_ile *h, int code, const char *what, cudaError_t ce = cudaSuccess) {
  if (h) {
    if (ce != cudaSuccess)
      snprintf(h->err, sizeof(h->err), "%s: %s", what, cudaGetErrorString(ce));
    else
      snprintf(h->err, sizeof(h->err), "%s", what);
  }
  return code;
}

#define CU(h, call)                                                   \
  do {                                                                \
    cudaError_t e__ = (call);                                         \
    if (e__ != cudaSuccess) {                                         \
      cudaGetLastError();                                             \
      return fail(h, e__ == cudaErrorMemoryAllocation ? RIFT_ENOMEM : RIFT_ECUDA, #call, e__); \
    }                                                                 \
  } while (0)

// RAII-less helper: record an event pair around a launch when profiling is on
struct ProfSpan {
  rift_ile *h;
  cudaStream_t s;
  rift_ile::Span sp{};
  bool on = false;
  ProfSpan(rift_ile *h_, int kind, cudaStream_t s_) : h(h_), s(s_) {
    if (h->profiling && cudaEventCreate(&sp.a) == cudaSuccess) {
      if (cudaEventCreate(&sp.b) == cudaSuccess) {
        sp.kind = kind;
        on = true;
        cudaEventRecord(sp.a, s);
      } else {
        cudaEventDestroy(sp.a);
      }
    }
  }
  void end() {
    if (on) {
      cudaEventRecord(sp.b, s);
      h->spans.push_back(sp);
      on = false;
    }
  }
};

double factorial(int n) {
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f *= i;
  return f;
}

// Term table of -2Y_lm (reading G3): coefficient, power of cos(theta/2), power of sin(theta/2).
void build_mode(int l, int m, ModeEntry &e) {
  memset(&e, 0, sizeof(e));
  e.l = l;
  e.m = m;
  const int k0 = (m - 2 > 0) ? m - 2 : 0;
  const int k1 = (l + m < l - 2) ? l + m : l - 2;
  const long double pref = sqrtl((long double)factorial(l + m) * factorial(l - m) * factorial(l + 2) * factorial(l - 2)) *
                           sqrtl((2.0L * l + 1.0L) / (4.0L * 3.14159265358979323846264338327950288L));
  int n = 0;
  for (int k = k0; k <= k1; ++k, ++n) {
    const long double den = (long double)factorial(l + m - k) * factorial(l - 2 - k) * factorial(k) * factorial(k - m + 2);
    e.coef[n] = (double)(((k & 1) ? -1.0L : 1.0L) * pref / den);
    e.pc[n] = 2 * l + m - 2 - 2 * k;
    e.ps[n] = 2 * k - m + 2;
  }
  e.n_terms = n;
}

void free_handle(rift_ile *h) {
  if (!h) return;
  for (auto &sp : h->spans) {
    cudaEventDestroy(sp.a);
    cudaEventDestroy(sp.b);
  }
  for (auto &e : h->host_ev) cudaEventDestroy(e);
  if (h->s_h2d) cudaStreamDestroy(h->s_h2d);
  if (h->s_d2h) cudaStreamDestroy(h->s_d2h);
  cudaFree(h->d_hp);
  cudaFree(h->d_hl);
  cudaFree(h->d_dm_nodes);
  cudaFree(h->d_dm_dist);
  cudaFree(h->d_modes);
  cudaFree(h->d_Q);
  cudaFree(h->d_Qe);
  cudaFree(h->d_Qtc);
  cudaFree(h->d_Qm);
  cudaFree(h->d_Qsky);
  cudaFree(h->d_Qsky64);
  cudaFree(h->d_qscale_sky);
  cudaFree(h->sky_buf);
  cudaFree(h->sky_orig);
  cudaFree(h->d_qscale);
  cudaFree(h->tc_blob);
  cudaFree(h->tc_c);
  cudaFree(h->tc_quad);
  cudaFree(h->tc_part);
  cudaFree(h->tc_xacc);
  cudaFree(h->d_Qs);
  cudaFree(h->tcs_key);
  cudaFree(h->tcs_perm);
  cudaFree(h->tcs_bkt);
  cudaFree(const_cast<uint32_t *>(h->qp.ent_full));
  cudaFree(const_cast<double2 *>(h->qp.uv ? h->qp.uv : h->qp_uv_saved));
  cudaFree(h->d_Qg);
  cudaFree(h->d_U);
  cudaFree(h->d_V);
  cudaFree(h->ws.coef);
  cudaFree(h->ws.scale_c);
  cudaFree(h->ws.quad);
  cudaFree(h->ws.shift);
  cudaFree(h->d_ids);
  cudaFree(h->d_state);
  cudaFree(h->d_state_hist);
  cudaFree(h->d_partial);
  cudaFree(h->d_out);
  if (h->h_out) cudaFreeHost(h->h_out);
  delete h;
}

int64_t coef_stride(const rift_ile *h) {          // Reals per sample, a multiple of 16 bytes
  const int64_t n = 2 * (int64_t)h->K * h->M;
  return h->precision == RIFT_PREC_MIXED ? ((n + 3) & ~3ll) : n;
}
size_t coef_bytes(const rift_ile *h) { return (size_t)coef_stride(h) * (h->precision == RIFT_PREC_MIXED ? 4 : 8); }

int ensure_workspace(rift_ile *h, int64_t n) {
  if (n <= h->ws_cap) return RIFT_OK;
  cudaFree(h->ws.coef);
  cudaFree(h->ws.scale_c);
  cudaFree(h->ws.quad);
  cudaFree(h->ws.shift);
  h->ws = Workspace{};
  h->ws_cap = 0;
  CU(h, cudaMalloc(&h->ws.coef, (size_t)n * coef_bytes(h)));
  h->ws.coef_stride = coef_stride(h);
  CU(h, cudaMalloc(&h->ws.scale_c, (size_t)n * sizeof(double)));
  CU(h, cudaMalloc(&h->ws.quad, (size_t)n * sizeof(double)));
  CU(h, cudaMalloc(&h->ws.shift, (size_t)n * h->K * sizeof(int32_t)));
  h->ws_cap = n;
  return RIFT_OK;
}

int upload_ids(rift_ile *h, int32_t n_seg, const int32_t *ids, cudaStream_t s) {
  for (int32_t i = 0; i < n_seg; ++i)
    if (ids[i] < 0 || ids[i] >= h->P) return fail(h, RIFT_ERANGE, "intrinsic id outside [0, n_points)");
  if (n_seg > h->ids_cap) {
    cudaFree(h->d_ids);
    h->d_ids = nullptr;
    h->ids_cap = 0;
    CU(h, cudaMalloc(&h->d_ids, (size_t)n_seg * sizeof(int32_t)));
    h->ids_cap = n_seg;
    h->ids_last.clear();
  }
  if (h->ids_stream == s && (int32_t)h->ids_last.size() == n_seg &&
      memcmp(h->ids_last.data(), ids, (size_t)n_seg * sizeof(int32_t)) == 0)
    return RIFT_OK;
  h->ids_last.clear();
  CU(h, cudaMemcpyAsync(h->d_ids, ids, (size_t)n_seg * sizeof(int32_t), cudaMemcpyHostToDevice, s));
  h->ids_last.assign(ids, ids + n_seg);
  h->ids_stream = s;
  return RIFT_OK;
}

// chunk size in samples: keep the per-chunk workspace near 64 MiB so that it lives in the 126 MB L2
int64_t chunk_samples(const rift_ile *h) {
  const size_t per = coef_bytes(h) + 16 + 4 * (size_t)h->K;
  int64_t n = (int64_t)((64u << 20) / per);
  if (n < 65536) n = 65536;
  return n;
}

bool q_fits_smem(const rift_ile *h) {
  const bool fp32 = h->precision == RIFT_PREC_MIXED;
  return lnl_direct_smem_bytes(h->qs, fp32, true) <= 227u * 1024u;
}


// ---- tensor-core path ------------------------------------------------------------------------------------------------
void make_tc_plan(rift_ile *h, double delta_t) {
  TcPlan &tp = h->tc;
  tp = TcPlan{};
  tp.K = h->K;
  tp.M = h->M;
  tp.n_t = h->n_t;
  tp.nt = (h->n_t + 127) / 128;
  tp.n_tau = h->n_tau;
  tp.j0 = (h->n_t - h->n_tau) / 2;
  tp.n_sub = (h->M + 7) / 8;                        // mode subsets of at most 8 modes, one pass of lnl_tc each
  tp.m_sub = (h->M + tp.n_sub - 1) / tp.n_sub;
  tp.kp = (6 * tp.m_sub + 15) & ~15;
  tp.nch = tp.kp / 8;
  tp.acols = tp.kp / 2;
  tp.H = 0;
  for (int k = 1; k < h->K; ++k) {
    double d2 = 0;
    for (int i = 0; i < 3; ++i) {
      const double d = h->geom.loc[k][i] - h->geom.loc[0][i];
      d2 += d * d;
    }
    const double dm = std::ceil(std::sqrt(d2) / (RIFT_C_LIGHT * delta_t)) + 1.0;
    if (dm > 1e6) return;
    tp.dmax[k] = (int)dm;
    if (tp.dmax[k] > tp.H) tp.H = tp.dmax[k];
  }
  tp.pitch = lnl_tc_pitch(tp.n_t, tp.H);
  tp.blob_words = tp.K * tp.nch * 64 + tp.K * 16 + 16;
  tp.dcol0 = tp.K * tp.nt * tp.acols;
  const bool fits = h->precision == RIFT_PREC_MIXED && tp.nt <= 4 && h->M <= RIFT_MAX_MODES && h->K <= 5 &&
                    (tp.n_sub == 1 || h->n_tau == h->n_t) &&
                    tp.K * tp.nt * (tp.acols + RIFT_TC_NB) <= 512 && tp.H < tp.n_t && tp.pitch > 0 &&
                    lnl_tc_smem_bytes(tp) <= 227u * 1024u;
  tp.ok = fits ? 1 : 0;
  // sorted variant: detector 1 fused by the tensor core (lnl_tcs.cu)
  if (tp.ok && tp.K >= 2) {
    int hs = 0;
    for (int k = 2; k < tp.K; ++k) hs = tp.dmax[k] > hs ? tp.dmax[k] : hs;
    tp.n_bkt = 2 * tp.dmax[1] + 1;
    tp.as_rows = tp.nt * 128 + 2 * tp.dmax[1];
    tp.pitch_s = tp.K > 2 ? lnl_tc_pitch(tp.n_t, hs) : 256;
    tp.blob_words_s = (tp.blob_words + 4 + 31) & ~31;                 // + batch header, stages stay 128-byte aligned
    tp.dcol0_s = (tp.K - 1) * tp.nt * tp.acols;
    tp.srt_ok = (tp.pitch_s > 0 && tp.dmax[1] < tp.n_t && (tp.K - 1) * tp.nt * (tp.acols + RIFT_TC_NB) <= 512 &&
                 tp.as_rows * 16 < (1 << 18) && lnl_tcs_smem_bytes(tp) <= 227u * 1024u)
                    ? 1
                    : 0;
  }
}

// fp64 mode: plan of the DMMA kernel (windows of up to 512 samples).  Whole Q block of a point resident in shared memory when
// it fits beside the exchange buffer, else streamed in (detector, k-step) chunks through a 4- or 3-slot ring.
void make_mma_plan(rift_ile *h, double delta_t) {
  MmaPlan &p = h->mma;
  p = MmaPlan{};
  if (h->precision != RIFT_PREC_FP64) return;
  int halo = 0;
  for (int k = 1; k < h->K; ++k) {
    double d2 = 0;
    for (int i = 0; i < 3; ++i) {
      const double d = h->geom.loc[k][i] - h->geom.loc[0][i];
      d2 += d * d;
    }
    const double dm = std::ceil(std::sqrt(d2) / (RIFT_C_LIGHT * delta_t)) + 1.0;
    if (dm > 1e6) return;
    if ((int)dm > halo) halo = (int)dm;
  }
  // resident with three or two warp groups (three windows must fit beside the Q block), then streamed with the deepest ring that
  // fits (a refill takes about as long as 4 k-steps of tensor work)
  const int cand[][3] = {{0, 0, 3}, {0, 0, 2}, {1, 8, 2}, {1, 8, 1}, {1, 6, 1}, {1, 4, 1}, {1, 3, 1}};   // stream, slots, groups
  for (const auto &c : cand) {
    p = MmaPlan{};
    p.K = h->K;
    p.M = h->M;
    p.n_t = h->n_t;
    p.n_tau = h->n_tau;
    p.H = halo;
    p.stream = c[0];
    p.slots = c[1];
    p.groups = c[2];
    if (lnl_mma_finish_plan(p) && lnl_mma_smem_bytes(p) <= 227u * 1024u) {
      p.ok = 1;
      return;
    }
  }
  p.ok = 0;
}

// mixed mode, circular window: plan of the sky-sorted kernel (any window length; the operand row [Q_hi | Q_lo | Q_hi] of
// 6 M fp16 elements is cut into K pieces of at most 64 elements, one ring slot each)
void make_sky_plan(rift_ile *h, double delta_t) {
  SkyPlan &p = h->sky;
  p = SkyPlan{};
  if (h->precision != RIFT_PREC_MIXED || h->n_tau != h->n_t || h->K > 8) return;
  double dmax = 0;
  for (int k = 1; k < h->K; ++k) {
    double d2 = 0;
    for (int i = 0; i < 3; ++i) {
      const double d = h->geom.loc[k][i] - h->geom.loc[0][i];
      d2 += d * d;
    }
    dmax = std::max(dmax, std::sqrt(d2) / (RIFT_C_LIGHT * delta_t));
  }
  if (dmax > 1e5) return;
  const int dm = (int)std::ceil(dmax) + 1;
  p.K = h->K;
  p.M = h->M;
  p.n_t = h->n_t;
  p.n_pc = (6 * h->M + 63) / 64;
  p.ppp = 2 * ((6 * h->M + 16 * p.n_pc - 1) / (16 * p.n_pc));
  p.kp = 8 * p.n_pc * p.ppp;
  p.rowb = 2 * p.kp;
  p.R0 = ((dm + 7) & ~7) + 8;                       // a chunk starts at the 8-row group holding its first row
  p.n_blocks = (h->n_t + SKY_TBO - 1) / SKY_TBO;
  p.rows_ext = (p.R0 + (p.n_blocks - 1) * SKY_TBO + dm + SKY_TBR + 8 + 7) & ~7;
  p.point_stride = (int64_t)p.K * p.rows_ext * p.rowb;
  if (lnl_sky_smem_bytes(p) > 227u * 1024u) return;
  if (!sky_make_cells(dmax, SKY_E, h->sky_cells)) return;
  p.ok = 1;
}

// fp64 mode, circular window: plan of lnl_sky64 (windows of any length; up to ~10 modes: three 256-row chunks of fp64 rows)
void make_sky64_plan(rift_ile *h, double delta_t) {
  Sky64Plan &p = h->sky64;
  p = Sky64Plan{};
  if (h->precision != RIFT_PREC_FP64 || h->n_tau != h->n_t || h->K > 8) return;
  double dmax = 0;
  for (int k = 1; k < h->K; ++k) {
    double d2 = 0;
    for (int i = 0; i < 3; ++i) {
      const double d = h->geom.loc[k][i] - h->geom.loc[0][i];
      d2 += d * d;
    }
    dmax = std::max(dmax, std::sqrt(d2) / (RIFT_C_LIGHT * delta_t));
  }
  if (dmax > 1e5) return;
  const int dm = (int)std::ceil(dmax) + 1;
  p.K = h->K;
  p.M = h->M;
  p.n_t = h->n_t;
  p.kp = (2 * h->M + 3) & ~3;
  if ((p.kp & 7) == 0) p.kp += 4;                      // rows 32 bytes apart modulo 64: conflict-free fragment loads
  p.KS = p.kp / 4;
  p.R0 = dm + 8;
  p.n_blocks = (h->n_t + 223) / 224;
  p.rows_ext = p.R0 + (p.n_blocks - 1) * 224 + dm + 256 + 8;
  p.point_stride = (int64_t)p.K * p.rows_ext * p.kp * 8;
  for (int slots = 3; slots >= 2; --slots) {
    p.slots = slots;
    if (lnl_sky64_smem_bytes(p) <= 227u * 1024u) {
      p.ok = sky_make_cells(dmax, SKY64_E, h->sky_cells) ? 1 : 0;
      return;
    }
  }
}

// The sky-sorted kernel pays for its padding (about 32 slots per sky cell and segment): AUTO takes it for segments of at
// least 256 samples per cell when the tcgen05 kernels do not apply (windows of more than 512 samples: C4).
bool use_sky(const rift_ile *h, int64_t n_per_seg) {
  if (h->precision == RIFT_PREC_FP64) {
    if (!h->sky64.ok || h->d_Qsky64 == nullptr) return false;
    if (h->kernel_variant == RIFT_KERNEL_SKY) return true;
    return h->kernel_variant == RIFT_KERNEL_AUTO && !h->mma.ok && n_per_seg >= 256 * (int64_t)h->sky_cells.n_cells;
  }
  if (!h->sky.ok || h->d_Qsky == nullptr) return false;
  if (h->kernel_variant == RIFT_KERNEL_SKY) return true;
  return h->kernel_variant == RIFT_KERNEL_AUTO && !h->tc.ok && n_per_seg >= 256 * (int64_t)h->sky_cells.n_cells;
}

bool use_mma(const rift_ile *h) {
  return h->mma.ok && h->d_Qm != nullptr && h->kernel_variant != RIFT_KERNEL_DIRECT;
}

bool use_tc(const rift_ile *h) {
  if (!h->tc.ok || h->d_Qtc == nullptr || h->kernel_variant == RIFT_KERNEL_SKY) return false;
  return h->kernel_variant != RIFT_KERNEL_DIRECT;              // a variant of the other precision mode = AUTO
}

// Sorted variant: worth it when the padding of the shift buckets (about 7.5 slots per bucket and segment) stays small:
// segments of at least 100 samples per bucket (7.5 % padding; the fused kernel gains 24 %)
bool use_tcs(const rift_ile *h, int32_t n_seg, int64_t n_per_seg) {
  if (!h->tc.srt_ok || h->d_Qs == nullptr) return false;
  if (h->kernel_variant == RIFT_KERNEL_TCS) return true;
  const bool auto_on = h->opt_tc_sort != 0;                              // RIFT_OPT_TC_SORT = 0: never pick it automatically
  // small calls are launch-bound and the bucketing adds five launches (C0: 0.10 -> 0.125 ms)
  return auto_on && h->kernel_variant == RIFT_KERNEL_AUTO && n_per_seg >= 100 * (int64_t)h->tc.n_bkt &&
         (int64_t)n_seg * n_per_seg >= 32768;
}

int ensure_tc_workspace(rift_ile *h, int64_t n_batches, int blob_words = 0) {
  if (blob_words < h->tc.blob_words) blob_words = h->tc.blob_words;
  if (h->tc.srt_ok && blob_words < h->tc.blob_words_s) blob_words = h->tc.blob_words_s;   // one size for both variants
  if (n_batches <= h->tc_cap) return RIFT_OK;
  cudaFree(h->tc_blob);
  cudaFree(h->tc_c);
  cudaFree(h->tc_quad);
  cudaFree(h->tc_part);
  cudaFree(h->tc_xacc);
  h->tc_blob = nullptr;
  h->tc_c = h->tc_quad = nullptr;
  h->tc_part = nullptr;
  h->tc_xacc = nullptr;
  h->tc_cap = 0;
  const size_t slots = (size_t)n_batches * RIFT_TC_NB;
  CU(h, cudaMalloc(&h->tc_blob, (size_t)h->tc.n_sub * n_batches * blob_words * sizeof(float)));
  CU(h, cudaMalloc(&h->tc_c, slots * sizeof(double)));
  CU(h, cudaMalloc(&h->tc_quad, slots * sizeof(double)));
  CU(h, cudaMalloc(&h->tc_part, slots * 4 * sizeof(float2)));
  if (h->tc.n_sub > 1) CU(h, cudaMalloc(&h->tc_xacc, slots * (size_t)h->tc.nt * 128 * sizeof(float)));
  h->tc_cap = n_batches;
  return RIFT_OK;
}

// chunks of whole 16-sample batches.  The per-chunk workspace is at most 4 GiB by default (RIFT_OPT_TC_CHUNK_MIB overrides;
// a call that needs less allocates less): measured on C1, every extra launch of the fused kernel costs ~30 us (tensor-memory
// allocation, A-operand load, pipeline fill, tail), far more than keeping the blobs L2-resident saves (64 MiB chunks: 1.39 ms
// per step, one chunk: 1.24 ms); on C3 (2^24 samples x 6 points) 1 GiB chunks are 103 launches per step and 58.6 ms of lnl_tcs,
// 4 GiB chunks 26 launches and 57.8 ms, 16 GiB chunks 57.6 ms
// sizes the workspace of run_chunks_tc for a call shape (also rift_ile_reserve); *cap_out = batches per chunk
int prepare_tc(rift_ile *h, int32_t n_seg, int64_t n_per_seg, int64_t *cap_out) {
  const int64_t nbps = (n_per_seg + RIFT_TC_NB - 1) / RIFT_TC_NB;
  const int64_t total = (int64_t)n_seg * nbps;
  const size_t per_batch = (size_t)h->tc.n_sub * h->tc.blob_words * 4 + (size_t)RIFT_TC_NB * (16 + 32);
  const int64_t chunk_mib = h->opt_tc_chunk_mib;
  int64_t cap = (int64_t)(((size_t)chunk_mib << 20) / per_batch);
  if (cap < 8 * (int64_t)h->n_sm) cap = 8 * (int64_t)h->n_sm;
  // mode-subset passes stream their window sums through HBM anyway and reload the A operand per launch: larger chunks
  if (h->tc.n_sub > 1 && cap < 65536) cap = 65536;
  *cap_out = cap;
  return ensure_tc_workspace(h, total < cap ? total : cap);
}

int run_chunks_tc(rift_ile *h, int32_t n_seg, int64_t n_per_seg, const double *const params[6], double *lnL_out,
                  int32_t *shift_out, cudaStream_t s) {
  const int64_t nbps = (n_per_seg + RIFT_TC_NB - 1) / RIFT_TC_NB;
  const int64_t total = (int64_t)n_seg * nbps;
  if (total == 0) return RIFT_OK;
  int64_t cap = 0;
  int rc = prepare_tc(h, n_seg, n_per_seg, &cap);
  if (rc != RIFT_OK) return rc;
  for (int64_t gb0 = 0; gb0 < total; gb0 += cap) {
    TcChunk c{};
    c.n_per_seg = n_per_seg;
    c.nbps = nbps;
    c.gb0 = gb0;
    c.n_batches = (total - gb0 < cap) ? total - gb0 : cap;
    c.ids = h->d_ids;
    c.qscale = h->d_qscale;
    c.blob = h->tc_blob;
    c.scale_c = h->tc_c;
    c.quad = h->tc_quad;
    c.part = h->tc_part;
    c.xacc = h->tc_xacc;
    {
      ProfSpan ps(h, 0, s);
      CU(h, launch_geometry_tc(h->geom, h->d_modes, h->tc, c, params, h->d_U, h->d_V, h->qp, shift_out, s));
      ps.end();
    }
    ++h->launches;
    int nl = 0;
    ProfSpan ps(h, 1, s);
    if (h->tc.n_sub == 1) {
      CU(h, launch_lnl_tc(h->tc, h->d_Qtc, c, RIFT_TC_PASS_SINGLE, lnL_out, h->n_sm, s, &nl));
    } else {
      // one pass per mode subset: its own A operand and blobs, window sums handed on through tc_xacc
      const size_t a_words = (size_t)h->P * h->K * h->tc.nt * 128 * h->tc.acols;
      for (int sub = 0; sub < h->tc.n_sub; ++sub) {
        TcChunk cs = c;
        cs.blob = h->tc_blob + (size_t)sub * c.n_batches * h->tc.blob_words;
        const int pass = sub == 0 ? RIFT_TC_PASS_FIRST : (sub == h->tc.n_sub - 1 ? RIFT_TC_PASS_LAST : RIFT_TC_PASS_MIDDLE);
        CU(h, launch_lnl_tc(h->tc, h->d_Qtc + sub * a_words, cs, pass, lnL_out, h->n_sm, s, &nl));
      }
    }
    ps.end();
    h->launches += nl;
  }
  h->kernel_name = h->tc.n_sub == 1 ? "lnl_tc<f16x3>" : "lnl_tc<f16x3,passes>";
  return RIFT_OK;
}

// Sorted tensor-core variant: per chunk, bucket the samples by (segment, d_1), let the geometry kernel write every sample
// into the next free slot of its bucket, run lnl_tcs over the sorted batches and scatter lnL back.
int ensure_i32(rift_ile *h, int32_t **p, int64_t *cap, int64_t need) {
  if (need <= *cap) return RIFT_OK;
  cudaFree(*p);
  *p = nullptr;
  *cap = 0;
  CU(h, cudaMalloc(p, (size_t)need * sizeof(int32_t)));
  *cap = need;
  return RIFT_OK;
}

int prepare_tcs(rift_ile *h, int32_t n_seg, int64_t n_per_seg, int64_t *cap_out) {
  const TcPlan &tp = h->tc;
  const int64_t nbps = (n_per_seg + RIFT_TC_NB - 1) / RIFT_TC_NB;
  const int64_t total = (int64_t)n_seg * nbps;
  const size_t per_batch = (size_t)tp.n_sub * tp.blob_words_s * 4 + (size_t)RIFT_TC_NB * (16 + 32 + 8);
  const int64_t chunk_mib = h->opt_tc_chunk_mib;
  int64_t cap = (int64_t)(((size_t)chunk_mib << 20) / per_batch);
  if (cap < 8 * (int64_t)h->n_sm) cap = 8 * (int64_t)h->n_sm;
  if (tp.n_sub > 1 && cap < 65536) cap = 65536;                              // mode-subset passes: as in run_chunks_tc
  *cap_out = cap;
  const int64_t nb_max = total < cap ? total : cap;
  int64_t lseg_max = nb_max / nbps + 2;
  if (lseg_max > n_seg) lseg_max = n_seg;
  int rc = ensure_tc_workspace(h, nb_max + lseg_max * tp.n_bkt);
  if (rc == RIFT_OK) rc = ensure_i32(h, &h->tcs_key, &h->tcs_key_cap, 2 * nb_max * RIFT_TC_NB);   // keys, positions
  if (rc == RIFT_OK) rc = ensure_i32(h, &h->tcs_perm, &h->tcs_perm_cap, (nb_max + lseg_max * tp.n_bkt) * RIFT_TC_NB);
  if (rc == RIFT_OK) rc = ensure_i32(h, &h->tcs_bkt, &h->tcs_bkt_cap, 2 * lseg_max * tp.n_bkt + lseg_max + 1);
  return rc;
}

int run_chunks_tcs(rift_ile *h, int32_t n_seg, int64_t n_per_seg, const double *const params[6], double *lnL_out,
                   int32_t *shift_out, cudaStream_t s) {
  const TcPlan &tp = h->tc;
  const int64_t nbps = (n_per_seg + RIFT_TC_NB - 1) / RIFT_TC_NB;
  const int64_t total = (int64_t)n_seg * nbps;
  if (total == 0) return RIFT_OK;
  int64_t cap = 0;
  int rc = prepare_tcs(h, n_seg, n_per_seg, &cap);
  if (rc != RIFT_OK) return rc;
  for (int64_t gb0 = 0; gb0 < total; gb0 += cap) {
    TcChunk c{};
    c.n_per_seg = n_per_seg;
    c.nbps = nbps;
    c.gb0 = gb0;
    c.n_batches = (total - gb0 < cap) ? total - gb0 : cap;
    c.ids = h->d_ids;
    c.qscale = h->d_qscale;
    c.blob = h->tc_blob;
    c.scale_c = h->tc_c;
    c.quad = h->tc_quad;
    c.part = h->tc_part;
    c.n_lseg = (int32_t)((gb0 + c.n_batches - 1) / nbps - gb0 / nbps + 1);
    c.cap_sorted = c.n_batches + (int64_t)c.n_lseg * tp.n_bkt;
    const int64_t nbk = (int64_t)c.n_lseg * tp.n_bkt;
    c.key = h->tcs_key;
    c.pos = h->tcs_key + c.n_batches * RIFT_TC_NB;
    c.perm = h->tcs_perm;
    c.count = h->tcs_bkt;
    c.base = h->tcs_bkt + nbk;
    c.seg_begin = h->tcs_bkt + 2 * nbk;
    int nl = 0;
    {
      ProfSpan ps(h, 0, s);
      CU(h, launch_tcs_buckets(h->geom, tp, c, params, s, &nl));
      CU(h, launch_geometry_tc(h->geom, h->d_modes, tp, c, params, h->d_U, h->d_V, h->qp, shift_out, s));
      ++nl;
      ps.end();
    }
    c.xacc = h->tc_xacc;
    ProfSpan ps(h, 1, s);
    if (tp.n_sub == 1) {
      CU(h, launch_lnl_tcs(tp, h->d_Qtc, h->d_Qs, c, RIFT_TC_PASS_SINGLE, lnL_out, h->n_sm, s, &nl));
    } else {
      // one pass per mode subset: its own A operands and blobs ([sub][cap_sorted][blob_words_s]), window sums through tc_xacc
      const size_t a_words = (size_t)h->P * h->K * tp.nt * 128 * tp.acols;
      const size_t as_halfs = (size_t)h->P * (tp.kp >> 3) * tp.as_rows * 8;
      for (int sub = 0; sub < tp.n_sub; ++sub) {
        TcChunk cs = c;
        cs.blob = h->tc_blob + (size_t)sub * c.cap_sorted * tp.blob_words_s;
        const int pass = sub == 0 ? RIFT_TC_PASS_FIRST : (sub == tp.n_sub - 1 ? RIFT_TC_PASS_LAST : RIFT_TC_PASS_MIDDLE);
        CU(h, launch_lnl_tcs(tp, h->d_Qtc + sub * a_words, h->d_Qs + sub * as_halfs, cs, pass, lnL_out, h->n_sm, s, &nl));
      }
    }
    ps.end();
    h->launches += nl;
  }
  h->kernel_name = tp.n_sub == 1 ? "lnl_tcs<f16x3>" : "lnl_tcs<f16x3,passes>";
  return RIFT_OK;
}

// Sky-sorted path: per chunk (whole segments, up to 2^23 samples) bucket the samples by (segment, sky cell), let the geometry
// kernel write every sample into its sorted slot (padding slots are null samples), run lnl_sky over the batches of 64 slots.
int run_chunks_sky(rift_ile *h, int32_t n_seg, int64_t n_per_seg, const double *const params[6], double *lnL_out,
                   int32_t *shift_out, cudaStream_t s) {
  const int64_t total = (int64_t)n_seg * n_per_seg;
  if (total == 0) return RIFT_OK;
  const int n_cells = h->sky_cells.n_cells;
  int64_t cap = (int64_t)1 << 23;
  if (n_per_seg <= cap) cap = (cap / n_per_seg) * n_per_seg;
  const int64_t n_max = total < cap ? total : cap;
  const int64_t lseg_max = n_max / n_per_seg + 2 < n_seg ? n_max / n_per_seg + 2 : n_seg;
  const int64_t nbk_max = lseg_max * n_cells;
  const int64_t slots_max = ((n_max + nbk_max * (SKY_NB - 1)) + SKY_NB - 1) / SKY_NB * SKY_NB;
  int rc = ensure_workspace(h, slots_max);
  if (rc == RIFT_OK) rc = ensure_i32(h, &h->sky_orig, &h->sky_orig_cap, slots_max);
  if (rc == RIFT_OK) rc = ensure_i32(h, &h->sky_buf, &h->sky_buf_cap, 2 * n_max + 2 * nbk_max + slots_max + 8);
  if (rc != RIFT_OK) return rc;
  for (int64_t g0 = 0; g0 < total; g0 += cap) {
    Batch b;
    b.n_per_seg = n_per_seg;
    b.g0 = g0;
    b.n = (total - g0 < cap) ? total - g0 : cap;
    b.ids = h->d_ids;
    const int n_lseg = (int)((g0 + b.n - 1) / n_per_seg - g0 / n_per_seg + 1);
    const int64_t nbk = (int64_t)n_lseg * n_cells;
    const int64_t slots = ((b.n + nbk * (SKY_NB - 1)) + SKY_NB - 1) / SKY_NB * SKY_NB;
    int32_t *key = h->sky_buf, *pos = key + n_max, *count = pos + n_max, *base = count + nbk_max, *perm = base + nbk_max,
            *n_batches = perm + slots_max;
    int nl = 0;
    Workspace ws = h->ws;
    ws.orig = h->sky_orig;
    {
      ProfSpan ps(h, 0, s);
      CU(h, launch_sky_sort(h->sky_cells, h->geom.gmst, b, params, n_lseg, key, pos, count, base, perm, slots, n_batches, s, &nl));
      Batch bs = b;
      bs.n = slots;                                                // one thread per sorted slot; padding slots return at once
      CU(h, launch_geometry(h->geom, h->d_modes, bs, params, h->d_U, h->d_V, h->qp, h->precision == RIFT_PREC_MIXED, ws, shift_out,
                            nullptr, nullptr, perm, s));
      ++nl;
      ps.end();
    }
    {
      ProfSpan ps(h, 1, s);
      if (h->precision == RIFT_PREC_MIXED)
        CU(h, launch_lnl_sky(h->sky, h->d_Qsky, h->d_qscale_sky, b, ws, n_batches, slots / SKY_NB, lnL_out, h->n_sm, s, &nl));
      else
        CU(h, launch_lnl_sky64(h->sky64, h->d_Qsky64, b, ws, n_batches, slots / SKY_NB, lnL_out, h->n_sm, s, &nl));
      ps.end();
    }
    h->launches += nl;
  }
  h->kernel_name = h->precision == RIFT_PREC_MIXED ? "lnl_sky<f16x3>" : "lnl_sky<f64>";
  return RIFT_OK;
}

int ensure_reduce_state(rift_ile *h, int32_t n_seg, int32_t nb) {
  if (h->state_nseg == n_seg && h->state_nbins == nb) return RIFT_OK;
  cudaFree(h->d_state);
  cudaFree(h->d_state_hist);
  h->d_state = nullptr;
  h->d_state_hist = nullptr;
  h->state_nseg = 0;
  h->state_nbins = -1;
  CU(h, cudaMalloc(&h->d_state, sizeof(ReduceState) * n_seg));
  if (nb > 0) CU(h, cudaMalloc(&h->d_state_hist, sizeof(double) * (size_t)n_seg * 6 * nb));
  h->state_nseg = n_seg;
  h->state_nbins = nb;
  return RIFT_OK;
}

int ensure_reduce_buffers(rift_ile *h, int32_t n_seg, int64_t n_per_seg, int32_t nb) {
  const int32_t bps = reduce_blocks_per_seg(n_per_seg, n_seg);
  const size_t need_partial = reduce_partial_doubles(n_seg, bps, nb);
  if (need_partial > h->partial_cap) {
    cudaFree(h->d_partial);
    h->d_partial = nullptr;
    h->partial_cap = 0;
    CU(h, cudaMalloc(&h->d_partial, need_partial * sizeof(double)));
    h->partial_cap = need_partial;
  }
  const size_t need_out = (size_t)n_seg * (4 + 6 * (size_t)nb);
  if (need_out > h->out_cap) {
    cudaFree(h->d_out);
    if (h->h_out) cudaFreeHost(h->h_out);
    h->d_out = nullptr;
    h->h_out = nullptr;
    h->out_cap = 0;
    CU(h, cudaMalloc(&h->d_out, need_out * sizeof(double)));
    CU(h, cudaMallocHost(&h->h_out, need_out * sizeof(double)));
    h->out_cap = need_out;
  }
  return RIFT_OK;
}

int run_chunks(rift_ile *h, int32_t n_seg, int64_t n_per_seg, const double *const params[6], double *lnL_out,
               int32_t *shift_out, double *dbg_F, double *dbg_Y, double *dbg_quad, cudaStream_t s, int dm_nodes = 0) {
  const int64_t total = (int64_t)n_seg * n_per_seg;
  if (total == 0) return RIFT_OK;
  const int64_t cap = chunk_samples(h);
  int rc = ensure_workspace(h, total < cap ? total : cap);
  if (rc != RIFT_OK) return rc;
  const bool fp32 = h->precision == RIFT_PREC_MIXED;
  const bool in_smem = q_fits_smem(h);
  for (int64_t g0 = 0; g0 < total; g0 += cap) {
    Batch b;
    b.n_per_seg = n_per_seg;
    b.g0 = g0;
    b.n = (total - g0 < cap) ? total - g0 : cap;
    b.ids = h->d_ids;
    Workspace ws = h->ws;
    ws.orig = nullptr;
    {
      ProfSpan ps(h, 0, s);
      CU(h, launch_geometry(h->geom, h->d_modes, b, params, h->d_U, h->d_V, h->qp, fp32, ws, shift_out, dbg_F, dbg_Y, nullptr, s));
      ps.end();
    }
    ++h->launches;
    if (dbg_quad) CU(h, cudaMemcpyAsync(dbg_quad + g0, ws.quad, (size_t)b.n * sizeof(double), cudaMemcpyDeviceToDevice, s));
    if (lnL_out) {
      int nl = 0;
      ProfSpan ps(h, 1, s);
      if (dm_nodes > 0) {                                   // distance-marginalised variant of the direct kernel
        const bool fits = lnl_direct_dm_smem_bytes(h->qs, fp32, true, dm_nodes) <= 227u * 1024u;
        const bool ext = !fits && h->d_Qg != nullptr;
        CU(h, launch_lnl_direct_dmarg(ext ? h->qsg : h->qs, fp32, fits, ext, b, ws, h->K, dm_nodes, h->d_dm_nodes,
                                      h->d_dm_nodes + dm_nodes, lnL_out, h->n_sm, s, &nl));
        h->kernel_name = fp32 ? "lnl_direct_dmarg<f32>" : "lnl_direct_dmarg<f64>";
      } else if (!fp32 && use_mma(h)) {
        CU(h, launch_lnl_mma(h->mma, h->d_Qm, b, ws, lnL_out, h->n_sm, s, &nl));
        h->kernel_name = h->mma.stream ? "lnl_mma<f64,stream>" : "lnl_mma<f64,resident>";
      } else if (h->d_Qe != nullptr && fp32) {
        CU(h, launch_lnl_direct_ext(h->qse, fp32, b, ws, h->K, lnL_out, h->n_sm, s, &nl));
        h->kernel_name = "lnl_direct_ext<f32>";
      } else {
        const bool ext = !in_smem && h->d_Qg != nullptr;
        CU(h, launch_lnl_direct(ext ? h->qsg : h->qs, fp32, in_smem, ext, b, ws, h->K, lnL_out, h->n_sm, s, &nl));
        h->kernel_name = fp32 ? (in_smem ? "lnl_direct<f32,smem>" : (ext ? "lnl_direct<f32,global,ext>" : "lnl_direct<f32,global>"))
                              : (in_smem ? "lnl_direct<f64,smem>" : (ext ? "lnl_direct<f64,global,ext>" : "lnl_direct<f64,global>"));
      }
      ps.end();
      h->launches += nl;
    }
  }
  return RIFT_OK;
}

}  // namespace

extern "C" {

const char *rift_ile_strerror(int code) {
  switch (code) {
    case RIFT_OK: return "ok";
    case RIFT_EINVAL: return "invalid argument";
    case RIFT_ENOMEM: return "out of memory";
    case RIFT_ECUDA: return "CUDA error";
    case RIFT_EWINDOW: return "marginalisation window plus delay guard band exceeds the stored Q window";
    case RIFT_ERANGE: return "intrinsic id out of range";
    case RIFT_ESTATE: return "reduce state does not match (n_seg / n_bins changed under merge=1)";
    default: return "unknown error";
  }
}

const char *rift_ile_last_error(const rift_ile_t *h) { return h ? h->err : ""; }
int64_t rift_ile_launch_count(const rift_ile_t *h) { return h ? h->launches : 0; }
const char *rift_ile_kernel_name(const rift_ile_t *h) { return h ? h->kernel_name : "none"; }

int rift_ile_create(const rift_ile_config *cfg, rift_ile_t **out) {
  if (!cfg || !out) return RIFT_EINVAL;
  if (cfg->n_det < 1 || cfg->n_det > RIFT_MAX_DET || !cfg->det_location_m || !cfg->det_response) return RIFT_EINVAL;
  if (cfg->n_modes < 1 || cfg->n_modes > RIFT_MAX_MODES || !cfg->mode_l || !cfg->mode_m) return RIFT_EINVAL;
  if (cfg->n_points < 1 || cfg->n_t < 1 || !(cfg->delta_t > 0.0) || !(cfg->d_ref_mpc > 0.0)) return RIFT_EINVAL;
  if (cfg->n_tau < 1 || cfg->n_tau > cfg->n_t || ((cfg->n_t - cfg->n_tau) & 1)) return RIFT_EINVAL;
  if (!cfg->Q || !cfg->U || !cfg->V) return RIFT_EINVAL;
  if (cfg->input_mem != RIFT_MEM_HOST && cfg->input_mem != RIFT_MEM_DEVICE) return RIFT_EINVAL;
  if (cfg->precision != RIFT_PREC_FP64 && cfg->precision != RIFT_PREC_MIXED) return RIFT_EINVAL;
  if (cfg->q_storage != RIFT_Q_C128 && cfg->q_storage != RIFT_Q_C64) return RIFT_EINVAL;
  if (cfg->precision == RIFT_PREC_FP64 && cfg->q_storage != RIFT_Q_C128) return RIFT_EINVAL;
  if (cfg->precision == RIFT_PREC_MIXED && cfg->q_storage != RIFT_Q_C64) return RIFT_EINVAL;
  if (!std::isfinite(cfg->gmst_rad)) return RIFT_EINVAL;
  int l_max = 0;
  for (int a = 0; a < cfg->n_modes; ++a) {
    const int l = cfg->mode_l[a], m = cfg->mode_m[a];
    if (l < 2 || l > 8 || m < -l || m > l) return RIFT_EINVAL;
    for (int b = 0; b < a; ++b)
      if (cfg->mode_l[b] == l && cfg->mode_m[b] == m) return RIFT_EINVAL;
    if (l > l_max) l_max = l;
  }
  // guard band: S_max = max_k ceil(|r_k| / (c delta_t))
  if (cfg->n_tau < cfg->n_t) {
    int s_max = 0;
    for (int k = 0; k < cfg->n_det; ++k) {
      const double *r = cfg->det_location_m + 3 * k;
      const double d = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]) / (RIFT_C_LIGHT * cfg->delta_t);
      const int s = (int)std::ceil(d);
      if (s > s_max) s_max = s;
    }
    if ((int64_t)cfg->n_tau + 2 * (int64_t)s_max > cfg->n_t) return RIFT_EWINDOW;
  }

  rift_ile *h = new (std::nothrow) rift_ile();
  if (!h) return RIFT_ENOMEM;
  int rc = RIFT_OK;
  auto bail = [&](int code) {
    free_handle(h);
    return code;
  };
#define CUC(call)                                                              \
  do {                                                                         \
    cudaError_t e__ = (call);                                                  \
    if (e__ != cudaSuccess) {                                                  \
      cudaGetLastError();                                                      \
      return bail(e__ == cudaErrorMemoryAllocation ? RIFT_ENOMEM : RIFT_ECUDA); \
    }                                                                          \
  } while (0)

  CUC(cudaGetDevice(&h->device));
  CUC(cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device));
  h->P = cfg->n_points;
  h->K = cfg->n_det;
  h->M = cfg->n_modes;
  h->n_t = cfg->n_t;
  h->n_tp = (cfg->n_t + 1) & ~1;
  h->n_tau = cfg->n_tau;
  h->precision = cfg->precision;
  h->q_storage = cfg->q_storage;
  h->geom.n_det = h->K;
  h->geom.n_modes = h->M;
  h->geom.l_max = l_max;
  h->geom.gmst = cfg->gmst_rad;
  h->geom.delta_t = cfg->delta_t;
  h->geom.d_ref = cfg->d_ref_mpc;
  for (int k = 0; k < h->K; ++k) {
    for (int i = 0; i < 3; ++i) h->geom.loc[k][i] = cfg->det_location_m[3 * k + i];
    for (int i = 0; i < 9; ++i) h->geom.resp[k][i] = cfg->det_response[9 * k + i];
  }
  {
    std::vector<ModeEntry> modes(h->M);
    for (int a = 0; a < h->M; ++a) build_mode(cfg->mode_l[a], cfg->mode_m[a], modes[a]);
    CUC(cudaMalloc(&h->d_modes, sizeof(ModeEntry) * h->M));
    CUC(cudaMemcpy(h->d_modes, modes.data(), sizeof(ModeEntry) * h->M, cudaMemcpyHostToDevice));
  }
  const cudaMemcpyKind kind = cfg->input_mem == RIFT_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
  const size_t uv_bytes = (size_t)h->P * h->K * h->M * h->M * 16;
  CUC(cudaMalloc(&h->d_U, uv_bytes));
  CUC(cudaMalloc(&h->d_V, uv_bytes));
  CUC(cudaMemcpy(h->d_U, cfg->U, uv_bytes, kind));
  CUC(cudaMemcpy(h->d_V, cfg->V, uv_bytes, kind));
  if (h->M > 8) {
    // pair program of the quadratic term (QuadProg, rift_internal.h): entries grouped by matrix and phase exponent
    const int M = h->M;
    int n_max = 0;
    for (int a = 0; a < M; ++a) n_max = std::max(n_max, 2 * std::abs(cfg->mode_m[a]));
    std::vector<uint32_t> ent;
    std::vector<int4> bins;
    auto add_bin = [&](int matrix, int n, int zstep) {
      const int first = (int)ent.size();
      for (int a = 0; a < M; ++a)
        for (int b = a; b < M; ++b) {
          const int ma = cfg->mode_m[a], mb = cfg->mode_m[b];
          if (matrix == 0) {
            if (std::abs(mb - ma) == n) ent.push_back((uint32_t)a | (uint32_t)b << 8 | (mb < ma ? 1u << 17 : 0u));
          } else if (ma + mb == n) {
            ent.push_back((uint32_t)a | (uint32_t)b << 8 | 1u << 16);
          }
        }
      bins.push_back(make_int4(first, (int)ent.size(), matrix, zstep));
    };
    for (int n = 0; n <= n_max; ++n) add_bin(0, n, n == 0 ? 0 : 1);
    for (int n = 0; n <= n_max; ++n) add_bin(1, n, n == 0 ? 0 : 1);
    for (int n = 1; n <= n_max; ++n) add_bin(1, -n, n == 1 ? 2 : 3);
    if (ent.size() <= RIFT_QP_MAX_ENT && bins.size() <= RIFT_QP_MAX_BINS) {
      h->qp.n_entries = (int32_t)ent.size();
      h->qp.n_bins = (int32_t)bins.size();
      for (size_t e = 0; e < ent.size(); ++e) h->qp.ent[e] = make_uint2((ent[e] & 0xffu) * RIFT_QP_AMP_STRIDE, ((ent[e] >> 8) & 0xffu) * RIFT_QP_AMP_STRIDE);
      for (size_t i = 0; i < bins.size(); ++i) {
        h->qp.bin_begin[i] = (uint16_t)bins[i].x;
        h->qp.bin_kind[i] = (uint8_t)(bins[i].z | bins[i].w << 1);
      }
      h->qp.bin_begin[bins.size()] = (uint16_t)ent.size();
      uint32_t *d_ent = nullptr;
      double2 *d_uv = nullptr;
      CUC(cudaMalloc(&d_ent, ent.size() * sizeof(uint32_t)));
      h->qp.ent_full = d_ent;
      CUC(cudaMemcpy(d_ent, ent.data(), ent.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
      CUC(cudaMalloc(&d_uv, (size_t)h->P * ent.size() * h->K * sizeof(double2)));
      h->qp_uv_saved = d_uv;                                 // owned by the handle from here on (free_handle)
      CUC(launch_build_quad_uv(h->qp, h->d_U, h->d_V, h->P, h->K, h->M, d_uv, 0));
      CUC(cudaStreamSynchronize(0));
      h->qp.uv = d_uv;
      h->qp_uv_saved = nullptr;
    }
  }
  {
    const bool fp32 = cfg->q_storage == RIFT_Q_C64;
    const int64_t rows = (int64_t)h->P * h->K * h->M;
    const size_t csz = fp32 ? 8 : 16;
    const size_t src_bytes = (size_t)rows * h->n_t * 16;
    CUC(cudaMalloc(&h->d_Q, (size_t)rows * h->n_tp * csz));
    const double *src = reinterpret_cast<const double *>(cfg->Q);
    void *tmp = nullptr;
    if (cfg->input_mem == RIFT_MEM_HOST) {
      CUC(cudaMalloc(&tmp, src_bytes));
      cudaError_t e = cudaMemcpy(tmp, cfg->Q, src_bytes, cudaMemcpyHostToDevice);
      if (e != cudaSuccess) {
        cudaFree(tmp);
        return bail(RIFT_ECUDA);
      }
      src = reinterpret_cast<const double *>(tmp);
    }
    cudaError_t e = launch_convert_q(src, h->d_Q, rows, h->n_t, h->n_tp, fp32, 0);
    // interleaved, circularly extended copy for the direct_ext kernel, if one point's block fits in shared memory
    {
      const int32_t n_te = (h->n_t + RIFT_EXT + 1) & ~1;
      QStore q0{};                                        // the plain block as lnl_direct would stage it (h->qs is set below)
      q0.km = h->K * h->M;
      q0.point_stride_bytes = (int64_t)h->K * h->M * h->n_tp * csz;
      const bool block_fits = lnl_direct_smem_bytes(q0, fp32, true) <= 227u * 1024u;
      QStore qe{};
      qe.n_t = h->n_t;
      qe.n_tp = n_te;
      qe.n_tau = h->n_tau;
      qe.km = h->K * h->M;
      qe.point_stride_bytes = (int64_t)h->K * h->M * n_te * csz;
      if (e == cudaSuccess && fp32 && lnl_direct_ext_smem_bytes(qe, fp32) <= 227u * 1024u) {   // fp64: measured slower than direct
        e = cudaMalloc(&h->d_Qe, (size_t)h->P * qe.point_stride_bytes);
        if (e == cudaSuccess) e = launch_convert_q_ext(src, h->d_Qe, rows, h->n_t, n_te, fp32, 0);
        qe.data = h->d_Qe;
        h->qse = qe;
        ++h->launches;
      } else if (e == cudaSuccess && !block_fits) {
        e = cudaMalloc(&h->d_Qg, (size_t)h->P * qe.point_stride_bytes);
        if (e == cudaSuccess) e = launch_convert_q_ext(src, h->d_Qg, rows, h->n_t, n_te, fp32, 0);
        qe.data = h->d_Qg;
        h->qsg = qe;
        ++h->launches;
      }
    }
    // Q operand of the fp64 tensor-core kernel.  An allocation failure of this optional layout leaves the variant unavailable.
    make_mma_plan(h, cfg->delta_t);
    if (e == cudaSuccess && h->mma.ok) {
      if (cudaMalloc(&h->d_Qm, (size_t)h->P * h->mma.point_stride) == cudaSuccess) {
        e = launch_convert_q_mma(src, h->d_Qm, h->mma, h->P, 0);
        ++h->launches;
      } else {
        cudaGetLastError();
        h->d_Qm = nullptr;
      }
    }
    // Q operand of the sky-sorted kernel (optional layout: an allocation failure leaves the variant unavailable)
    make_sky_plan(h, cfg->delta_t);
    if (e == cudaSuccess && h->sky.ok) {
      if (cudaMalloc(&h->d_Qsky, (size_t)h->P * h->sky.point_stride) == cudaSuccess &&
          cudaMalloc(&h->d_qscale_sky, sizeof(float) * h->P) == cudaSuccess) {
        e = launch_convert_q_sky(src, h->d_Qsky, h->d_qscale_sky, h->sky, h->P, 0);
        h->launches += 3;
      } else {
        cudaGetLastError();
        cudaFree(h->d_Qsky);
        h->d_Qsky = nullptr;
      }
    }
    make_sky64_plan(h, cfg->delta_t);
    if (e == cudaSuccess && h->sky64.ok) {
      if (cudaMalloc(&h->d_Qsky64, (size_t)h->P * h->sky64.point_stride) == cudaSuccess) {
        e = launch_convert_q_sky64(src, h->d_Qsky64, h->sky64, h->P, 0);
        ++h->launches;
      } else {
        cudaGetLastError();
        h->d_Qsky64 = nullptr;
      }
    }
    // A operand of the tensor-core path (fp16 hi | lo pieces), when the configuration fits tensor memory
    make_tc_plan(h, cfg->delta_t);
    if (e == cudaSuccess && h->tc.ok) {
      const size_t words = (size_t)h->tc.n_sub * h->P * h->K * h->tc.nt * 128 * h->tc.acols;
      e = cudaMalloc(&h->d_Qtc, words * sizeof(uint32_t));
      if (e == cudaSuccess) e = cudaMalloc(&h->d_qscale, sizeof(float) * h->P);
      if (e == cudaSuccess) e = launch_convert_q_tc(src, h->d_Qtc, h->d_qscale, h->tc, h->P, 0);
      h->launches += 3;
      if (e == cudaSuccess && h->tc.srt_ok) {
        e = cudaMalloc(&h->d_Qs, (size_t)h->tc.n_sub * h->P * (h->tc.kp >> 3) * h->tc.as_rows * 8 * sizeof(uint16_t));
        if (e == cudaSuccess) e = launch_convert_q_tcs(src, h->d_Qs, h->d_qscale, h->tc, h->P, 0);
        ++h->launches;
      }
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    cudaFree(tmp);
    if (e != cudaSuccess) return bail(RIFT_ECUDA);
    ++h->launches;
    h->qs.data = h->d_Q;
    h->qs.n_t = h->n_t;
    h->qs.n_tp = h->n_tp;
    h->qs.n_tau = h->n_tau;
    h->qs.km = h->K * h->M;
    h->qs.point_stride_bytes = (int64_t)h->K * h->M * h->n_tp * csz;
  }
#undef CUC
  (void)rc;
  *out = h;
  return RIFT_OK;
}

int rift_ile_destroy(rift_ile_t *h) {
  if (!h) return RIFT_EINVAL;
  DeviceGuard g(h->device);
  free_handle(h);
  return RIFT_OK;
}

int rift_ile_set_kernel(rift_ile_t *h, int32_t variant) {
  if (!h) return RIFT_EINVAL;
  if (variant != RIFT_KERNEL_AUTO && variant != RIFT_KERNEL_DIRECT && variant != RIFT_KERNEL_TC && variant != RIFT_KERNEL_TCS &&
      variant != RIFT_KERNEL_MMA && variant != RIFT_KERNEL_SKY)
    return fail(h, RIFT_EINVAL, "unknown kernel variant");
  h->kernel_variant = variant;
  return RIFT_OK;
}

int rift_ile_set_option(rift_ile_t *h, int32_t option, int64_t value) {
  if (!h) return RIFT_EINVAL;
  switch (option) {
    case RIFT_OPT_TC_CHUNK_MIB:
      if (value < 1 || value > (1 << 20)) return fail(h, RIFT_EINVAL, "RIFT_OPT_TC_CHUNK_MIB out of range");
      h->opt_tc_chunk_mib = value;
      return RIFT_OK;
    case RIFT_OPT_TC_SORT:
      h->opt_tc_sort = value != 0;
      return RIFT_OK;
    case RIFT_OPT_QUAD_PROG:
      if ((value != 0) != (h->opt_quad_prog != 0)) {            // the program's W table is kept while the option is off
        std::swap(h->qp.uv, h->qp_uv_saved);
        h->opt_quad_prog = value != 0;
      }
      return RIFT_OK;
    default:
      return fail(h, RIFT_EINVAL, "unknown option");
  }
}

int rift_ile_reserve(rift_ile_t *h, int32_t n_seg, int64_t n_per_seg, int32_t n_bins) {
  if (!h) return RIFT_EINVAL;
  if (n_seg < 0 || n_seg > 65535 || n_per_seg < 0 || n_bins < 0 || n_bins > 1024) return fail(h, RIFT_EINVAL, "bad size");
  if (n_seg == 0 || n_per_seg == 0) return RIFT_OK;
  DeviceGuard g(h->device);
  if (n_seg > h->ids_cap) {
    cudaFree(h->d_ids);
    h->d_ids = nullptr;
    h->ids_cap = 0;
    h->ids_last.clear();
    CU(h, cudaMalloc(&h->d_ids, (size_t)n_seg * sizeof(int32_t)));
    h->ids_cap = n_seg;
  }
  int rc = RIFT_OK;
  int64_t cap = 0;
  if (use_tc(h) && use_tcs(h, n_seg, n_per_seg)) {
    rc = prepare_tcs(h, n_seg, n_per_seg, &cap);
  } else if (use_tc(h)) {
    rc = prepare_tc(h, n_seg, n_per_seg, &cap);
  } else {
    const int64_t total = (int64_t)n_seg * n_per_seg, c = chunk_samples(h);
    rc = ensure_workspace(h, total < c ? total : c);
  }
  if (rc == RIFT_OK) rc = ensure_reduce_buffers(h, n_seg, n_per_seg, n_bins);
  if (rc == RIFT_OK) rc = ensure_reduce_state(h, n_seg, n_bins);       // a changed shape discards the pooled reduce state
  return rc;
}

static int eval_batch_device(rift_ile *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                             const double *const params[RIFT_N_PARAMS], double *lnL_out, int32_t *shift_out, cudaStream_t s) {
  int rc = upload_ids(h, n_seg, intrinsic_ids, s);
  if (rc != RIFT_OK) return rc;
  if (use_sky(h, n_per_seg)) return run_chunks_sky(h, n_seg, n_per_seg, params, lnL_out, shift_out, s);
  if (use_tc(h) && use_tcs(h, n_seg, n_per_seg)) return run_chunks_tcs(h, n_seg, n_per_seg, params, lnL_out, shift_out, s);
  if (use_tc(h)) return run_chunks_tc(h, n_seg, n_per_seg, params, lnL_out, shift_out, s);
  return run_chunks(h, n_seg, n_per_seg, params, lnL_out, shift_out, nullptr, nullptr, nullptr, s);
}

int rift_ile_eval_batch(rift_ile_t *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                        const double *const params[RIFT_N_PARAMS], double *lnL_out, int32_t *shift_out,
                        void *cuda_stream) {
  if (!h) return RIFT_EINVAL;
  if (n_seg < 0 || n_per_seg < 0) return fail(h, RIFT_EINVAL, "negative size");
  if (n_seg == 0 || n_per_seg == 0) return RIFT_OK;
  if (!intrinsic_ids || !params || !lnL_out) return fail(h, RIFT_EINVAL, "null pointer");
  for (int d = 0; d < RIFT_N_PARAMS; ++d)
    if (!params[d]) return fail(h, RIFT_EINVAL, "null parameter array");
  DeviceGuard g(h->device);
  return eval_batch_device(h, n_seg, intrinsic_ids, n_per_seg, params, lnL_out, shift_out,
                           reinterpret_cast<cudaStream_t>(cuda_stream));
}

int rift_ile_eval_batch_host(rift_ile_t *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                             const double *const params[RIFT_N_PARAMS], const double *ln_weight, double *lnL_out,
                             int32_t n_slices, void *cuda_stream) {
  if (!h) return RIFT_EINVAL;
  if (n_seg < 0 || n_per_seg < 0 || n_slices < 0) return fail(h, RIFT_EINVAL, "negative size");
  if (n_seg == 0 || n_per_seg == 0) return RIFT_OK;
  if (!intrinsic_ids || !params || !lnL_out) return fail(h, RIFT_EINVAL, "null pointer");
  for (int d = 0; d < RIFT_N_PARAMS; ++d)
    if (!params[d]) return fail(h, RIFT_EINVAL, "null parameter array");
  for (int32_t i = 0; i < n_seg; ++i)
    if (intrinsic_ids[i] < 0 || intrinsic_ids[i] >= h->P) return fail(h, RIFT_ERANGE, "intrinsic id outside [0, n_points)");
  DeviceGuard g(h->device);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int64_t total = (int64_t)n_seg * n_per_seg;
  if (total > h->host_cap) {
    if (h->host_cap > 0) CU(h, cudaDeviceSynchronize());         // an earlier call may still read the staging buffers
    cudaFree(h->d_hp);
    cudaFree(h->d_hl);
    h->d_hp = h->d_hl = nullptr;
    h->host_cap = 0;
    CU(h, cudaMalloc(&h->d_hp, (size_t)total * 7 * sizeof(double)));
    CU(h, cudaMalloc(&h->d_hl, (size_t)total * sizeof(double)));
    h->host_cap = total;
  }
  if (!h->s_h2d) CU(h, cudaStreamCreateWithFlags(&h->s_h2d, cudaStreamNonBlocking));
  if (!h->s_d2h) CU(h, cudaStreamCreateWithFlags(&h->s_d2h, cudaStreamNonBlocking));
  int G = n_slices > 0 ? n_slices : 4;                           // measured on C1: 2 / 4 / 8 / 16 slices -> 7.1 / 7.7 / 7.3 / 6.2e8 evals/s
  if (G > n_seg) G = n_seg;
  while ((int)h->host_ev.size() < 2 * G + 2) {
    cudaEvent_t e;
    CU(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    h->host_ev.push_back(e);
  }
  cudaEvent_t ev_start = h->host_ev[2 * G], ev_end = h->host_ev[2 * G + 1];
  h->host_n = total;
  h->host_has_w = ln_weight != nullptr;
  const int64_t cap = h->host_cap;
  // uploads: ordered after whatever the caller's stream still does with the staging buffers of the previous call
  CU(h, cudaEventRecord(ev_start, s));
  CU(h, cudaStreamWaitEvent(h->s_h2d, ev_start, 0));
  CU(h, cudaStreamWaitEvent(h->s_d2h, ev_start, 0));
  for (int gi = 0; gi < G; ++gi) {
    const int64_t a = (int64_t)((int64_t)n_seg * gi / G) * n_per_seg, b = (int64_t)((int64_t)n_seg * (gi + 1) / G) * n_per_seg;
    for (int d = 0; d < RIFT_N_PARAMS; ++d)
      CU(h, cudaMemcpyAsync(h->d_hp + d * cap + a, params[d] + a, (size_t)(b - a) * sizeof(double), cudaMemcpyHostToDevice, h->s_h2d));
    if (ln_weight)
      CU(h, cudaMemcpyAsync(h->d_hp + 6 * cap + a, ln_weight + a, (size_t)(b - a) * sizeof(double), cudaMemcpyHostToDevice, h->s_h2d));
    CU(h, cudaEventRecord(h->host_ev[gi], h->s_h2d));
  }
  // evaluation of slice g on the caller's stream while slice g + 1 uploads and slice g - 1 reads back
  for (int gi = 0; gi < G; ++gi) {
    const int32_t s0 = (int32_t)((int64_t)n_seg * gi / G), s1 = (int32_t)((int64_t)n_seg * (gi + 1) / G);
    const int64_t a = (int64_t)s0 * n_per_seg, b = (int64_t)s1 * n_per_seg;
    const double *p[RIFT_N_PARAMS];
    for (int d = 0; d < RIFT_N_PARAMS; ++d) p[d] = h->d_hp + d * cap + a;
    CU(h, cudaStreamWaitEvent(s, h->host_ev[gi], 0));
    const int rc = eval_batch_device(h, s1 - s0, intrinsic_ids + s0, n_per_seg, p, h->d_hl + a, nullptr, s);
    if (rc != RIFT_OK) return rc;
    CU(h, cudaEventRecord(h->host_ev[G + gi], s));
    CU(h, cudaStreamWaitEvent(h->s_d2h, h->host_ev[G + gi], 0));
    CU(h, cudaMemcpyAsync(lnL_out + a, h->d_hl + a, (size_t)(b - a) * sizeof(double), cudaMemcpyDeviceToHost, h->s_d2h));
  }
  CU(h, cudaEventRecord(ev_end, h->s_d2h));
  CU(h, cudaStreamWaitEvent(s, ev_end, 0));                      // the caller's stream is complete when lnL_out is
  return RIFT_OK;
}

int rift_ile_eval_batch_dmarg(rift_ile_t *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                              const double *const params[5], double d_min_mpc, double d_max_mpc, int32_t n_dist,
                              double *lnL_out, int32_t *shift_out, void *cuda_stream) {
  if (!h) return RIFT_EINVAL;
  if (n_seg < 0 || n_per_seg < 0) return fail(h, RIFT_EINVAL, "negative size");
  if (!(d_min_mpc > 0.0) || !(d_max_mpc > d_min_mpc) || !std::isfinite(d_max_mpc)) return fail(h, RIFT_EINVAL, "distance range");
  if (n_dist < 8 || n_dist > 512 || (n_dist & 7)) return fail(h, RIFT_EINVAL, "n_dist must be a multiple of 8 in [8, 512]");
  if (n_seg == 0 || n_per_seg == 0) return RIFT_OK;
  if (!intrinsic_ids || !params || !lnL_out) return fail(h, RIFT_EINVAL, "null pointer");
  for (int d = 0; d < 5; ++d)
    if (!params[d]) return fail(h, RIFT_EINVAL, "null parameter array");
  DeviceGuard g(h->device);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (h->dm_n != n_dist || h->dm_dmin != d_min_mpc || h->dm_dmax != d_max_mpc) {
    // composite 8-point Gauss-Legendre rule in u = ln D on n_dist / 8 equal panels: c_i = D_ref / D_i and
    // ln W_i, W_i = w_i p(D_i) D_i with the d_L^2 prior p(D) = 3 D^2 / (D_max^3 - D_min^3)
    static const double gx[4] = {0.1834346424956498049, 0.5255324099163289858, 0.7966664774136267396, 0.9602898564975362317};
    static const double gw[4] = {0.3626837833783619830, 0.3137066458778872873, 0.2223810344533744706, 0.1012285362903762591};
    std::vector<double> tab(2 * (size_t)n_dist);
    const int n_panels = n_dist / 8;
    const double u0 = std::log(d_min_mpc), hp = (std::log(d_max_mpc) - u0) / n_panels;
    const double ln_norm = std::log(3.0) - std::log(d_max_mpc * d_max_mpc * d_max_mpc - d_min_mpc * d_min_mpc * d_min_mpc);
    for (int p = 0; p < n_panels; ++p)
      for (int q = 0; q < 8; ++q) {
        const double xi = q < 4 ? -gx[3 - q] : gx[q - 4], wi = q < 4 ? gw[3 - q] : gw[q - 4];
        const double u = u0 + hp * (p + 0.5 * (1.0 + xi));
        tab[8 * p + q] = h->geom.d_ref / std::exp(u);
        tab[n_dist + 8 * p + q] = std::log(0.5 * hp * wi) + ln_norm + 3.0 * u;
      }
    if (h->dm_n != n_dist) {
      cudaFree(h->d_dm_nodes);
      h->d_dm_nodes = nullptr;
      h->dm_n = 0;
      CU(h, cudaMalloc(&h->d_dm_nodes, tab.size() * sizeof(double)));
    }
    CU(h, cudaStreamSynchronize(s));                             // an earlier call on this stream may still read the table
    CU(h, cudaMemcpy(h->d_dm_nodes, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice));
    h->dm_n = n_dist;
    h->dm_dmin = d_min_mpc;
    h->dm_dmax = d_max_mpc;
  }
  const int64_t total = (int64_t)n_seg * n_per_seg;
  if (total > h->dm_dist_cap) {                                  // the geometry kernel runs at D = D_ref: c = 1, q = b
    cudaFree(h->d_dm_dist);
    h->d_dm_dist = nullptr;
    h->dm_dist_cap = 0;
    CU(h, cudaMalloc(&h->d_dm_dist, (size_t)total * sizeof(double)));
    h->dm_dist_cap = total;
    CU(h, launch_fill_f64(h->d_dm_dist, total, h->geom.d_ref, s));
    ++h->launches;
  }
  const double *p6[RIFT_N_PARAMS] = {params[0], params[1], params[2], params[3], params[4], h->d_dm_dist};
  int rc = upload_ids(h, n_seg, intrinsic_ids, s);
  if (rc != RIFT_OK) return rc;
  return run_chunks(h, n_seg, n_per_seg, p6, lnL_out, shift_out, nullptr, nullptr, nullptr, s, n_dist);
}

int rift_ile_staged(rift_ile_t *h, const double *params_dev[RIFT_N_PARAMS], const double **ln_weight_dev,
                    const double **lnL_dev, int64_t *n) {
  if (!h) return RIFT_EINVAL;
  if (h->host_n == 0) return fail(h, RIFT_ESTATE, "no rift_ile_eval_batch_host call has staged anything");
  if (params_dev)
    for (int d = 0; d < RIFT_N_PARAMS; ++d) params_dev[d] = h->d_hp + d * h->host_cap;
  if (ln_weight_dev) *ln_weight_dev = h->host_has_w ? h->d_hp + 6 * h->host_cap : nullptr;
  if (lnL_dev) *lnL_dev = h->d_hl;
  if (n) *n = h->host_n;
  return RIFT_OK;
}

int rift_ile_geometry(rift_ile_t *h, int32_t intrinsic_id, int64_t n, const double *const params[RIFT_N_PARAMS],
                      void *F, void *Y, int32_t *shift, double *quad, void *cuda_stream) {
  if (!h) return RIFT_EINVAL;
  if (n < 0) return fail(h, RIFT_EINVAL, "negative size");
  if (n == 0) return RIFT_OK;
  if (!params) return fail(h, RIFT_EINVAL, "null pointer");
  for (int d = 0; d < RIFT_N_PARAMS; ++d)
    if (!params[d]) return fail(h, RIFT_EINVAL, "null parameter array");
  DeviceGuard g(h->device);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  int rc = upload_ids(h, 1, &intrinsic_id, s);
  if (rc != RIFT_OK) return rc;
  return run_chunks(h, 1, n, params, nullptr, shift, reinterpret_cast<double *>(F), reinterpret_cast<double *>(Y), quad,
                    s);
}

int rift_ile_reduce(rift_ile_t *h, int32_t n_seg, int64_t n_per_seg, const double *lnL, const double *ln_weight,
                    const double *const params[RIFT_N_PARAMS], const double lo[RIFT_N_PARAMS],
                    const double hi[RIFT_N_PARAMS], int32_t n_bins, int32_t merge, double *lnZ, double *rel_err,
                    double *n_eff, double *n_ess, double *hist, void *cuda_stream) {
  if (!h) return RIFT_EINVAL;
  if (n_seg < 1 || n_seg > 65535 || n_per_seg < 0) return fail(h, RIFT_EINVAL, "bad n_seg / n_per_seg");
  if ((n_per_seg > 0 && !lnL) || !lnZ || !rel_err || !n_eff || !n_ess) return fail(h, RIFT_EINVAL, "null pointer");
  const bool want_hist = hist != nullptr;
  if (want_hist) {
    if (!params || !lo || !hi || n_bins < 1 || n_bins > 1024) return fail(h, RIFT_EINVAL, "histogram arguments");
    for (int d = 0; d < RIFT_N_PARAMS; ++d)
      if (!params[d] || !(hi[d] > lo[d])) return fail(h, RIFT_EINVAL, "histogram range / parameter array");
  }
  const int nb = want_hist ? n_bins : 0;
  if (merge && h->state_nseg == 0) merge = 0;      // nothing stored yet: the first accumulate is a reset
  if (merge && (h->state_nseg != n_seg || h->state_nbins != nb))
    return fail(h, RIFT_ESTATE, "merge=1 with a different n_seg / n_bins than the stored state");
  DeviceGuard g(h->device);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);

  if (!merge) {
    const int rc = ensure_reduce_state(h, n_seg, nb);
    if (rc != RIFT_OK) return rc;
  }
  const int32_t bps = reduce_blocks_per_seg(n_per_seg, n_seg);
  const size_t need_out = (size_t)n_seg * (4 + 6 * (size_t)nb);
  {
    const int rc = ensure_reduce_buffers(h, n_seg, n_per_seg, nb);
    if (rc != RIFT_OK) return rc;
  }
  double *d_scalars = h->d_out, *d_hist = h->d_out + 4 * (size_t)n_seg;
  int nl = 0;
  {
    ProfSpan ps(h, 2, s);
    CU(h, launch_reduce(n_seg, n_per_seg, lnL, ln_weight, want_hist ? params : nullptr, lo, hi, nb, merge ? 1 : 0,
                        h->d_state, h->d_state_hist, h->d_partial, bps, d_scalars, d_hist, s, &nl));
    ps.end();
  }
  h->launches += nl;
  CU(h, cudaMemcpyAsync(h->h_out, h->d_out, need_out * sizeof(double), cudaMemcpyDeviceToHost, s));
  CU(h, cudaStreamSynchronize(s));
  memcpy(lnZ, h->h_out, sizeof(double) * n_seg);
  memcpy(rel_err, h->h_out + n_seg, sizeof(double) * n_seg);
  memcpy(n_eff, h->h_out + 2 * (size_t)n_seg, sizeof(double) * n_seg);
  memcpy(n_ess, h->h_out + 3 * (size_t)n_seg, sizeof(double) * n_seg);
  if (want_hist) memcpy(hist, h->h_out + 4 * (size_t)n_seg, sizeof(double) * (size_t)n_seg * 6 * nb);
  return RIFT_OK;
}

int rift_ile_precompute(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_freq, const void *h_modes,
                        const void *data, const double *weight, const double *freq_hz_host, const double *freq_hz, int32_t n_t,
                        double delta_t, void *Q, void *U, void *V, void *cuda_stream) {
  if (n_points < 1 || n_det < 1 || n_det > RIFT_MAX_DET || n_modes < 1 || n_modes > RIFT_MAX_MODES || n_freq < 1 || n_t < 1 ||
      !(delta_t > 0.0))
    return RIFT_EINVAL;
  if (!h_modes || !data || !weight || !freq_hz_host || !freq_hz || !Q || !U || !V) return RIFT_EINVAL;
  // equally spaced bins (the usual case): one exact phase per run of 32 bins, rotations in between
  int equal = n_freq > 1 ? 1 : 0;
  const double df = n_freq > 1 ? (freq_hz_host[n_freq - 1] - freq_hz_host[0]) / (n_freq - 1) : 0.0;
  for (int32_t n = 0; n < n_freq && equal; ++n)
    if (std::fabs(freq_hz_host[n] - (freq_hz_host[0] + n * df)) > 1e-12 * std::fmax(1.0, std::fabs(freq_hz_host[n]))) equal = 0;
  const cudaError_t e = launch_precompute(n_points, n_det, n_modes, n_freq, h_modes, data, weight, freq_hz, equal, df, n_t, delta_t,
                                          Q, U, V, reinterpret_cast<cudaStream_t>(cuda_stream));
  return e == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}

int rift_ile_rho_guess(rift_ile_t *h, double *rho_guess) {
  if (!h) return RIFT_EINVAL;
  if (!rho_guess) return fail(h, RIFT_EINVAL, "null pointer");
  DeviceGuard g(h->device);
  double *d_out = nullptr;
  if (cudaMalloc(&d_out, sizeof(double) * h->P) != cudaSuccess) {
    cudaGetLastError();
    return fail(h, RIFT_ENOMEM, "cudaMalloc failed");
  }
  cudaError_t e = launch_rho_guess(h->qs, h->q_storage == RIFT_Q_C64, h->d_U, h->P, h->K, h->M, d_out, 0);
  ++h->launches;
  if (e == cudaSuccess) e = cudaMemcpy(rho_guess, d_out, sizeof(double) * h->P, cudaMemcpyDeviceToHost);
  cudaFree(d_out);
  if (e != cudaSuccess) return fail(h, RIFT_ECUDA, cudaGetErrorString(e));
  return RIFT_OK;
}

int rift_ile_profile(rift_ile_t *h, int32_t enable) {
  if (!h) return RIFT_EINVAL;
  h->profiling = enable != 0;
  return RIFT_OK;
}

int rift_ile_profile_read(rift_ile_t *h, double ms[4], int64_t launches[4]) {
  if (!h || !ms || !launches) return RIFT_EINVAL;
  DeviceGuard g(h->device);
  for (int i = 0; i < 4; ++i) {
    ms[i] = 0.0;
    launches[i] = 0;
  }
  int rc = RIFT_OK;
  for (auto &sp : h->spans) {
    float t = 0.f;
    cudaError_t e = cudaEventSynchronize(sp.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, sp.a, sp.b);
    if (e == cudaSuccess) {
      ms[sp.kind] += t;
      launches[sp.kind] += (sp.kind == 2) ? 2 : (sp.kind == 3 ? 3 : 1);
    } else {
      rc = fail(h, RIFT_ECUDA, "profile event", e);
    }
    cudaEventDestroy(sp.a);
    cudaEventDestroy(sp.b);
  }
  h->spans.clear();
  return rc;
}

int rift_ile_fma_peak(int32_t fp64, int32_t iters, double *tflops, void *cuda_stream) {
  if (!tflops || iters < 1) return RIFT_EINVAL;
  cudaError_t e = run_fma_peak(fp64, iters, tflops, reinterpret_cast<cudaStream_t>(cuda_stream));
  return e == cudaSuccess ? RIFT_OK : RIFT_ECUDA;
}

}  // extern "C"
