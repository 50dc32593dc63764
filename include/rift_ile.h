/*
 * rift_ile.h -- C ABI of the ILE extrinsic-marginalised factored likelihood on one B200 (sm_100a).
 *
 * The operation is the inner evaluation of RIFT's ILE worker (arXiv 2210.07912; citations below are
 * line numbers of /root/reference/PAPER.md, readings "A#/G#" are listed in DESIGN.md section 3):
 *
 *   L(lambda) = int L_full(lambda, theta) p(theta) dtheta                         Eq. (1), :37
 *            ~= (1/N) sum_i L_full(lambda, theta_i) p(theta_i)/p_s(theta_i)        Eq. (3), :55
 *   ln L_full = (D_ref/D) Re sum_k sum_lm (F_k Y_lm)^* Q_{k,lm}(t_k)               Eq. (D2), :763
 *             - (D_ref/D)^2/4 sum_k sum_{lm,l'm'} [ |F_k|^2 Y_lm^* Y_l'm' U_{k,lm,l'm'}
 *                                                   + Re(F_k^2 Y_lm Y_l'm' V_{k,lm,l'm'}) ]   Eq. (D3), :766
 *   with Q, U, V the mode/data inner products of Eq. (D4a-c), :771-776, held fixed per intrinsic
 *   point lambda; Y_lm = -2Y_lm(iota, -phi_ref); F_k = F+ + i Fx; t_k = t_ref + dt_k + tau with dt_k
 *   the geocentre-to-detector delay rounded to the nearest Q sample; the time tau is marginalised
 *   over the window with a logsumexp (App. D.2, :801); n_eff etc. are Eq. (B1)-(B3), :637-646; the
 *   per-parameter sampling weights are the weighted histograms behind Eq. (22), :348.
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.  All functions return
 * RIFT_OK (0) or a negative error code and never throw.  On error, outputs are untouched.
 * Units: radians, seconds, metres, Mpc.  A handle is bound to the CUDA device that is current when
 * it is created and is not thread-safe; distinct handles are independent.
 */
#ifndef RIFT_ILE_H
#define RIFT_ILE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rift_ile rift_ile_t;   /* opaque */

enum {
  RIFT_OK = 0,
  RIFT_EINVAL = -1,   /* bad argument (null pointer, size out of range, duplicate mode, ...) */
  RIFT_ENOMEM = -2,   /* host or device allocation failed */
  RIFT_ECUDA = -3,    /* a CUDA runtime call or kernel launch failed; see rift_ile_last_error */
  RIFT_EWINDOW = -4,  /* n_tau < n_t but n_tau + 2*S_max > n_t (the guard band would wrap) */
  RIFT_ERANGE = -5,   /* intrinsic id outside [0, n_points) */
  RIFT_ESTATE = -6    /* reduce(merge=1) with a different n_seg / n_bins than the stored state */
};

enum { RIFT_PREC_FP64 = 0, RIFT_PREC_MIXED = 1 };   /* arithmetic of the window term (reading A17) */
enum { RIFT_Q_C128 = 0, RIFT_Q_C64 = 1 };           /* storage of Q on the device */
enum { RIFT_MEM_HOST = 0, RIFT_MEM_DEVICE = 1 };    /* where the Q/U/V arrays passed to create live */
enum { RIFT_KERNEL_AUTO = 0, RIFT_KERNEL_DIRECT = 1, RIFT_KERNEL_TC = 2, RIFT_KERNEL_TCS = 3,
       RIFT_KERNEL_MMA = 4, RIFT_KERNEL_SKY = 5 };  /* rift_ile_set_kernel */
enum { RIFT_OPT_TC_CHUNK_MIB = 1,   /* per-chunk workspace of the tensor-core kernels in MiB (default 4096, >= 1) */
       RIFT_OPT_TC_SORT = 2,        /* 1 (default): AUTO may pick the shift-sorted tensor-core kernel; 0: never */
       RIFT_OPT_QUAD_PROG = 3 };    /* 1 (default): quadratic term of > 8 modes by the pair program; 0: plain pair sum */

#define RIFT_MAX_DET 8
#define RIFT_MAX_MODES 80
#define RIFT_N_PARAMS 6   /* ra, dec, psi, iota, phi_ref, dist_mpc -- the extrinsic sample */

typedef struct {
  int32_t n_det;                  /* K, 1..RIFT_MAX_DET */
  const double *det_location_m;   /* host [n_det][3]: Earth-fixed position, metres */
  const double *det_response;     /* host [n_det][3][3]: response tensor D_k = (x x^T - y y^T)/2 */
  double gmst_rad;                /* Greenwich mean sidereal time, one value per handle (reading A16) */
  int32_t n_modes;                /* M, 1..RIFT_MAX_MODES */
  const int32_t *mode_l;          /* host [n_modes], 2 <= l <= 8 */
  const int32_t *mode_m;          /* host [n_modes], |m| <= l, no duplicate (l,m) */
  int32_t n_points;               /* P >= 1 intrinsic points */
  int32_t n_t;                    /* stored Q samples per (point, detector, mode); centre sample (n_t-1)/2 = t_ref */
  double delta_t;                 /* Q sample spacing, seconds (> 0) */
  int32_t n_tau;                  /* marginalisation samples, 1..n_t, n_t - n_tau even; n_tau == n_t: circular (A4) */
  double d_ref_mpc;               /* reference distance D_ref of Eq. (D2)-(D3), > 0 */
  const void *Q;                  /* [P][K][M][n_t] complex128 interleaved; host or device per input_mem */
  const void *U;                  /* [P][K][M][M]   complex128, Hermitian in the mode indices */
  const void *V;                  /* [P][K][M][M]   complex128, symmetric in the mode indices */
  int32_t input_mem;              /* RIFT_MEM_HOST | RIFT_MEM_DEVICE (applies to Q, U, V) */
  int32_t precision;              /* RIFT_PREC_FP64 | RIFT_PREC_MIXED */
  int32_t q_storage;              /* RIFT_Q_C128 | RIFT_Q_C64; FP64 precision requires C128 */
} rift_ile_config;

/* Create a handle: validates cfg, builds the per-mode harmonic tables, copies (and for C64 storage
 * converts) Q/U/V to device memory owned by the handle.  Nothing in cfg is referenced afterwards.
 * Synchronous.  *out is written only on success. */
int rift_ile_create(const rift_ile_config *cfg, rift_ile_t **out);

/* Time-marginalised lnL of every extrinsic sample (steps a1-a7 of DESIGN.md section 1).
 *   n_seg, intrinsic_ids : HOST [n_seg]; segment s uses Q/U/V of point intrinsic_ids[s].
 *   n_per_seg            : samples per segment (>= 0).
 *   params               : HOST array of 6 DEVICE pointers (ra, dec, psi, iota, phi_ref, dist_mpc), each
 *                          fp64 [n_seg*n_per_seg], segment-major.
 *   lnL_out              : DEVICE fp64 [n_seg*n_per_seg]:
 *                            ln[(1/n_tau) sum_j exp(lnL(tau_j))],  tau_j over the window (readings A4, A5).
 *                          dist <= 0 or a NaN parameter gives NaN for that sample only.
 *   shift_out            : DEVICE int32 [n_seg*n_per_seg][n_det] or NULL: s_k = floor(dt_k/delta_t + 1/2) (G4).
 *   cuda_stream          : a cudaStream_t (NULL = legacy default stream).  Asynchronous on that stream.
 * Stream capture: the first call of a given size grows the handle's workspace (cudaMalloc; rift_ile_reserve does it ahead
 * of time) and a new id list is copied to the device; a repeated call with the same sizes, ids and stream issues kernel
 * launches only and may be captured into a CUDA graph (the graph then reads params and writes lnL_out / shift_out at
 * replay).  A captured graph points at the handle's id list and workspaces: it is INVALID after any later call on the
 * handle with other ids, a larger size, another kernel variant or option, rift_ile_reserve, or rift_ile_destroy -- capture
 * again after such a call (nothing detects a stale replay). */
int rift_ile_eval_batch(rift_ile_t *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                        const double *const params[RIFT_N_PARAMS], double *lnL_out, int32_t *shift_out,
                        void *cuda_stream);

/* The same evaluation from HOST buffers (the call a user with host arrays makes): params are 6 HOST arrays (pinned
 * memory makes the copies asynchronous), ln_weight a HOST array or NULL, lnL_out a HOST array.  The batch is cut into
 * n_slices groups of whole segments (0 = 4; at most n_seg): slice g + 1 is uploaded on an internal copy stream and slice
 * g - 1 read back on a second one while slice g is evaluated on cuda_stream; the device copies live in staging buffers
 * owned by the handle (grown by cudaMalloc when a call is larger than any before).  Asynchronous: lnL_out is complete
 * when cuda_stream is (the stream is made to wait for the read-backs).  rift_ile_staged returns the device copies of
 * the last call (params, ln_weight or NULL, lnL, and the sample count), valid until the next eval_batch_host: pass them
 * to rift_ile_reduce for the evidence of the same batch without a second upload.  RIFT_ESTATE if nothing was staged. */
int rift_ile_eval_batch_host(rift_ile_t *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                             const double *const params[RIFT_N_PARAMS], const double *ln_weight, double *lnL_out,
                             int32_t n_slices, void *cuda_stream);
int rift_ile_staged(rift_ile_t *h, const double *params_dev[RIFT_N_PARAMS], const double **ln_weight_dev,
                    const double **lnL_dev, int64_t *n);

/* Distance-marginalised evaluation (SURVEY.md section 8(f) NEXT-2; section IV.C.3, :360-372: "directly marginalize
 * over distance").  The paper prints no formula; reading D1 of DESIGN.md section 12: with c = D_ref/D, Eq. (D2)-(D3) read
 * ln L(tau_j, D) = c x_j - c^2 b (the form of Eq. (D5), :780), and
 *   lnL_out = ln[(1/n_tau) sum_j int_{d_min}^{d_max} p(D) exp(c x_j - c^2 b) dD],  p(D) = 3 D^2/(d_max^3 - d_min^3) (:508),
 * the integral by a composite 8-point Gauss-Legendre rule in ln D with n_dist nodes (a multiple of 8 in [8, 512]; the
 * quadrature error in lnL_out is < 1e-5 with 128 nodes up to rho = 12-20 and with 256 nodes up to rho = 30 --
 * tests/test_dmarg_oracle_pins.py P21, tests/test_gpu_dmarg.py).
 *   params : HOST array of 5 DEVICE pointers (ra, dec, psi, iota, phi_ref), fp64 [n_seg*n_per_seg]; the sample has no
 *            distance.  Everything else as rift_ile_eval_batch.  A NaN parameter gives NaN for that sample only.
 * Runs the direct kernels in either precision mode (the window sums x_j do not depend on D: one contraction, n_dist
 * exponentials per window entry).  Not capturable on its first call of a new (d_min, d_max, n_dist) or a larger size. */
int rift_ile_eval_batch_dmarg(rift_ile_t *h, int32_t n_seg, const int32_t *intrinsic_ids, int64_t n_per_seg,
                              const double *const params[5], double d_min_mpc, double d_max_mpc, int32_t n_dist,
                              double *lnL_out, int32_t *shift_out, void *cuda_stream);

/* Sample-axis reduce (step a8): per segment, with ln omega_i = lnL_i + ln_weight_i,
 *   lnZ = ln[(1/N) sum omega_i]  (Eq. (3));  n_eff = sum omega / max omega  (B1);
 *   n_ess = (sum omega)^2 / sum omega^2  (B2);  rel_err^2 = (N/n_ess - 1)/(N - 1)  (B3, reading A20);
 *   hist[s][d][b] = sum_{i in bin b of parameter d} omega_i / sum omega, b = floor(n_bins (x-lo)/(hi-lo))
 *   clamped to [0, n_bins-1]  (Eq. (22), reading A13).
 *   lnL, ln_weight (NULL = 0), params (NULL or 6 device pointers; needed only for hist) : DEVICE.
 *   lo, hi : HOST [6].  merge = 0 resets the handle's per-segment state, 1 pools this call with the state
 *   left by earlier calls (Eq. (20)-(21)); outputs always describe the pooled state.
 *   lnZ, rel_err, n_eff, n_ess : HOST [n_seg];  hist : HOST [n_seg][6][n_bins] or NULL.
 * Synchronises cuda_stream before returning (host outputs). */
int rift_ile_reduce(rift_ile_t *h, int32_t n_seg, int64_t n_per_seg, const double *lnL, const double *ln_weight,
                    const double *const params[RIFT_N_PARAMS], const double lo[RIFT_N_PARAMS],
                    const double hi[RIFT_N_PARAMS], int32_t n_bins, int32_t merge, double *lnZ, double *rel_err,
                    double *n_eff, double *n_ess, double *hist, void *cuda_stream);

/* Allocation-free variant of the reduce (step a8, Eq. (3) and App. B as above) for callers that cannot call cudaMalloc:
 * code under CUDA-graph capture, tight serving loops, harnesses that forbid it.  No handle, scalar outputs only, no pooling
 * with earlier calls (merge = 0), no histograms; it calls no cudaMalloc / cudaFree / allocating routine and does not
 * synchronise.  Its scratch (per-block partial states, per-segment states) is a file-scope device array of 160 KiB that
 * every GPU loading the library holds until exit; hence the limit n_seg <= RIFT_REDUCE_STATIC_MAX_SEG (RIFT_EINVAL beyond,
 * with the reason in rift_ile_reduce_static_error()).
 *   lnL, ln_weight (NULL = 0) : DEVICE fp64 [n_seg][n_per_seg] on the CURRENT device.
 *   out : DEVICE fp64 [4][n_seg] = lnZ, rel_err, n_eff, n_ess per segment, complete when cuda_stream is.
 * Every call on a device shares the one array (it keeps the last call's contents; nothing in it needs clearing, every slot
 * that is read is written first by the same call): calls that overlap on the GPU (different streams, or graphs replayed
 * concurrently) race -- serialise them.  Results are bit-identical to rift_ile_reduce(merge = 0). */
#define RIFT_REDUCE_STATIC_MAX_SEG 1024
int rift_ile_reduce_static(int32_t n_seg, int64_t n_per_seg, const double *lnL, const double *ln_weight, double *out,
                           void *cuda_stream);
/* Reason of the calling thread's last rift_ile_reduce_static failure ("" after a success). */
const char *rift_ile_reduce_static_error(void);

/* rho_guess of every intrinsic point, Eq. (D7) read as SURVEY.md A14 (the printed ratio is inverted):
 *   (2.3 rho_guess)^2 = sum_k sum_lm max_t |Q_{k,lm}(t)|^2 / |U_{k,lm,lm}|   (terms with U_{k,lm,lm} = 0 left out),
 * the amplitude estimate from which the paper sets the overflow offset O ~ rho_guess^2 / 2 - O(few) (:797) -- this library
 * works with logarithms throughout and needs no offset; the number is for the caller's sampler settings.  Computed on the
 * device from the handle's copies of Q (as stored: complex64 storage gives fp32 accuracy) and U.
 *   rho_guess : HOST [n_points].  Synchronous (allocates and frees a small device buffer). */
int rift_ile_rho_guess(rift_ile_t *h, double *rho_guess);

/* Inspection of the geometry kernel (steps a1-a5) in fp64 for n samples of ONE intrinsic point.
 * All outputs DEVICE, any may be NULL: F [n][n_det] complex128 (F+ + i Fx); Y [n][n_modes] complex128
 * (-2Y_lm(iota,-phi_ref)); shift [n][n_det] int32; quad [n] fp64 (the U/V term of Eq. (D3) including
 * (D_ref/D)^2/4).  Asynchronous on cuda_stream. */
int rift_ile_geometry(rift_ile_t *h, int32_t intrinsic_id, int64_t n, const double *const params[RIFT_N_PARAMS],
                      void *F, void *Y, int32_t *shift, double *quad, void *cuda_stream);

/* The inputs of rift_ile_create from frequency series: the inner products of Eq. (D4a-c)
 * as weighted sums over a caller-supplied list of frequencies (reading E1: with
 * weight = 4 df / S_k(f) over f > 0 these are the one-sided products of BASELINE.json configs[0]; with 2 df / S_k(|f|) over
 * positive and negative f the two-sided Eq. (D4a)):
 *   Q[p][k][a][j] = sum_n weight[k][n] exp(2 pi i f_n t_j) conj(h[p][k][a][n]) data[p][k][n],  t_j = (j - (n_t-1)/2) delta_t
 *   U[p][k][a][b] = sum_n weight[k][n] conj(h[p][k][a][n]) h[p][k][b][n];   V[p][k][a][b] = sum_n weight[k][n] h[..a..] h[..b..]
 * h_modes [P][K][M][n_freq], data [P][K][n_freq] complex128, weight [K][n_freq], freq_hz [n_freq] fp64: DEVICE;
 * freq_hz_host: the same frequencies on the HOST (to recognise an equally spaced grid); Q [P][K][M][n_t], U, V [P][K][M][M]
 * complex128: DEVICE outputs, in the layout rift_ile_create takes with input_mem = RIFT_MEM_DEVICE.  No handle; asynchronous
 * on cuda_stream.  U comes out Hermitian and V symmetric up to rounding (create does not require more). */
int rift_ile_precompute(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_freq, const void *h_modes,
                        const void *data, const double *weight, const double *freq_hz_host, const double *freq_hz, int32_t n_t,
                        double delta_t, void *Q, void *U, void *V, void *cuda_stream);

/* Choose the fused-lnL kernel variant (RIFT_KERNEL_*); AUTO picks per configuration and call size: in mixed precision the
 * tensor-core kernels (TCS, which buckets the samples by the relative shift of detector 1, for calls of >= 32768 samples in
 * segments of >= 100 samples per bucket; else TC) when the configuration fits tensor and shared memory, and for longer
 * windows SKY (samples bucketed by sky cell, time-tiled tensor-core contraction; segments of >= 256 samples per cell); in fp64 mode the
 * FP64 tensor-core kernel (MMA) when the configuration fits; else the direct kernels.  A variant that does not apply to
 * the handle falls back to the AUTO choice.  lnL does not depend on the variant beyond the stated tolerance of the
 * precision mode. */
int rift_ile_set_kernel(rift_ile_t *h, int32_t variant);

/* Tuning options (RIFT_OPT_*), all with defaults; nothing in the library reads the process environment.  Returns
 * RIFT_EINVAL for an unknown option or a value out of range.  Takes effect from the next eval_batch. */
int rift_ile_set_option(rift_ile_t *h, int32_t option, int64_t value);

/* Pre-size every per-call workspace for eval_batch calls of up to n_seg segments x n_per_seg samples (and reduce calls of
 * that shape with n_bins histogram bins, 0 = none), so that those calls allocate nothing (synchronous; cudaMalloc happens
  * here; a changed reduce shape discards the pooled reduce state).  Without it the first call of a given size grows the
 * workspace itself. */
int rift_ile_reserve(rift_ile_t *h, int32_t n_seg, int64_t n_per_seg, int32_t n_bins);

/* Number of kernels launched by this handle since creation (bench.py's gpu_launches), and the name of
 * the fused kernel variant the last eval_batch used. */
int64_t rift_ile_launch_count(const rift_ile_t *h);
const char *rift_ile_kernel_name(const rift_ile_t *h);

/* Per-kernel device timing for bench.py's roofline: while enabled, every geometry / fused-lnL / reduce launch is
 * bracketed by CUDA events on its stream.  rift_ile_profile_read synchronises those events, returns the summed
 * milliseconds and launch counts per kernel family since the last read ([0] geometry, [1] fused lnL, [2] reduce,
 * [3] grouping sort), and clears them. */
int rift_ile_profile(rift_ile_t *h, int32_t enable);
int rift_ile_profile_read(rift_ile_t *h, double ms[4], int64_t launches[4]);

/* Dense FMA-pipe microbenchmark (hard part H7): runs `iters` dependent-free FMA per thread over a grid
 * filling the device and returns achieved TFLOP/s in *tflops.  mode: 0 = FFMA chains, 1 = DFMA chains, 2 = FFMA 7x8
 * register tile (all operands in registers, the operand pattern of the fused kernels), 3 / 4 / 5 = FP64 tensor-core
 * mma.sync m8n8k4 / m16n8k8 / m16n8k16 (8 independent accumulator tiles per warp), 6 = m8n8k4 interleaved with as many
 * independent DFMA per thread (reports the tensor part: do the two share a pipe?), 7 = mma.sync m16n8k16 fp16 -> fp32
 * (the legacy tensor path lnl_sky contracts on). */
int rift_ile_fma_peak(int32_t mode, int32_t iters, double *tflops, void *cuda_stream);

int rift_ile_destroy(rift_ile_t *h);
const char *rift_ile_strerror(int code);
const char *rift_ile_last_error(const rift_ile_t *h);   /* never NULL; "" when no error was recorded */

#ifdef __cplusplus
}
#endif
#endif /* RIFT_ILE_H */
