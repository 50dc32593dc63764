/*
 * rift_ac.h -- C ABI of the on-device adaptive-cartesian (AC) sampler that feeds rift_ile_eval_batch (SURVEY.md section
 * 8(f), NEXT-1).
 *
 * arXiv 2210.07912 section IV.C.2: the sampling prior is separable,
 * p_s(theta) = prod_k p_{s,k}(theta_k), and its adaptive dimensions are histograms with a fixed number of bins (Eq. (22), :348;
 * n_bins = 100, :350) refreshed from the weighted samples of the recent past; drawing on the GPU removes the host round trip the
 * paper blames for limiting ILE (:338).  The Monte Carlo estimate itself is Eq. (3), :55, computed by rift_ile_reduce from
 * lnL + ln_weight with ln_weight = ln p(theta) - ln p_s(theta).
 *
 * Readings: the histogram is integrand-weighted, optionally tempered and mixed with
 * a uniform floor; draws are inverse-CDF with a counter-based random number per (sample, dimension):
 *   u = splitmix64(seed + (index * n_dim + dim + 1) * 0x9E3779B97F4A7C15) >> 11, scaled by 2^-53.
 *
 * All functions return RIFT_OK (0) or a negative rift_ile.h error code.  Device pointers are fp64 arrays on the handle's
 * device; draw / ln_weight are asynchronous on the given stream, update / get_masses are host-side and synchronous.
 */
#ifndef RIFT_AC_H
#define RIFT_AC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rift_ac rift_ac_t;   /* opaque */

/* n_dim dimensions (1..16) with n_bins bins (1..1024, and 16 n_dim n_bins + 16 n_dim <= 200 KiB: the draw kernel stages the
 * table in shared memory; else RIFT_EINVAL) over [lo[d], hi[d]) (HOST arrays, hi > lo); the bin masses start
 * uniform. */
int rift_ac_create(int32_t n_dim, int32_t n_bins, const double *lo, const double *hi, rift_ac_t **out);

/* Draw samples index offset .. offset + n - 1 of stream `seed`.
 *   x      : HOST array of n_dim DEVICE pointers, each fp64 [n]: x[d][i] in [lo[d], hi[d]).
 *   ln_ps  : DEVICE fp64 [n]: ln p_s(x_i) = sum_d ln(mass of the drawn bin / bin width). */
int rift_ac_draw(rift_ac_t *h, int64_t n, uint64_t seed, uint64_t offset, double *const *x, double *ln_ps,
                 void *cuda_stream);

/* New bin masses from normalised weighted histograms hist (HOST [n_dim][n_bins], e.g. the hist output of
 * rift_ile_reduce computed with the same lo, hi, n_bins):
 *   m'[d][b] = (1 - floor_mix) hist[d][b]^temper / sum_b hist[d][b]^temper + floor_mix / n_bins   (uniform if the sum is 0).
 * 0 <= floor_mix <= 1, temper > 0. */
int rift_ac_update(rift_ac_t *h, const double *hist, double floor_mix, double temper);

/* The same with a per-dimension switch: adapt (HOST [n_dim], or NULL = all) != 0 refreshes the dimension, 0 keeps its current
 * masses -- the "frozen" dimensions of a production run, which adapts the sky for a few rounds and then holds it (:452). */
int rift_ac_update_dims(rift_ac_t *h, const double *hist, double floor_mix, double temper, const int32_t *adapt);

/* Copy the current bin masses to masses (HOST [n_dim][n_bins]). */
int rift_ac_get_masses(const rift_ac_t *h, double *masses);

/* ln_weight[i] = ln p(theta_i) - ln_ps[i] for the six extrinsic parameters of rift_ile_eval_batch with the priors of the
 * synthetic configs (SURVEY.md reading A18): RA, psi, phi_ref uniform on [0, 2 pi), [0, pi), [0, 2 pi); dec ~ cos(dec)/2;
 * iota ~ sin(iota)/2; distance ~ 3 D^2 / (d_max^3 - d_min^3) on [d_min, d_max]; -inf outside the support.
 *   params : HOST array of 6 DEVICE pointers (ra, dec, psi, iota, phi_ref, dist_mpc), fp64 [n]; ln_ps, ln_weight DEVICE [n]. */
int rift_ac_ile_ln_weight(int64_t n, const double *const params[6], double d_min_mpc, double d_max_mpc, const double *ln_ps,
                          double *ln_weight, void *cuda_stream);

int rift_ac_destroy(rift_ac_t *h);

#ifdef __cplusplus
}
#endif
#endif /* RIFT_AC_H */
