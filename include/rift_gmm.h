/*
 * rift_gmm.h -- C ABI of the Gaussian-mixture adaptive sampler.
 *
 * arXiv 2210.07912 section IV.C.1 and Appendix A (:562-625): the sampling prior of a group
 * of correlated dimensions is a mixture of Gaussians truncated to the rectangular domain,
 *     p_s(x) = sum_k pi_k N(x | mu_k, Sigma_k) / Z_k   on [lo, hi),   Z_k = mass of component k inside the domain   (Eq. (19), G5),
 * refitted every adaptive iteration from the weighted samples by expectation-maximisation (Eq. (A1)-(A7)), optionally merged
 * into the model of the iterations before (Eq. (A8)-(A11)), and sampled by box proposals in the eigenbasis with rejection
 * (Eq. (A12)-(A13)).  One handle = one group of n_dim = 1 or 2 dimensions ("pairwise-correlated"); a sampler over more
 * dimensions holds one handle per group (the groups are independent factors of p_s).  The evidence and its variance are pooled
 * over iterations by rift_ile_reduce(merge = 1) (Eq. (20)-(21)).
 *
 * Readings G1-G6 of DESIGN.md section 14 (weighted EM: r_nk = N_k pi_k / sum_j N_j pi_j, p_nk = w_n r_nk, sum_n w_n = 1;
 * eigenvalues ascending, eigenvectors signed so that their largest component is positive; a draw picks its component once and
 * retries the box proposal up to 64 times; counter-based random numbers u = splitmix64(seed + (c + 1) * 0x9E3779B97F4A7C15)
 * >> 11 scaled by 2^-53 with c = (sample * 64 + try) * 4 + j, j = 0 the component, j = 1 + dim the proposal).
 *
 * All functions return RIFT_OK (0) or a negative rift_ile.h error code.  Device arrays are fp64 on the handle's device.
 */
#ifndef RIFT_GMM_H
#define RIFT_GMM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rift_gmm rift_gmm_t;   /* opaque */

#define RIFT_GMM_MAX_COMP 8
#define RIFT_GMM_MAX_TRIES 64

/* n_dim in {1, 2}, n_comp in 1..RIFT_GMM_MAX_COMP, domain [lo[d], hi[d]) (HOST arrays, hi > lo).  The model starts with equal
 * weights, means spread evenly along the diagonal of the domain and axis-aligned covariances ((hi - lo) / n_comp)^2, trained
 * on 0 samples.  Allocates the handle's reduction buffers (no later call allocates). */
int rift_gmm_create(int32_t n_dim, int32_t n_comp, const double *lo, const double *hi, rift_gmm_t **out);

/* Replace / read the model: mu [n_comp][n_dim], cov [n_comp][n_dim][n_dim] (symmetric positive definite), pi [n_comp] (>= 0,
 * sum 1), n_trained = the number of samples it stands for in Eq. (A9)-(A11).  HOST arrays. */
int rift_gmm_set_model(rift_gmm_t *h, const double *mu, const double *cov, const double *pi, double n_trained);
int rift_gmm_get_model(const rift_gmm_t *h, double *mu, double *cov, double *pi, double *n_trained);

/* Expectation-maximisation on n weighted samples, starting from the handle's model (G3).
 *   x        : HOST array of n_dim DEVICE pointers, each fp64 [n];  ln_w : DEVICE fp64 [n] = ln of the sample weights
 *              (e.g. lnL + ln_weight of the evaluation; NULL = equal weights; -inf = weight 0; NaN is treated as -inf).
 *   n_iter   : at most this many M-steps;  tol : stop when |ln L - ln L_prev| < tol (0 = never);  reg : added to the diagonal
 *              of every Sigma_k (Eq. (A5)).
 *   merge    : 0 = the fitted model replaces the handle's (n_trained = n); 1 = it is matched to the handle's model by the
 *              permutation that minimises Eq. (A8) and merged into it by Eq. (A9)-(A11) with N = n_trained, M = n (a model
 *              trained on 0 samples is replaced).
 *   iters_done, loglik : HOST outputs (may be NULL): M-steps done, ln L of the last E-step.
 * The whole iteration runs on the device (E-step with the M-step's sums, a fixed-order add, the M-step and its convergence and
 * validity tests in a one-thread kernel, the model in device memory); the host reads the state back every 8 iterations and once
 * at the end.  RIFT_ESTATE if every weight is zero, a component empties or a covariance stops being positive definite (the
 * handle's model is then unchanged). */
int rift_gmm_fit(rift_gmm_t *h, int64_t n, const double *const *x, const double *ln_w, int32_t n_iter, double tol, double reg,
                 int32_t merge, int32_t *iters_done, double *loglik, void *cuda_stream);

/* rift_gmm_fit on tempered weights w_n^temper (reading G7; not in the paper, whose sampler is described for weights that
 * already spread over many samples): temper is the largest value in [0, 1], found by 20 bisection steps from [0, 1], whose
 * tempered effective sample size (sum_n w_n^temper)^2 / sum_n w_n^(2 temper) is at least ess_min; 1 if the plain weights
 * already reach it.  A round whose weight sits on a handful of samples (a loud signal seen through a wide proposal) would
 * otherwise collapse the mixture onto those samples.  The evidence stays unbiased whatever p_s is.  ess_min = 0: rift_gmm_fit.
 *   temper_used : HOST output (may be NULL). */
int rift_gmm_fit_tempered(rift_gmm_t *h, int64_t n, const double *const *x, const double *ln_w, double ess_min, int32_t n_iter,
                          double tol, double reg, int32_t merge, double *temper_used, int32_t *iters_done, double *loglik,
                          void *cuda_stream);

/* Draw samples index offset .. offset + n - 1 of stream `seed` from p_s and evaluate ln p_s at them.
 *   x : HOST array of n_dim DEVICE pointers, each fp64 [n];  ln_ps : DEVICE fp64 [n] (may be NULL).
 *   n_failed : HOST output or NULL: draws that found no point of the domain in RIFT_GMM_MAX_TRIES proposals (they are set to
 *              the domain-clipped mean of their component); a non-NULL pointer makes the call synchronise. */
int rift_gmm_draw(rift_gmm_t *h, int64_t n, uint64_t seed, uint64_t offset, double *const *x, double *ln_ps,
                  int64_t *n_failed, void *cuda_stream);

/* ln_ps[i] = ln p_s(x_i), -inf outside the domain.  Asynchronous. */
int rift_gmm_ln_density(rift_gmm_t *h, int64_t n, const double *const *x, double *ln_ps, void *cuda_stream);

/* Z [n_comp] (HOST): the mass of every component inside the domain (exact for n_dim = 1; composite Gauss-Legendre over x_1 of
 * the exact conditional integral over x_2 for n_dim = 2, relative error < 1e-9 for |correlation| <= 0.999). */
int rift_gmm_box_mass(rift_gmm_t *h, double *Z);

/* out[i] = terms[0][i] + ... + terms[n_terms - 1][i] (left to right), 1 <= n_terms <= 8: the log-density of a sampler made of
 * several independent groups (sum of the groups' ln p_s), or the log-weight ln omega_i = lnL_i + ln_weight_i that rift_gmm_fit
 * takes.  terms: HOST array of DEVICE fp64 [n] pointers; out: DEVICE fp64 [n] (may alias a term).  Asynchronous. */
int rift_gmm_add(int64_t n, int32_t n_terms, const double *const *terms, double *out, void *cuda_stream);

int rift_gmm_destroy(rift_gmm_t *h);

#ifdef __cplusplus
}
#endif
#endif /* RIFT_GMM_H */
