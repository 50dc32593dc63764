/*
 * rift_sky.h -- C ABI of the rotated detector-network-frame sky coordinates.
 *
 * arXiv 2210.07912 section III: "a coordinate system for the sky where the nominal north pole
 * corresponds to a vector connecting two of the interferometers": the posterior of a two-detector network lies along lines of
 * constant nominal declination, so an adaptive sampler with separable or pairwise-correlated dimensions resolves it.  The
 * sampler draws (lambda, beta) in this frame; rift_sky_network_to_radec turns them into the (RA, dec) that
 * rift_ile_eval_batch takes.  A rotation preserves solid angle: the isotropic prior is cos(beta) / (4 pi) in either frame.
 *
 * The paper gives no formula; readings F1-F2 of DESIGN.md section 14:
 *   n(ra, dec) = (cos dec cos(ra - gmst), cos dec sin(ra - gmst), sin dec)          Earth-fixed direction, as in step a3
 *   z' = (r_b - r_a) / |r_b - r_a|;  x' = (e_z x z') / |e_z x z'|  (e_x when the baseline is parallel to the Earth's axis e_z);
 *   y' = z' x x';  R = [x' y' z'] (columns);  n = R (cos beta cos lambda, cos beta sin lambda, sin beta).
 *
 * All functions return RIFT_OK (0) or a negative rift_ile.h error code.  The transforms are asynchronous on cuda_stream.
 */
#ifndef RIFT_SKY_H
#define RIFT_SKY_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* R (HOST [9], row-major R[3 i + j] = R_ij) of the frame whose pole points from detector a to detector b; loc_a_m, loc_b_m:
 * HOST [3] Earth-fixed positions in metres.  RIFT_EINVAL if the two coincide. */
int rift_sky_network_frame(const double *loc_a_m, const double *loc_b_m, double *R);

/* ra[i] in [0, 2 pi), dec[i] in [-pi/2, pi/2] of the network coordinates (lambda[i], beta[i]).  R: HOST [9]; the four arrays:
 * DEVICE fp64 [n] (in-place allowed: ra = lambda, dec = beta). */
int rift_sky_network_to_radec(int64_t n, const double *R, double gmst_rad, const double *lambda, const double *beta, double *ra,
                              double *dec, void *cuda_stream);

/* The inverse: lambda[i] in [0, 2 pi), beta[i] of (ra[i], dec[i]). */
int rift_sky_radec_to_network(int64_t n, const double *R, double gmst_rad, const double *ra, const double *dec, double *lambda,
                              double *beta, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* RIFT_SKY_H */
