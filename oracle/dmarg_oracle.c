/*
 * dmarg_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Oracle of SURVEY.md section 8(f) NEXT-2, distance marginalisation (section IV.C.3, :360-372): "directly
 * marginalize over distance".  The paper prints no formula (it defers to its ref. [85], which is not in this container), so
 * the oracle is the definition written out (reading D1 of DESIGN.md section 12): with c = D_ref/D and Eq. (D2)-(D3) in the form
 * of Eq. (D5), ln L(tau_j, D) = c x_j - c^2 b, where x_j is the window sum of Eq. (D2) WITHOUT its factor
 * D_ref/D and b the bracket of Eq. (D3) WITHOUT its factor (D_ref/D)^2 / 4 -- i.e. x_j - b is ln L(tau_j) at D = D_ref --,
 *
 *   lnL_dm = ln[ (1/N_tau) sum_j  int_{D_min}^{D_max} p(D) exp(c x_j - c^2 b) dD ],
 *   p(D) = (alpha + 1) D^alpha / (D_max^(alpha+1) - D_min^(alpha+1))     (alpha = 2: the d_L^2 prior of PAPER.md:508),
 *
 * the integral by plain composite Gauss-Legendre quadrature: n_panels equal panels in u = ln D, 8 nodes per panel
 * (p(D) dD = p(D) D du).  The caller chooses n_panels: a large value (>= 512) is the converged definition, the value the
 * CUDA path uses gives the rule-for-rule comparison.  Plain loops over (panel, node, tau); two passes (max, then sum).
 *
 * Pins (tests/test_dmarg_oracle_pins.py): P19 closed form in erf for alpha = -2 (p(D) dD proportional to dc) and one tau;
 * P20 scipy.integrate.quad on the same integrand for alpha = 2; P21 convergence in n_panels; P22 the 6-D Monte Carlo
 * evidence of the plain oracle against the 5-D Monte Carlo evidence of this one on the same intrinsic point.
 *
 * Built into liboracle.so together with rift_oracle.c (oracle.py: build()), whose geometry and core routines it calls.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* rift_oracle.c */
void oracle_antenna_one(double ra, double dec, double psi, double gmst, const double *D9, double *F2);
int oracle_swsh_m2(int l, int m, double theta, double phi, double *out2);
void oracle_delay_one(double ra, double dec, double gmst, const double *r3, double delta_t, double *dt, int32_t *s,
                      uint8_t *fragile);
double oracle_lnl_core(int K, int M, int n_t, int n_tau, const double *F_, const double *Y_, double c, const int32_t *shift,
                       const double *Q_, const double *U_, const double *V_, double *lnL_j, double *quad);

/* 8-point Gauss-Legendre rule on [-1, 1] (Abramowitz & Stegun table 25.4) */
static const double GL8_X[8] = {-0.9602898564975363, -0.7966664774136267, -0.5255324099163290, -0.1834346424956498,
                                0.1834346424956498,  0.5255324099163290,  0.7966664774136267,  0.9602898564975363};
static const double GL8_W[8] = {0.1012285362903763, 0.2223810344533745, 0.3137066458778873, 0.3626837833783620,
                                0.3626837833783620, 0.3137066458778873, 0.2223810344533745, 0.1012285362903763};

/* Nodes of the rule: D_i (Mpc) and W_i = w_i p(D_i) D_i (sum_i W_i -> 1).  Arrays of 8 n_panels entries. */
void oracle_dmarg_rule(double d_min, double d_max, double alpha, int n_panels, double *D, double *W) {
    const double u0 = log(d_min), u1 = log(d_max), hp = (u1 - u0) / n_panels;
    double norm;
    if (alpha == -1.0)
        norm = 1.0 / (u1 - u0);
    else
        norm = (alpha + 1.0) / (pow(d_max, alpha + 1.0) - pow(d_min, alpha + 1.0));
    for (int p = 0; p < n_panels; ++p)
        for (int g = 0; g < 8; ++g) {
            const double u = u0 + hp * (p + 0.5 * (1.0 + GL8_X[g]));
            const double d = exp(u);
            D[8 * p + g] = d;
            W[8 * p + g] = 0.5 * hp * GL8_W[g] * norm * pow(d, alpha) * d;
        }
}

/* ln[(1/n_tau) sum_j sum_i W_i exp(c_i x_j - c_i^2 b)] */
double oracle_dmarg_core(int n_tau, const double *x, double b, double d_ref, double d_min, double d_max, double alpha,
                         int n_panels) {
    const int n = 8 * n_panels;
    double *D = (double *)malloc(sizeof(double) * 2 * (size_t)n), *W = D + n;
    oracle_dmarg_rule(d_min, d_max, alpha, n_panels, D, W);
    double mx = -INFINITY;
    int bad = 0;
    for (int i = 0; i < n; ++i) {
        const double c = d_ref / D[i];
        for (int j = 0; j < n_tau; ++j) {
            const double t = log(W[i]) + c * x[j] - c * c * b;
            if (isnan(t)) bad = 1;
            if (t > mx) mx = t;
        }
    }
    double res;
    if (bad) {
        res = NAN;
    } else if (isinf(mx)) {
        res = mx;
    } else {
        double s = 0.0;
        for (int i = 0; i < n; ++i) {
            const double c = d_ref / D[i];
            for (int j = 0; j < n_tau; ++j) s += exp(log(W[i]) + c * x[j] - c * c * b - mx);
        }
        res = mx + log(s) - log((double)n_tau);
    }
    free(D);
    return res;
}

/* Batch over samples of ONE intrinsic point: five arrays [n] (ra, dec, psi, iota, phi_ref).  Geometry exactly as
 * oracle_eval_batch (the same routines); x_j and b from oracle_lnl_core at c = 1 (lnL_j = x_j - b, quad = b). */
int oracle_eval_batch_dmarg(int K, const double *det_location, const double *det_response, double gmst, int M,
                            const int32_t *mode_l, const int32_t *mode_m, int n_t, int n_tau, double delta_t,
                            double d_ref_mpc, const double *Q, const double *U, const double *V, int64_t n,
                            const double *ra, const double *dec, const double *psi, const double *iota,
                            const double *phi_ref, double d_min, double d_max, double alpha, int n_panels, double *lnL,
                            int32_t *shift_out, uint8_t *fragile) {
    if (K < 1 || M < 1 || n_t < 1 || n_tau < 1 || n_tau > n_t || ((n_t - n_tau) & 1)) return -1;
    if (K > 16 || M > 128 || n_panels < 1 || !(d_min > 0.0) || !(d_max > d_min)) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        double F[2 * 16], Y[2 * 128];
        int32_t s[16];
        uint8_t frag = 0;
        for (int k = 0; k < K; ++k) {
            uint8_t fk = 0;
            oracle_antenna_one(ra[i], dec[i], psi[i], gmst, det_response + 9 * k, F + 2 * k);
            oracle_delay_one(ra[i], dec[i], gmst, det_location + 3 * k, delta_t, NULL, &s[k], &fk);
            frag |= fk;
        }
        for (int a = 0; a < M; ++a) oracle_swsh_m2(mode_l[a], mode_m[a], iota[i], -phi_ref[i], Y + 2 * a);
        if (shift_out) memcpy(shift_out + (size_t)i * K, s, sizeof(int32_t) * (size_t)K);
        if (fragile) fragile[i] = frag;
        if (isnan(ra[i]) || isnan(dec[i]) || isnan(psi[i]) || isnan(iota[i]) || isnan(phi_ref[i])) {
            lnL[i] = NAN;
            continue;
        }
        double *x = (double *)malloc(sizeof(double) * (size_t)n_tau), b = 0.0;
        oracle_lnl_core(K, M, n_t, n_tau, F, Y, 1.0, s, Q, U, V, x, &b);
        for (int j = 0; j < n_tau; ++j) x[j] += b;
        lnL[i] = oracle_dmarg_core(n_tau, x, b, d_ref_mpc, d_min, d_max, alpha, n_panels);
        free(x);
    }
    return 0;
}
