/*
 * rift_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the ILE factored-likelihood hot path
 * computes, written from the paper (arXiv 2210.07912; citations are PAPER.md line numbers) and
 * the readings listed in DESIGN.md section 3.  Naive loops over (sample, tau, detector, mode); no
 * blocking, no fusion, no reordering.  OpenMP only across samples.  Shares no code with the CUDA
 * path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * Build:  gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC rift_oracle.c -o liboracle.so -lm
 * (-ffp-contract=off: the integer shift of reading G4 must use individually rounded operations.)
 *
 * Pins (tests/test_oracle_pins.py): P1 harmonics, P2 antenna, P3 delays, P4 Eq. (D1) identity,
 * P5 rho^2/2, P6 distance parabola, P7 time marginal, P8 layout, P9 logsumexp, P10-P11 reduce,
 * P12 direct quadrature.  Not pinned by anything external: the absolute scale conventions of the
 * Q/U/V inputs (they are opaque inputs here) -- see DESIGN.md.
 *
 * Layouts: row-major; complex numbers are interleaved (re, im) doubles.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C_LIGHT 299792458.0
#define ORACLE_PI 3.14159265358979323846264338327950288

typedef double complex cplx;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * a1. Antenna factor F_k = F+ + i Fx (reading G2; F_k of Eq. (D2)-(D3); the
 * paper defers the detector response to its refs [16,17]).
 *   gha = gmst - ra
 *   X = (-cos psi sin gha - sin psi cos gha sin dec, -cos psi cos gha + sin psi sin gha sin dec,  sin psi cos dec)
 *   Y = ( sin psi sin gha - cos psi cos gha sin dec,  sin psi cos gha + cos psi sin gha sin dec,  cos psi cos dec)
 *   F+ = X^T D X - Y^T D Y,   Fx = X^T D Y + Y^T D X
 * ------------------------------------------------------------------------------------------ */
void oracle_antenna_one(double ra, double dec, double psi, double gmst, const double D[9], double F[2]) {
    const double gha = gmst - ra;
    const double X[3] = { -cos(psi) * sin(gha) - sin(psi) * cos(gha) * sin(dec),
                          -cos(psi) * cos(gha) + sin(psi) * sin(gha) * sin(dec),
                           sin(psi) * cos(dec) };
    const double Y[3] = {  sin(psi) * sin(gha) - cos(psi) * cos(gha) * sin(dec),
                           sin(psi) * cos(gha) + cos(psi) * sin(gha) * sin(dec),
                           cos(psi) * cos(dec) };
    double xdx = 0.0, ydy = 0.0, xdy = 0.0, ydx = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            xdx += X[i] * D[3 * i + j] * X[j];
            ydy += Y[i] * D[3 * i + j] * Y[j];
            xdy += X[i] * D[3 * i + j] * Y[j];
            ydx += Y[i] * D[3 * i + j] * X[j];
        }
    F[0] = xdx - ydy;
    F[1] = xdy + ydx;
}

/* ------------------------------------------------------------------------------------------
 * a2. Spin-weight -2 spherical harmonic (reading G3):
 *   -2Y_lm(theta,phi) = sqrt((2l+1)/4pi) e^{i m phi} sum_{k=max(0,m-2)}^{min(l+m,l-2)} (-1)^k
 *      sqrt((l+m)!(l-m)!(l+2)!(l-2)!) / [(l+m-k)! (l-2-k)! k! (k-m+2)!]
 *      cos(theta/2)^{2l+m-2-2k} sin(theta/2)^{2k-m+2}
 * The likelihood uses -2Y_lm(iota, -phi_ref) (BASELINE.json north_star).
 * ------------------------------------------------------------------------------------------ */
static double fact(int n) {
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= (double)i;
    return f;
}

static double ipow(double x, int n) {   /* x^n by repeated multiplication, n >= 0 (0^0 = 1) */
    double r = 1.0;
    for (int i = 0; i < n; ++i) r *= x;
    return r;
}

int oracle_swsh_m2(int l, int m, double theta, double phi, double out[2]) {
    if (l < 2 || m < -l || m > l) return -1;
    const double ch = cos(0.5 * theta), sh = sin(0.5 * theta);
    const int k0 = (m - 2 > 0) ? m - 2 : 0;
    const int k1 = (l + m < l - 2) ? l + m : l - 2;
    const double pref = sqrt(fact(l + m) * fact(l - m) * fact(l + 2) * fact(l - 2));
    double sum = 0.0;
    for (int k = k0; k <= k1; ++k) {
        const double den = fact(l + m - k) * fact(l - 2 - k) * fact(k) * fact(k - m + 2);
        const double term = pref / den * ipow(ch, 2 * l + m - 2 - 2 * k) * ipow(sh, 2 * k - m + 2);
        sum += (k & 1) ? -term : term;
    }
    const double amp = sqrt((2.0 * l + 1.0) / (4.0 * ORACLE_PI)) * sum;
    out[0] = amp * cos(m * phi);
    out[1] = amp * sin(m * phi);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * a3. Geocentre-to-detector delay and integer shift, reading G4 (pinned operation order, every
 * operation individually rounded):
 *   nx = cd*ch; ny = cd*sh; nz = sd; dot = (rx*nx + ry*ny) + rz*nz; dt = -(dot/c); x = dt/delta_t;
 *   s = floor(x + 0.5),   cd = cos(dec), sd = sin(dec), ch = cos(ra-gmst), sh = sin(ra-gmst).
 * t_k of Eq. (D2),(D4a).  fragile != NULL receives 1 when x+0.5 lies within
 * 1e-9 of an integer (a last-ulp difference in sin/cos could flip the shift; hard part H6).
 * ------------------------------------------------------------------------------------------ */
void oracle_delay_one(double ra, double dec, double gmst, const double r[3], double delta_t,
                      double *dt_out, int32_t *shift_out, uint8_t *fragile) {
    const double cd = cos(dec), sd = sin(dec);
    const double ch = cos(ra - gmst), sh = sin(ra - gmst);
    const double nx = cd * ch, ny = cd * sh, nz = sd;
    const double dot = (r[0] * nx + r[1] * ny) + r[2] * nz;
    const double dt = -(dot / ORACLE_C_LIGHT);
    const double x = dt / delta_t;
    const double y = x + 0.5;
    const double fl = floor(y);
    if (dt_out) *dt_out = dt;
    if (shift_out) *shift_out = (int32_t)fl;
    if (fragile) {
        const double frac = y - fl;
        *fragile = (frac < 1e-9 || 1.0 - frac < 1e-9) ? 1 : 0;
    }
}

/* ------------------------------------------------------------------------------------------
 * a4-a7 core for ONE sample, given its coefficients (reading A1
 * of Eq. (D1)-(D3)):
 *   x_j   = Re sum_k sum_lm conj(F_k Y_lm) Q_{k,lm}[(j0 + s_k + j) mod N_t],  j0 = (N_t-N_tau)/2
 *   q     = (c^2/4) sum_k [ |F_k|^2 sum Y*_lm U_{k,lm,l'm'} Y_l'm' + Re(F_k^2 sum Y_lm V_{k,lm,l'm'} Y_l'm') ]
 *   lnL_j = c x_j - q
 * Q[K][M][N_t], U[K][M][M], V[K][M][M] complex; F[K], Y[M] complex; shift[K].
 * Writes lnL_j[N_tau] (may be NULL) and *quad = q.  Returns the time-marginalised value
 *   lnL_tm = ln[(1/N_tau) sum_j exp(lnL_j)]  by a max-subtracted two-pass sum
 * (logsumexp of App. D.2; uniform prior over the window, rectangle rule, reading A5).
 * ------------------------------------------------------------------------------------------ */
static int pmod(long a, long n) {
    long r = a % n;
    return (int)(r < 0 ? r + n : r);
}

double oracle_lnl_core(int K, int M, int n_t, int n_tau, const double *F_, const double *Y_, double c,
                       const int32_t *shift, const double *Q_, const double *U_, const double *V_,
                       double *lnL_j, double *quad) {
    const cplx *F = (const cplx *)F_, *Y = (const cplx *)Y_;
    const cplx *Q = (const cplx *)Q_, *U = (const cplx *)U_, *V = (const cplx *)V_;
    const int j0 = (n_t - n_tau) / 2;

    double q = 0.0;
    for (int k = 0; k < K; ++k) {
        cplx yuy = 0.0, yvy = 0.0;
        for (int a = 0; a < M; ++a)
            for (int b = 0; b < M; ++b) {
                yuy += conj(Y[a]) * U[((size_t)k * M + a) * M + b] * Y[b];
                yvy += Y[a] * V[((size_t)k * M + a) * M + b] * Y[b];
            }
        const double f2 = creal(F[k]) * creal(F[k]) + cimag(F[k]) * cimag(F[k]);
        q += f2 * creal(yuy) + creal(F[k] * F[k] * yvy);
    }
    q *= 0.25 * c * c;
    if (quad) *quad = q;

    double *buf = lnL_j ? lnL_j : (double *)malloc(sizeof(double) * (size_t)n_tau);
    double mx = -INFINITY;
    for (int j = 0; j < n_tau; ++j) {
        cplx acc = 0.0;
        for (int k = 0; k < K; ++k) {
            const int idx = pmod((long)j0 + shift[k] + j, n_t);
            for (int a = 0; a < M; ++a)
                acc += conj(F[k] * Y[a]) * Q[((size_t)k * M + a) * n_t + idx];
        }
        buf[j] = c * creal(acc) - q;
        if (buf[j] > mx) mx = buf[j];
    }
    double res;
    if (isnan(mx)) {
        res = NAN;
    } else if (isinf(mx)) {
        res = mx;                       /* all -inf (or a +inf): the max is the answer */
    } else {
        double s = 0.0;
        int nan_seen = 0;
        for (int j = 0; j < n_tau; ++j) {
            if (isnan(buf[j])) nan_seen = 1;
            s += exp(buf[j] - mx);
        }
        res = nan_seen ? NAN : mx + log(s) - log((double)n_tau);
    }
    if (!lnL_j) free(buf);
    return res;
}

/* logsumexp of a plain vector minus ln n (the time marginal alone; pin P9) */
double oracle_logmeanexp(int n, const double *x) {
    double mx = -INFINITY;
    for (int i = 0; i < n; ++i) {
        if (isnan(x[i])) return NAN;
        if (x[i] > mx) mx = x[i];
    }
    if (isinf(mx)) return mx;
    double s = 0.0;
    for (int i = 0; i < n; ++i) s += exp(x[i] - mx);
    return mx + log(s) - log((double)n);
}

/* ------------------------------------------------------------------------------------------
 * a1-a7 for a batch of samples of ONE intrinsic point.
 * params: six arrays [n]: ra, dec, psi, iota, phi_ref, dist_mpc.
 * Outputs: lnL[n]; shift_out[n][K] (may be NULL); fragile[n] (may be NULL).
 * dist <= 0 or a NaN parameter gives lnL = NaN for that sample only.
 * ------------------------------------------------------------------------------------------ */
int oracle_eval_batch(int K, const double *det_location /*[K][3]*/, const double *det_response /*[K][9]*/,
                      double gmst, int M, const int32_t *mode_l, const int32_t *mode_m,
                      int n_t, int n_tau, double delta_t, double d_ref_mpc,
                      const double *Q, const double *U, const double *V,
                      int64_t n, const double *ra, const double *dec, const double *psi,
                      const double *iota, const double *phi_ref, const double *dist_mpc,
                      double *lnL, int32_t *shift_out, uint8_t *fragile) {
    if (K < 1 || M < 1 || n_t < 1 || n_tau < 1 || n_tau > n_t || ((n_t - n_tau) & 1)) return -1;
    if (K > 16 || M > 128) return -1;
#pragma omp parallel for schedule(dynamic, 64)
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
        const double D = dist_mpc[i];
        if (!(D > 0.0) || isnan(ra[i]) || isnan(dec[i]) || isnan(psi[i]) || isnan(iota[i]) || isnan(phi_ref[i])) {
            lnL[i] = NAN;
            continue;
        }
        const double c = d_ref_mpc / D;
        lnL[i] = oracle_lnl_core(K, M, n_t, n_tau, F, Y, c, s, Q, U, V, NULL, NULL);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * a8. Sample-axis reduce: Eq. (3); (B1)-(B3)
 * PAPER.md:637-646 (reading A20: unbiased variance of the mean); Eq. (22) PAPER.md:348 (reading
 * A13: weighted, normalised 1-D histograms); mergeable state for Eq. (20)-(21) PAPER.md:326-328.
 *
 * State of one segment: m = max_i ln omega_i (ln omega_i = lnL_i + ln w_i), S1 = sum e^{ln omega - m},
 * S2 = sum e^{2(ln omega - m)}, N, H[6][n_bins] = per-bin sums of e^{ln omega - m}.
 *   lnZ = m + ln S1 - ln N;  n_eff = S1 (B1);  n_ess = S1^2/S2 (B2);
 *   rel_err^2 = (N/n_ess - 1)/(N - 1) (B3/A20; 0 when N = 1);  hist = H / S1.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    double m, s1, s2;
    int64_t n;
    int32_t n_bins;
    double *hist;                        /* [6][n_bins] or NULL */
} oracle_reduce_state;

oracle_reduce_state *oracle_reduce_new(int32_t n_bins, int want_hist) {
    oracle_reduce_state *st = (oracle_reduce_state *)calloc(1, sizeof(*st));
    st->m = -INFINITY;
    st->n_bins = n_bins;
    if (want_hist && n_bins > 0) st->hist = (double *)calloc((size_t)6 * n_bins, sizeof(double));
    return st;
}

void oracle_reduce_free(oracle_reduce_state *st) {
    if (st) { free(st->hist); free(st); }
}

static void rescale_state(oracle_reduce_state *st, double new_m) {
    if (st->m == new_m || isinf(st->m)) { st->m = new_m; return; }
    const double f = exp(st->m - new_m);
    st->s1 *= f;
    st->s2 *= f * f;
    if (st->hist)
        for (int i = 0; i < 6 * st->n_bins; ++i) st->hist[i] *= f;
    st->m = new_m;
}

/* accumulate n samples into the state (Eq. (20)-(21): pooling chunk sums is the running mean) */
void oracle_reduce_accumulate(oracle_reduce_state *st, int64_t n, const double *lnL, const double *ln_w,
                              const double *const params[6], const double lo[6], const double hi[6]) {
    double mx = st->m;
    for (int64_t i = 0; i < n; ++i) {
        const double v = lnL[i] + (ln_w ? ln_w[i] : 0.0);
        if (isnan(v)) { mx = NAN; break; }
        if (v > mx) mx = v;
    }
    if (isnan(mx)) { st->m = NAN; st->n += n; return; }
    if (isnan(st->m)) { st->n += n; return; }
    if (mx > st->m) rescale_state(st, mx);
    st->n += n;
    if (isinf(mx)) return;              /* every sample so far has weight 0 */
    for (int64_t i = 0; i < n; ++i) {
        const double v = lnL[i] + (ln_w ? ln_w[i] : 0.0);
        const double w = exp(v - mx);
        st->s1 += w;
        st->s2 += w * w;
        if (st->hist && params)
            for (int d = 0; d < 6; ++d) {
                int b = (int)floor(st->n_bins * (params[d][i] - lo[d]) / (hi[d] - lo[d]));
                if (b < 0) b = 0;
                if (b > st->n_bins - 1) b = st->n_bins - 1;
                st->hist[d * st->n_bins + b] += w;
            }
    }
}

void oracle_reduce_finalize(const oracle_reduce_state *st, double *lnZ, double *rel_err, double *n_eff,
                            double *n_ess, double *hist /*[6][n_bins] or NULL*/) {
    const double N = (double)st->n;
    if (isnan(st->m)) {
        *lnZ = *rel_err = *n_eff = *n_ess = NAN;
    } else if (st->n == 0 || isinf(st->m)) {
        *lnZ = (st->n == 0) ? NAN : st->m;
        *rel_err = NAN; *n_eff = 0.0; *n_ess = 0.0;
    } else {
        *lnZ = st->m + log(st->s1) - log(N);
        *n_eff = st->s1;
        *n_ess = st->s1 * st->s1 / st->s2;
        if (st->n > 1) {
            const double r2 = (N / *n_ess - 1.0) / (N - 1.0);
            *rel_err = sqrt(r2 > 0.0 ? r2 : 0.0);
        } else {
            *rel_err = 0.0;
        }
    }
    if (hist && st->hist)
        for (int i = 0; i < 6 * st->n_bins; ++i)
            hist[i] = (st->s1 > 0.0 && isfinite(st->m)) ? st->hist[i] / st->s1 : 0.0;
}
