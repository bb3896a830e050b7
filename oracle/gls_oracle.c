/*
 * gls_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain CPU definition of the GENERALISED Lomb-Scargle periodogram (floating mean + per-point errors), the paper's second
 * mode ("the latter includes photometric error and floats the mean", section 4.11: "the Astropy
 * generalized LSP algorithm that takes as input the photometric error and floats the mean"; reference L520, Zechmeister &
 * Kuerster 2009).  The paper prints no formula for it; the quantity has a plain definition, so the oracle IS that
 * definition (reading a15): with weights w_j = sigma_j^-2 / sum_i sigma_i^-2,
 *
 *     chi0^2     = sum_j w_j (y_j - ybar)^2,                      ybar = sum_j w_j y_j           (constant model)
 *     chi^2(f)   = min over (a, b, c) of sum_j w_j (y_j - a cos wt_j - b sin wt_j - c)^2,  w = 2 pi f   (sinusoid + offset)
 *     P(f)       = (chi0^2 - chi^2(f)) / chi0^2      in [0, 1]   (ZK09 Eq. 4; Astropy's "standard" normalisation)
 *
 * evaluated literally: per (object, frequency) the 3 x 3 weighted normal equations are formed and solved by Gaussian
 * elimination with partial pivoting, all in long double, and chi^2 is recomputed from the residuals of the fitted model (no
 * closed form, no single-scan refactoring).  The same exact-product phase reduction as lsp_oracle.c keeps the phase error
 * below 1e-16 cycles at f t ~ 1e5.  Shares no source with the CUDA path.
 *
 * Degenerate points: N_t = 0 or chi0^2 = 0 -> P = 0; a pivot below 1e-13 (aliased design matrix, N_t < 3) drops that unknown.
 *
 * Pins (tests/test_oracle_gls_pins.py): numpy lstsq of the same model, ZK09's closed form (Eq. 5) typed independently,
 * invariance to y -> y + const and to sigma -> k sigma, P = 1 for a noiseless sinusoid + offset, reduction to the classic
 * oracle (Eq. 2 / (1/2 sum y^2)) when the weighted means of cos and sin vanish, scipy.signal.lombscargle(weights=,
 * floating_mean=True) by library call.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GLS_PI 3.14159265358979323846264338327950288L

static long double gls_phase_cycles(double f, double t)
{
    double p = f * t;
    double e = fma(f, t, -p);
    return ((long double)p - nearbyintl((long double)p)) + (long double)e;
}

static double gls_power_one(const double *t, const double *y, const double *sigma, int64_t n_t, double f)
{
    if (n_t <= 0) return 0.0;
    long double wsum = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) wsum += 1.0L / ((long double)sigma[j] * (long double)sigma[j]);
    long double ybar = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) ybar += (1.0L / ((long double)sigma[j] * sigma[j]) / wsum) * y[j];
    long double chi0 = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) {
        long double w = 1.0L / ((long double)sigma[j] * sigma[j]) / wsum, d = y[j] - ybar;
        chi0 += w * d * d;
    }
    if (!(chi0 > 0.0L)) return 0.0;
    /* normal equations  M x = r  for the basis (cos, sin, 1) */
    long double M[3][4] = {{0}};
    for (int64_t j = 0; j < n_t; ++j) {
        long double w = 1.0L / ((long double)sigma[j] * sigma[j]) / wsum;
        long double a = 2.0L * GLS_PI * gls_phase_cycles(f, t[j]);
        long double b[3] = {cosl(a), sinl(a), 1.0L};
        for (int r = 0; r < 3; ++r) {
            for (int c = 0; c < 3; ++c) M[r][c] += w * b[r] * b[c];
            M[r][3] += w * b[r] * y[j];
        }
    }
    long double x[3] = {0.0L, 0.0L, 0.0L};
    int used[3] = {0, 0, 0}, prow[3] = {-1, -1, -1};
    for (int c = 0; c < 3; ++c) {              /* elimination with partial pivoting; tiny pivots drop the unknown */
        int best = -1;
        long double bv = 1e-13L;
        for (int r = 0; r < 3; ++r)
            if (!used[r] && fabsl(M[r][c]) > bv) { bv = fabsl(M[r][c]); best = r; }
        if (best < 0) continue;
        used[best] = 1;
        prow[c] = best;
        for (int r = 0; r < 3; ++r) {
            if (r == best) continue;
            long double m = M[r][c] / M[best][c];
            for (int k = 0; k < 4; ++k) M[r][k] -= m * M[best][k];
        }
    }
    for (int c = 0; c < 3; ++c)
        if (prow[c] >= 0) x[c] = M[prow[c]][3] / M[prow[c]][c];
    long double chi = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) {
        long double w = 1.0L / ((long double)sigma[j] * sigma[j]) / wsum;
        long double a = 2.0L * GLS_PI * gls_phase_cycles(f, t[j]);
        long double d = y[j] - (x[0] * cosl(a) + x[1] * sinl(a) + x[2]);
        chi += w * d * d;
    }
    return (double)((chi0 - chi) / chi0);
}

/* CSR batch on the shared half-open grid f_k = f_min + k (f_max - f_min)/N_f; power [n_obj][n_k]. */
int gls_oracle_periodogram(int64_t n_obj, const int64_t *offsets, const double *t, const double *y, const double *sigma,
                           double f_min, double f_max, int64_t n_freq, int64_t n_k, const int64_t *k_list, double *power,
                           int n_threads)
{
    if (n_obj < 0 || n_freq < 1 || n_k < 0 || !offsets || !(f_max > f_min)) return -1;
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
    const double df = (f_max - f_min) / (double)n_freq;
#pragma omp parallel for schedule(dynamic, 16) collapse(2)
    for (int64_t o = 0; o < n_obj; ++o)
        for (int64_t i = 0; i < n_k; ++i) {
            const int64_t lo = offsets[o], n_t = offsets[o + 1] - offsets[o];
            const double f = f_min + df * (double)(k_list ? k_list[i] : i);
            power[o * n_k + i] = gls_power_one(t + lo, y + lo, sigma + lo, n_t, f);
        }
    return used;
}
