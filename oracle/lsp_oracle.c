/*
 * lsp_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, two-pass FP64 CPU evaluation of the classic Lomb-Scargle periodogram exactly as
 * arXiv 2105.04006 section 2 defines it (Eq. 1 and Eq. 2), used only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  It shares no source,
 * header, table or helper with the CUDA path under paper_2105_04006_b200/csrc and is never
 * imported, linked or called by it.
 *
 * What it computes, per object and per trial frequency (paper notation; X_j is called y here):
 *
 *   grid   (Listing 1 L152/L163):  df = (f_max - f_min)/N_f,  f_k = f_min + k*df,  k = 0..N_f-1
 *   omega:                       omega = 2*pi*f_k              (f in cycles per unit of t, reading a1)
 *   Eq. 1:                       tan 2*omega*tau = sum_j sin 2*omega*t_j / sum_j cos 2*omega*t_j
 *                                                (atan2 as in Listing 1; the branch is immaterial, reading a5)
 *   Eq. 2:                       P = 1/2 * ( [sum_j y_j cos omega(t_j - tau)]^2 / sum_j cos^2 omega(t_j - tau)
 *                                                          + [sum_j y_j sin omega(t_j - tau)]^2 / sum_j sin^2 omega(t_j - tau) )
 *   best:                 k* = argmax_k P(f_k), lowest k on exact ties, NaN never wins (reading a7);
 *                                                period = 1/f_k*  (cyclic-frequency form of the paper's p = 2*pi/f, reading a1/a8)
 *
 * Two scans over the time series per frequency, exactly as Eq. 1 then Eq. 2 read -- no single-scan
 * refactoring, no blocking, no recurrences.  y is used as given (the paper assumes it is already
 * mean-subtracted; reading a4).
 *
 * Arithmetic: FP64.  To keep this oracle's own error about two orders inside the FP64 GPU tolerance
 * (1e-9 * max P) at omega*t up to ~1e6 rad, the phase is formed in CYCLES with an exact product:
 *   p = f*t,  e = fma(f, t, -p)  (so f*t = p + e exactly),  r = (p - nearbyint(p)) + e,  |r| <= 1/2,
 * libm sin/cos are called on 2*pi*r (resp. 4*pi*r) and the sums are kept in long double.  The
 * `_ld` entry point repeats the same steps entirely in long double (sinl/cosl/fmal/atan2l); tests use it
 * on small inputs to bound this oracle's own rounding error (target <= 1e-11 * max P).
 *
 * Degenerate points (reading a6): N_t = 0 gives P = 0.  A term of Eq. 2 whose denominator is below
 * 1e-12 * N_t is dropped (its numerator vanishes at the same rate).  No BASELINE config reaches these.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): chi^2 reduction of a brute-force
 * least-squares sinusoid fit, time-shift and amplitude-scaling invariance, exact recovery of an on-grid
 * noiseless sinusoid, the N_t = 2 closed form, the even-sampling reduction to the textbook DFT
 * periodogram, scipy.signal.lombscargle (library call), the long-double self-bound, the phase reduction
 * against exact rational arithmetic at f*t ~ 1.8e5 cycles (p11: fractions.Fraction products mod 1), and the
 * object-parallel loop of the batch driver against single-object calls (n_threads = 1).
 * No printed P values exist in the paper, so "parity on paper data" is unpinned;
 * every function below is pinned by the identities listed.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LSP_ORACLE_PI  3.14159265358979323846264338327950288
#define LSP_ORACLE_PIL 3.14159265358979323846264338327950288L

/* f*t reduced to (-1/2, 1/2] cycles without losing the low bits of the product. */
static double phase_cycles(double f, double t)
{
    double p = f * t;
    double e = fma(f, t, -p);
    return (p - nearbyint(p)) + e;
}

/* One (object, frequency) value of Eq. 2, two passes (Eq. 1 then Eq. 2). */
static double lsp_power_one(const double *t, const double *y, int64_t n_t, double f)
{
    if (n_t <= 0) return 0.0;
    /* pass 1 -- Eq. 1 */
    long double s2 = 0.0L, c2 = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) {
        double a2 = 4.0 * LSP_ORACLE_PI * phase_cycles(f, t[j]);      /* 2*omega*t_j mod 4*pi */
        s2 += sin(a2);
        c2 += cos(a2);
    }
    double omega_tau = 0.5 * atan2((double)s2, (double)c2);            /* omega*tau, radians */
    /* pass 2 -- Eq. 2 */
    long double yc = 0.0L, ys = 0.0L, cc = 0.0L, ss = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) {
        double a = 2.0 * LSP_ORACLE_PI * phase_cycles(f, t[j]) - omega_tau;   /* omega*(t_j - tau) */
        double c = cos(a), s = sin(a);
        yc += (long double)y[j] * c;
        ys += (long double)y[j] * s;
        cc += (long double)c * c;
        ss += (long double)s * s;
    }
    const long double floor_den = 1e-12L * (long double)n_t;
    long double p = 0.0L;
    if (cc > floor_den) p += yc * yc / cc;
    if (ss > floor_den) p += ys * ys / ss;
    return (double)(0.5L * p);
}

/* Same steps, all in long double: the "oracle of the oracle" for small inputs. */
static double lsp_power_one_ld(const double *t, const double *y, int64_t n_t, double f)
{
    if (n_t <= 0) return 0.0;
    long double s2 = 0.0L, c2 = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) {
        long double p = (long double)f * (long double)t[j];             /* 53x53 bits: not exact in 64 */
        long double e = fmal((long double)f, (long double)t[j], -p);
        long double r = (p - nearbyintl(p)) + e;
        s2 += sinl(4.0L * LSP_ORACLE_PIL * r);
        c2 += cosl(4.0L * LSP_ORACLE_PIL * r);
    }
    long double omega_tau = 0.5L * atan2l(s2, c2);
    long double yc = 0.0L, ys = 0.0L, cc = 0.0L, ss = 0.0L;
    for (int64_t j = 0; j < n_t; ++j) {
        long double p = (long double)f * (long double)t[j];
        long double e = fmal((long double)f, (long double)t[j], -p);
        long double r = (p - nearbyintl(p)) + e;
        long double a = 2.0L * LSP_ORACLE_PIL * r - omega_tau;
        long double c = cosl(a), s = sinl(a);
        yc += y[j] * c;
        ys += y[j] * s;
        cc += c * c;
        ss += s * s;
    }
    const long double floor_den = 1e-12L * (long double)n_t;
    long double pw = 0.0L;
    if (cc > floor_den) pw += yc * yc / cc;
    if (ss > floor_den) pw += ys * ys / ss;
    return (double)(0.5L * pw);
}

/* Grid of PAPER.md:L53 / Listing 1 L152, L163. */
static double grid_freq(double f_min, double f_max, int64_t n_freq, int64_t k)
{
    double df = (f_max - f_min) / (double)n_freq;
    return f_min + df * (double)k;
}

void lsp_oracle_grid(double f_min, double f_max, int64_t n_freq, int64_t n_k, const int64_t *k_list, double *f_out)
{
    for (int64_t i = 0; i < n_k; ++i)
        f_out[i] = grid_freq(f_min, f_max, n_freq, k_list ? k_list[i] : i);
}

/*
 * Periodogram of a CSR batch on the shared grid, optionally only at the listed grid
 * indices.  power is row-major [n_obj][n_k].  k_list == NULL means k = 0..n_k-1 (pass n_k = n_freq for
 * the whole grid).  use_long_double != 0 selects the all-long-double variant.  n_threads <= 0 means
 * "whatever OpenMP defaults to".  Parallel plan as the paper's LSP-C: over objects
 * with a dynamic schedule for batches, over frequencies with a static schedule for a single object.
 * Returns the number of threads used, or -1 on a bad argument.
 */
int lsp_oracle_periodogram(int64_t n_obj, const int64_t *offsets, const double *t, const double *y,
                           double f_min, double f_max, int64_t n_freq,
                           int64_t n_k, const int64_t *k_list,
                           double *power, int use_long_double, int n_threads)
{
    if (n_obj < 0 || n_freq < 1 || n_k < 0 || !offsets || !(f_max > f_min)) return -1;
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
    double (*one)(const double *, const double *, int64_t, double) = use_long_double ? lsp_power_one_ld : lsp_power_one;
    if (n_obj >= 2 * (int64_t)used) {
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t o = 0; o < n_obj; ++o) {
            const int64_t lo = offsets[o], n_t = offsets[o + 1] - offsets[o];
            for (int64_t i = 0; i < n_k; ++i) {
                double f = grid_freq(f_min, f_max, n_freq, k_list ? k_list[i] : i);
                power[o * n_k + i] = one(t + lo, y + lo, n_t, f);
            }
        }
    } else {
        for (int64_t o = 0; o < n_obj; ++o) {
            const int64_t lo = offsets[o], n_t = offsets[o + 1] - offsets[o];
#pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < n_k; ++i) {
                double f = grid_freq(f_min, f_max, n_freq, k_list ? k_list[i] : i);
                power[o * n_k + i] = one(t + lo, y + lo, n_t, f);
            }
        }
    }
    return used;
}

/*
 * Best period per object from a full periodogram (argmax, then period from the grid
 * index; L105 for batches).  Lowest index wins exact ties, NaN never wins (reading a7).  An object with
 * no finite power (N_f of NaN) or power == NULL rows of length 0 gets index -1, power 0, period NaN.
 * Objects with N_t = 0 (all powers 0 by definition above) also get index -1 / NaN (reading a6).
 */
void lsp_oracle_best(int64_t n_obj, const int64_t *offsets, int64_t n_freq, const double *power,
                     double f_min, double f_max,
                     int64_t *best_index, double *best_power, double *best_period)
{
    for (int64_t o = 0; o < n_obj; ++o) {
        int64_t kb = -1;
        double pb = 0.0;
        if (offsets[o + 1] - offsets[o] > 0) {
            for (int64_t k = 0; k < n_freq; ++k) {
                double p = power[o * n_freq + k];
                if (p != p) continue;                 /* NaN never wins */
                if (kb < 0 || p > pb) { kb = k; pb = p; }
            }
        }
        best_index[o] = kb;
        best_power[o] = (kb < 0) ? 0.0 : pb;
        best_period[o] = (kb < 0) ? NAN : 1.0 / grid_freq(f_min, f_max, n_freq, kb);
    }
}
