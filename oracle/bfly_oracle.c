/*
 * bfly_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, float64 CPU statement of what the butterfly-filtering hot path
 * computes: direct time-domain correlation of a data series against chirp
 * templates, quadrature magnitude over the sliding data norm, maximum over lags
 * and its lag, and the thresholded time-frequency count map.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this.  It shares no code with the CUDA path
 * (paper_1802_01685_b200/): no common header, helper, table or constant.
 *
 * Source of the definition.  PAPER.md prints no formula for the template, rho or
 * the map (it describes matched filtering against a bank of ~1 s ascending and
 * descending chirps, PAPER.md:54-62 (sec. 2.1); correlation over a 16-s segment,
 * PAPER.md:70, 120 (sec. 2.2, Fig. 5 caption); thresholded output).
 * The formulas are those of BASELINE.json (north_star; configs[0]: "h(t) =
 * cos/sin(2 pi (f0 t + 1/2 f1 t^2)) for t in [0,1), each unit-L2-normalized ...
 * rho(tau) = sqrt(c^2+s^2)/||x_tau||"), in the readings C1-C12 listed in
 * DESIGN.md ("Readings of the paper") and SURVEY.md section 8(c).
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1 Cauchy-Schwarz,
 * P2 noise-free injection, P3 time reversal, P4 direct vs FFT, P5 scale
 * invariance, P6 DFT special case against numpy.fft, P7 Parseval sum, P8 noise
 * expectation 2/L, P9 matched injection in noise, P10 map by brute force,
 * P11 chunking; PS1-PS6 for the kappa-sigma tails (bfo_sigma*, bfo_tails*); PN1-PN4 for the
 * cubic-phase family, PE1-PE5 for the exponentially settling family, PD1-PD2 for the phase
 * reduction (C4).  Parity unpinned (fixed by DESIGN.md readings only, the paper
 * being silent): the choice of map coordinates (C10: time = start of the matched
 * window, frequency = f0) and the per-chunk hit semantics of streaming (C11).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py).
 * -ffp-contract=off and no -ffast-math: every sum below is evaluated in the order
 * written, in IEEE float64.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BFO_PI 3.14159265358979323846

/* cos and sin of a phase given in CYCLES (reading C4 of DESIGN.md: the phase is defined modulo one
 * turn, so it is reduced modulo 1 before the trigonometric call).  frac = cyc - floor(cyc) is
 * exact in float64; the nearest quarter turn is split off (also exact) so that the values at
 * multiples of a quarter turn are exactly 0 and +-1 -- the template (f0 = fs/2, f1 = 0) then has a
 * sine part that is identically zero, as the definition says, rather than rounding noise of
 * sin(pi k) that a later normalisation would blow up. */
static void bfo_sincos_cycles(double cyc, double *s, double *c)
{
    double frac = cyc - floor(cyc);                  /* in [0, 1) */
    int q = (int)floor(4.0 * frac + 0.5);            /* nearest quarter turn, 0..4 */
    double r = frac - 0.25 * (double)q;              /* in [-1/8, 1/8], exact */
    double s0 = sin(2.0 * BFO_PI * r), c0 = cos(2.0 * BFO_PI * r);
    switch (q & 3) {
        case 0: *s = s0;  *c = c0;  break;
        case 1: *s = c0;  *c = -s0; break;
        case 2: *s = -s0; *c = -c0; break;
        default: *s = -c0; *c = s0; break;
    }
}

/* C1 (BASELINE.json configs[0]): template samples
 *   t_k = k/fs, phi_k = 2 pi (f0 t_k + 1/2 f1 t_k^2), hc[k] = cos phi_k, hs[k] = sin phi_k,
 *   k = 0..L-1; phase zero at the first sample; no window.  The bracket is the phase in cycles. */
void bfo_template(double fs, int L, double f0, double f1, double *hc, double *hs)
{
    for (int k = 0; k < L; ++k) {
        double t = (double)k / fs;
        double cyc = f0 * t + 0.5 * f1 * t * t;
        bfo_sincos_cycles(cyc, &hs[k], &hc[k]);
    }
}

/* N1 (descending chirps that settle
 * towards a late-time plateau; the paper gives no waveform): the cubic-phase family is the chirp
 * with a constant second frequency derivative f2 [Hz/s^2],
 *   f(t) = f0 + f1 t + 1/2 f2 t^2,   phi_k = 2 pi (f0 t_k + 1/2 f1 t_k^2 + 1/6 f2 t_k^3),
 * which represents an exponentially settling chirp f_inf + D exp(-t/tc) over one template by its
 * frequency, slope and curvature at the template's first sample.  f2 = 0 is bfo_template. */
void bfo_template3(double fs, int L, double f0, double f1, double f2, double *hc, double *hs)
{
    if (f2 == 0.0) { bfo_template(fs, L, f0, f1, hc, hs); return; }
    for (int k = 0; k < L; ++k) {
        double t = (double)k / fs;
        double cyc = f0 * t + 0.5 * f1 * t * t + f2 * t * t * t / 6.0;
        bfo_sincos_cycles(cyc, &hs[k], &hc[k]);
    }
}

/* N2 (SURVEY.md section 8(f) rank 4 "exponentially settling descending chirps ... synthesised
 * from 3-4 parameters"; PAPER.md:21-26 (sec. 1, Eq. 1: descending chirps that "reach a late time
 * plateau" f_GW), PAPER.md:60 (Fig. 2, right)): the settling family itself,
 *   f(t) = f_inf + D exp(-t / tc),     phi_k = 2 pi ( f_inf t_k + D tc (1 - exp(-t_k / tc)) ),
 * D = f(0) - f_inf [Hz] (D > 0 descends towards the plateau f_inf), tc > 0 the settling time [s].
 * 1 - exp(-u) is taken as -expm1(-u), which keeps full precision for t << tc. */
void bfo_template_settle(double fs, int L, double f_inf, double D, double tc, double *hc, double *hs)
{
    for (int k = 0; k < L; ++k) {
        double t = (double)k / fs;
        double cyc = f_inf * t + D * tc * (-expm1(-t / tc));
        bfo_sincos_cycles(cyc, &hs[k], &hc[k]);
    }
}

/* One entry for both families: family 0 = (f0, f1, f2) polynomial phase (C1 / N1),
 * family 1 = (f_inf, D, tc) exponentially settling (N2). */
#define BFO_FAMILY_POLY 0
#define BFO_FAMILY_SETTLE 1
void bfo_template_family(int family, double fs, int L, double p0, double p1, double p2, double *hc,
                         double *hs)
{
    if (family == BFO_FAMILY_SETTLE) bfo_template_settle(fs, L, p0, p1, p2, hc, hs);
    else bfo_template3(fs, L, p0, p1, p2, hc, hs);
}

/* C2 ("each unit-L2-normalized", BASELINE.json configs[0]): the L2 norms of the
 * cosine and of the sine template, taken separately. */
void bfo_template_norms(int L, const double *hc, const double *hs, double *nc, double *ns)
{
    double a = 0.0, b = 0.0;
    for (int k = 0; k < L; ++k) {
        a += hc[k] * hc[k];
        b += hs[k] * hs[k];
    }
    *nc = sqrt(a);
    *ns = sqrt(b);
}

/* The literal definition at one (template, lag) (SURVEY.md section 8(c) pseudo-code):
 *   c  = sum_k x[tau+k] hc[k] / nc   (0 if nc == 0)           C2, C4
 *   s  = sum_k x[tau+k] hs[k] / ns   (0 if ns == 0)
 *   n2 = sum_k x[tau+k]^2                                      C6
 *   rho = n2 > 0 ? sqrt(c^2 + s^2) / sqrt(n2) : 0              C6, C7
 * Optionally returns the two normalised components c/||x_tau|| and s/||x_tau||.
 * x is the fp32 input, upcast (C12). */
double bfo_rho_at(const float *x, int64_t n_samples, double fs, int L, double f0, double f1,
                  int64_t tau, double *c_over_norm, double *s_over_norm)
{
    (void)n_samples;
    double *hc = (double *)malloc(sizeof(double) * (size_t)L);
    double *hs = (double *)malloc(sizeof(double) * (size_t)L);
    double nc, ns;
    bfo_template(fs, L, f0, f1, hc, hs);
    bfo_template_norms(L, hc, hs, &nc, &ns);
    double c = 0.0, s = 0.0, n2 = 0.0;
    for (int k = 0; k < L; ++k) {
        double xv = (double)x[tau + k];
        c += xv * hc[k];
        s += xv * hs[k];
        n2 += xv * xv;
    }
    c = (nc > 0.0) ? c / nc : 0.0;
    s = (ns > 0.0) ? s / ns : 0.0;
    double rho = 0.0, cn = 0.0, sn = 0.0;
    if (n2 > 0.0) {
        double nx = sqrt(n2);
        rho = sqrt(c * c + s * s) / nx;
        cn = c / nx;
        sn = s / nx;
    }
    if (c_over_norm) *c_over_norm = cn;
    if (s_over_norm) *s_over_norm = sn;
    free(hc);
    free(hs);
    return rho;
}

/* C6: sliding squared norm n2[tau] = sum_k x[tau+k]^2, each lag summed on its own
 * (no running-sum update), for lag_begin <= tau < lag_end. */
void bfo_sliding_n2(const float *x, int L, int64_t lag_begin, int64_t lag_end, double *n2)
{
#pragma omp parallel for schedule(static)
    for (int64_t tau = lag_begin; tau < lag_end; ++tau) {
        double a = 0.0;
        for (int k = 0; k < L; ++k) {
            double xv = (double)x[tau + k];
            a += xv * xv;
        }
        n2[tau - lag_begin] = a;
    }
}

/* Sums over k for a run of lags at once.  For every lag the sum over k is
 * accumulated in ascending k exactly as in bfo_rho_at (the loops over k and over
 * the lags of the run are interchanged so that the compiler can vectorise across
 * lags; no sum is re-associated; tests check bit-equality with bfo_rho_at). */
#define BFO_RUN 1024
static void bfo_dots_run(const double *restrict xd, int L, const double *restrict hc,
                         const double *restrict hs,
                         int64_t tau0, int n, double *restrict c, double *restrict s)
{
    for (int i = 0; i < n; ++i) { c[i] = 0.0; s[i] = 0.0; }
    for (int k = 0; k < L; ++k) {
        const double a = hc[k], b = hs[k];
        const double *xp = xd + tau0 + k;
        for (int i = 0; i < n; ++i) {
            c[i] += xp[i] * a;
            s[i] += xp[i] * b;
        }
    }
}

/* rho_j(tau) of ONE template for lag_begin <= tau < lag_end (needed for the argmax
 * rule and the pins).  c_out / s_out (optional) receive c/||x_tau||, s/||x_tau||. */
void bfo_rho_series_family(int family, const float *x, int64_t n_samples, double fs, int L,
                           double p0, double p1, double p2, int64_t lag_begin, int64_t lag_end,
                           double *rho, double *c_out, double *s_out);
void bfo_rho_series3(const float *x, int64_t n_samples, double fs, int L, double f0, double f1,
                     double f2, int64_t lag_begin, int64_t lag_end, double *rho, double *c_out,
                     double *s_out)
{
    bfo_rho_series_family(BFO_FAMILY_POLY, x, n_samples, fs, L, f0, f1, f2, lag_begin, lag_end, rho,
                          c_out, s_out);
}
void bfo_rho_series(const float *x, int64_t n_samples, double fs, int L, double f0, double f1,
                    int64_t lag_begin, int64_t lag_end, double *rho, double *c_out, double *s_out)
{
    bfo_rho_series3(x, n_samples, fs, L, f0, f1, 0.0, lag_begin, lag_end, rho, c_out, s_out);
}

/* The same for a template of either family (N1: p = (f0, f1, f2); N2: p = (f_inf, D, tc)). */
void bfo_rho_series_family(int family, const float *x, int64_t n_samples, double fs, int L,
                           double p0, double p1, double p2, int64_t lag_begin, int64_t lag_end,
                           double *rho, double *c_out, double *s_out)
{
    double *xd = (double *)malloc(sizeof(double) * (size_t)n_samples);
    for (int64_t i = 0; i < n_samples; ++i) xd[i] = (double)x[i];
    double *hc = (double *)malloc(sizeof(double) * (size_t)L);
    double *hs = (double *)malloc(sizeof(double) * (size_t)L);
    double nc, ns;
    bfo_template_family(family, fs, L, p0, p1, p2, hc, hs);
    bfo_template_norms(L, hc, hs, &nc, &ns);
    double c[BFO_RUN], s[BFO_RUN];
    for (int64_t tau0 = lag_begin; tau0 < lag_end; tau0 += BFO_RUN) {
        int n = (int)((lag_end - tau0 < BFO_RUN) ? (lag_end - tau0) : BFO_RUN);
        bfo_dots_run(xd, L, hc, hs, tau0, n, c, s);
        for (int i = 0; i < n; ++i) {
            double n2 = 0.0;
            for (int k = 0; k < L; ++k) n2 += xd[tau0 + i + k] * xd[tau0 + i + k];
            double cv = (nc > 0.0) ? c[i] / nc : 0.0;
            double sv = (ns > 0.0) ? s[i] / ns : 0.0;
            double r = 0.0, cn = 0.0, sn = 0.0;
            if (n2 > 0.0) {
                double nx = sqrt(n2);
                r = sqrt(cv * cv + sv * sv) / nx;
                cn = cv / nx;
                sn = sv / nx;
            }
            rho[tau0 - lag_begin + i] = r;
            if (c_out) c_out[tau0 - lag_begin + i] = cn;
            if (s_out) s_out[tau0 - lag_begin + i] = sn;
        }
    }
    free(hc); free(hs); free(xd);
}

/* The whole search (SURVEY.md section 8(c) pseudo-code; north_star): for each template
 * j, rho_max[j] = max over lag_begin <= tau < lag_end of rho_j(tau) and arg_lag[j] =
 * the smallest tau attaining it (strict '>' while scanning upwards, C8).  Valid
 * lags only (C5): requires 0 <= lag_begin <= lag_end <= n_samples - L + 1.
 * Templates are independent; OpenMP runs them on n_threads threads (0 = default).
 * Returns the number of threads used, or -1 on bad arguments. */
int bfo_correlate_family(int family, const float *x, int64_t n_samples, double fs, int L,
                         int64_t n_templates, const double *p0, const double *p1, const double *p2,
                         int64_t lag_begin, int64_t lag_end, double *rho_max, int32_t *arg_lag,
                         int n_threads);
int bfo_correlate3(const float *x, int64_t n_samples, double fs, int L, int64_t n_templates,
                   const double *f0, const double *f1, const double *f2, int64_t lag_begin,
                   int64_t lag_end, double *rho_max, int32_t *arg_lag, int n_threads)
{
    return bfo_correlate_family(BFO_FAMILY_POLY, x, n_samples, fs, L, n_templates, f0, f1, f2,
                                lag_begin, lag_end, rho_max, arg_lag, n_threads);
}
int bfo_correlate(const float *x, int64_t n_samples, double fs, int L, int64_t n_templates,
                  const double *f0, const double *f1, int64_t lag_begin, int64_t lag_end,
                  double *rho_max, int32_t *arg_lag, int n_threads)
{
    return bfo_correlate3(x, n_samples, fs, L, n_templates, f0, f1, 0, lag_begin, lag_end, rho_max,
                          arg_lag, n_threads);
}

/* The same for either family: per-template parameters (p0, p1, p2) = (f0, f1, f2) (N1) or
 * (f_inf, D, tc) (N2); p2 == NULL means 0 (polynomial family only). */
int bfo_correlate_family(int family, const float *x, int64_t n_samples, double fs, int L,
                         int64_t n_templates, const double *p0, const double *p1, const double *p2,
                         int64_t lag_begin, int64_t lag_end, double *rho_max, int32_t *arg_lag,
                         int n_threads)
{
    if (L < 1 || n_samples < L || lag_begin < 0 || lag_end < lag_begin ||
        lag_end > n_samples - L + 1)
        return -1;
    const int64_t n_lags = lag_end - lag_begin;
    double *xd = (double *)malloc(sizeof(double) * (size_t)n_samples);
    for (int64_t i = 0; i < n_samples; ++i) xd[i] = (double)x[i];
    double *n2 = (double *)malloc(sizeof(double) * (size_t)(n_lags > 0 ? n_lags : 1));
    bfo_sliding_n2(x, L, lag_begin, lag_end, n2);
    int used = 1;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
    used = n_threads;
#else
    n_threads = 1;
#endif
#pragma omp parallel num_threads(n_threads)
    {
        double *hc = (double *)malloc(sizeof(double) * (size_t)L);
        double *hs = (double *)malloc(sizeof(double) * (size_t)L);
        double c[BFO_RUN], s[BFO_RUN];
#pragma omp for schedule(dynamic, 1)
        for (int64_t j = 0; j < n_templates; ++j) {
            double nc, ns;
            bfo_template_family(family, fs, L, p0[j], p1[j], p2 ? p2[j] : 0.0, hc, hs);
            bfo_template_norms(L, hc, hs, &nc, &ns);
            double best = -1.0;
            int64_t arg = lag_begin;
            for (int64_t tau0 = lag_begin; tau0 < lag_end; tau0 += BFO_RUN) {
                int n = (int)((lag_end - tau0 < BFO_RUN) ? (lag_end - tau0) : BFO_RUN);
                bfo_dots_run(xd, L, hc, hs, tau0, n, c, s);
                for (int i = 0; i < n; ++i) {
                    double cv = (nc > 0.0) ? c[i] / nc : 0.0;
                    double sv = (ns > 0.0) ? s[i] / ns : 0.0;
                    double nn = n2[tau0 - lag_begin + i];
                    double r = (nn > 0.0) ? sqrt(cv * cv + sv * sv) / sqrt(nn) : 0.0;
                    if (r > best) { best = r; arg = tau0 + i; }
                }
            }
            if (n_lags == 0) best = 0.0;
            rho_max[j] = best;
            arg_lag[j] = (int32_t)arg;
        }
        free(hc); free(hs);
    }
    free(n2); free(xd);
    return used;
}

/* Threshold and map (C9, C10; "rho exceeding kappa sigma", PAPER.md:54
 * "chirp-based spectrograms"): for each template with rho_max[j] > kappa (strict),
 *   tbin = (lag_origin + arg_lag[j]) / samples_per_tbin   (integer division)
 *   fbin = floor((f0[j] - f_lo) / df)
 * and map[tbin][fbin] += 1 if the bin is inside the map.  counters[0] counts all
 * hits, counters[1] the hits that fell outside.  map is accumulated into. */
void bfo_map(int64_t n_templates, const double *f0, const double *rho_max, const int32_t *arg_lag,
             double kappa, int64_t lag_origin, int32_t samples_per_tbin, double f_lo, double df,
             int32_t n_fbins, int32_t n_tbins, uint32_t *map, uint64_t *counters)
{
    for (int64_t j = 0; j < n_templates; ++j) {
        if (!(rho_max[j] > kappa)) continue;
        counters[0] += 1;
        int64_t tbin = (lag_origin + (int64_t)arg_lag[j]) / samples_per_tbin;
        double fb = floor((f0[j] - f_lo) / df);
        if (tbin >= 0 && tbin < n_tbins && fb >= 0.0 && fb < (double)n_fbins)
            map[tbin * (int64_t)n_fbins + (int64_t)fb] += 1;
        else
            counters[1] += 1;
    }
}

/* ---------------------------------------------------------------------------------------
 * The paper's own reduction ("only tails of
 * butterfly output rho exceeding kappa sigma ... are communicated to the CPU"
 * "sigma is the standard deviation of the matched filtered output rho, computed in a predictor
 * step by Parseval's Theorem").  Readings S1-S3:
 *
 * S1  The matched-filter output whose spread sigma measures is what the paper's length-N FFT
 *     correlation of a segment produces: the CIRCULAR correlation of the N-sample segment with
 *     the unit-norm quadrature templates,
 *         c~(tau) = sum_k x[(tau+k) mod N] hc[k] / nc,   s~(tau) likewise,   tau = 0 .. N-1,
 *     and sigma is its root mean square per quadrature (the second moment about zero is what
 *     Parseval's theorem delivers from the spectra):
 *         sigma^2 = (1 / (2 N)) sum_tau ( c~(tau)^2 + s~(tau)^2 ).
 * S2  Tails are taken over the VALID lags only (reading C5), of the un-normalised magnitude:
 *         rho_sigma(tau) = sqrt(c(tau)^2 + s(tau)^2) / sigma  >  kappa      (strict, C9),
 *     with c, s the unit-norm-template sums of bfo_rho_at (not divided by ||x_tau||).
 * S3  sigma == 0 (all-zero segment): no hits.
 * The tails apply to whatever bank is searched, so every function below takes
 * the template family; bfo_sigma / bfo_tails are the linear-chirp entry points.
 * ------------------------------------------------------------------------------------- */

/* S1, written out in the time domain (N L multiply-adds), for a template of either family. */
double bfo_sigma_family(int family, const float *x, int64_t n_samples, double fs, int L, double p0,
                        double p1, double p2)
{
    double *hc = (double *)malloc(sizeof(double) * (size_t)L);
    double *hs = (double *)malloc(sizeof(double) * (size_t)L);
    double nc, ns, acc = 0.0;
    bfo_template_family(family, fs, L, p0, p1, p2, hc, hs);
    bfo_template_norms(L, hc, hs, &nc, &ns);
    for (int64_t tau = 0; tau < n_samples; ++tau) {
        double c = 0.0, s = 0.0;
        for (int k = 0; k < L; ++k) {
            int64_t i = tau + k;
            if (i >= n_samples) i -= n_samples;          /* circular: L <= N */
            double xv = (double)x[i];
            c += xv * hc[k];
            s += xv * hs[k];
        }
        c = (nc > 0.0) ? c / nc : 0.0;
        s = (ns > 0.0) ? s / ns : 0.0;
        acc += c * c + s * s;
    }
    free(hc); free(hs);
    return sqrt(acc / (2.0 * (double)n_samples));
}
double bfo_sigma(const float *x, int64_t n_samples, double fs, int L, double f0, double f1)
{
    return bfo_sigma_family(BFO_FAMILY_POLY, x, n_samples, fs, L, f0, f1, 0.0);
}

/* S1-S3 for a list of templates.  sigma[j] is always written.  Hits are stored in ascending
 * (template, lag) order, the first `capacity` of them; the return value is the total number
 * of hits (which may exceed capacity), or -1 on bad arguments. */
int64_t bfo_tails_family(int family, const float *x, int64_t n_samples, double fs, int L,
                         int64_t n_templates, const double *p0, const double *p1, const double *p2,
                         int64_t lag_begin, int64_t lag_end, double kappa, double *sigma,
                         int64_t capacity, int32_t *hit_template, int32_t *hit_lag, double *hit_rho,
                         int n_threads)
{
    if (L < 1 || n_samples < L || lag_begin < 0 || lag_end < lag_begin ||
        lag_end > n_samples - L + 1)
        return -1;
    double *xd = (double *)malloc(sizeof(double) * (size_t)n_samples);
    for (int64_t i = 0; i < n_samples; ++i) xd[i] = (double)x[i];
    int64_t *count = (int64_t *)calloc((size_t)n_templates, sizeof(int64_t));
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#else
    n_threads = 1;
#endif
    /* pass 1: sigma and the number of hits of every template */
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
    for (int64_t j = 0; j < n_templates; ++j)
        sigma[j] = bfo_sigma_family(family, x, n_samples, fs, L, p0[j], p1[j], p2 ? p2[j] : 0.0);
    int64_t total = 0;
    for (int pass = 0; pass < 2; ++pass) {
        /* pass 0 counts, pass 1 stores at the offsets the counts give (ascending order) */
        int64_t *offset = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n_templates + 1));
        offset[0] = 0;
        for (int64_t j = 0; j < n_templates; ++j) offset[j + 1] = offset[j] + count[j];
        total = offset[n_templates];
#pragma omp parallel num_threads(n_threads)
        {
            double *hc = (double *)malloc(sizeof(double) * (size_t)L);
            double *hs = (double *)malloc(sizeof(double) * (size_t)L);
            double c[BFO_RUN], s[BFO_RUN];
#pragma omp for schedule(dynamic, 1)
            for (int64_t j = 0; j < n_templates; ++j) {
                double nc, ns;
                bfo_template_family(family, fs, L, p0[j], p1[j], p2 ? p2[j] : 0.0, hc, hs);
                bfo_template_norms(L, hc, hs, &nc, &ns);
                int64_t n_hit = 0;
                for (int64_t tau0 = lag_begin; tau0 < lag_end && sigma[j] > 0.0; tau0 += BFO_RUN) {
                    int n = (int)((lag_end - tau0 < BFO_RUN) ? (lag_end - tau0) : BFO_RUN);
                    bfo_dots_run(xd, L, hc, hs, tau0, n, c, s);
                    for (int i = 0; i < n; ++i) {
                        double cv = (nc > 0.0) ? c[i] / nc : 0.0;
                        double sv = (ns > 0.0) ? s[i] / ns : 0.0;
                        double r = sqrt(cv * cv + sv * sv) / sigma[j];
                        if (r > kappa) {
                            if (pass == 1) {
                                int64_t at = offset[j] + n_hit;
                                if (at < capacity) {
                                    hit_template[at] = (int32_t)j;
                                    hit_lag[at] = (int32_t)(tau0 + i);
                                    hit_rho[at] = r;
                                }
                            }
                            ++n_hit;
                        }
                    }
                }
                count[j] = n_hit;
            }
            free(hc); free(hs);
        }
        free(offset);
    }
    free(count); free(xd);
    return total;
}
int64_t bfo_tails(const float *x, int64_t n_samples, double fs, int L, int64_t n_templates,
                  const double *f0, const double *f1, int64_t lag_begin, int64_t lag_end,
                  double kappa, double *sigma, int64_t capacity, int32_t *hit_template,
                  int32_t *hit_lag, double *hit_rho, int n_threads)
{
    return bfo_tails_family(BFO_FAMILY_POLY, x, n_samples, fs, L, n_templates, f0, f1, 0, lag_begin,
                            lag_end, kappa, sigma, capacity, hit_template, hit_lag, hit_rho, n_threads);
}

int bfo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
