/*
 * bfly.h -- C ABI of the B200 (sm_100a) butterfly-filtering search library.
 *
 * The hot path of arXiv:1802.01685 sec. 2 ("Deep searches by butterfly filtering"):
 * correlate a whitened time series against a bank of up to ~8 million 1-second chirp
 * templates (start frequency f0, frequency derivative f1, ascending and descending;
 * PAPER.md:54-62) over every time lag (one correlation = one template
 * against one 16-s segment), keep per template the maximum over lags of the quadrature
 * correlation magnitude normalised by the sliding data norm and the lag where it falls,
 * and count the templates exceeding a threshold kappa into a time-frequency "butterfly"
 * map ("chirp-based spectrograms"; "only tails of butterfly
 * output rho exceeding kappa sigma are communicated").  The formulas are those of
 * BASELINE.json (north_star, configs[0]) in the readings listed in DESIGN.md.
 *
 *   phi_k    = 2 pi (f0 k/fs + 1/2 f1 (k/fs)^2),              k = 0 .. L-1
 *   c_j(tau) = sum_k x[tau+k] cos(phi_k) / ||cos phi||_2
 *   s_j(tau) = sum_k x[tau+k] sin(phi_k) / ||sin phi||_2
 *   rho_j(tau) = sqrt(c^2 + s^2) / sqrt(sum_k x[tau+k]^2)      (0 where the window is all zero)
 *   rho_max[j] = max_tau rho_j(tau),  arg_lag[j] = smallest tau attaining it
 *
 * Conventions
 *  - Plain C.  No exceptions, no aborts, nothing is printed.  Every call returns a status
 *    (BFLY_OK = 0, negative = error); bfly_strerror() names it and bfly_last_error() gives a
 *    thread-local detail string (e.g. the CUDA error text).
 *  - "DEVICE" pointers are CUDA device pointers on the bank's device; "HOST" pointers are
 *    ordinary host memory.  The caller owns every buffer it passes in; the library owns only
 *    the bank and the workspace inside it (released by bfly_free_bank).
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls that
 *    take a stream are asynchronous: they enqueue work and return; kernel faults surface as
 *    BFLY_ECUDA at a later call or at the caller's synchronisation.
 *  - Invalid arguments return BFLY_EINVAL before anything is launched.
 *  - Every call that takes a bank runs on the bank's device and restores the calling thread's
 *    current CUDA device before it returns; one process may hold banks on several devices.
 *  - The workspace inside a bank is one set of buffers.  A call that uses it (bfly_correlate*,
 *    bfly_tails, bfly_search_host, bfly_bank_reserve) while another thread is inside such a call
 *    on the same bank returns BFLY_EINVAL ("in use") instead of racing; successive calls on
 *    different streams are ordered by the library (the later stream waits for the earlier
 *    call's kernels), so results are as if the calls had been issued on one stream.
 *  - There is no CPU fallback: on a machine without an sm_100 device every call that needs the
 *    GPU returns BFLY_EUNSUPPORTED or BFLY_ECUDA.
 */
#ifndef BFLY_H
#define BFLY_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bfly_bank bfly_bank; /* opaque; device-resident; owned by the library */

enum {
    BFLY_OK = 0,
    BFLY_EINVAL = -1,       /* bad argument */
    BFLY_ENOMEM = -2,       /* host or device allocation failed */
    BFLY_ECUDA = -3,        /* a CUDA runtime call failed; see bfly_last_error() */
    BFLY_EUNSUPPORTED = -4, /* device is not compute capability 10.x, or form unsupported */
    BFLY_ERANGE = -5        /* a size exceeds what the library supports (see each call) */
};

/* Correlation forms (the core, row A4 of DESIGN.md).  All produce the same quantities. */
enum {
    BFLY_FORM_DEFAULT = 0, /* the form bfly_correlate() uses: BFLY_FORM_FFT_TC */
    BFLY_FORM_FFT = 1,     /* hand-written batched overlap-save FFT correlate, fp32 CUDA cores */
    BFLY_FORM_DIRECT = 2,  /* fp32 CUDA-core time-domain sums; slow cross-check of the core */
    BFLY_FORM_DENSE_TC = 4,/* lagged-data Hankel tile x template tile dense contraction on tcgen05
                              tensor cores (north_star (3)(a)): templates synthesised into shared
                              memory, data tiles by TMA, fp16 operands, fp32 accumulators in tensor
                              memory, epilogue per TMEM lane.  Executes 109x the flops of the FFT
                              forms: a cross-check and the tensor-pipe measurement, not the default.
                              Needs L >= BFLY_TC_MIN_L like BFLY_FORM_FFT_TC */
    BFLY_FORM_FFT_TC = 3,  /* the same overlap-save FFT correlate with the butterflies on the
                              tensor cores: small DFT matrices x data in fp16, fp32 accumulate,
                              fp32 twiddles and epilogue.  |d rho| ~ 1e-5 + 5e-5 rho.
                              Needs L >= BFLY_TC_MIN_L (BFLY_EUNSUPPORTED otherwise); the default
                              form falls back to BFLY_FORM_FFT for shorter templates */
    BFLY_FORM_FFT_TC5 = 5  /* the same with the length-8192 transform as 64 x 128 on tcgen05.mma
                              (DFT matrices resident in tensor memory, fp32 accumulators in TMEM,
                              data through swizzled shared memory; csrc/bfly_fft_tc5.cu).  Needs
                              L >= BFLY_TC_MIN_L */
};
#define BFLY_TC_MIN_L 256

const char *bfly_strerror(int status);
const char *bfly_last_error(void);

/* ---- A1: the bank (a persistent bank of chirp templates) -------------
 * Explicit list of templates.  f0_hz / f1_hzps: HOST pointers, n_templates float64 each (Hz,
 * Hz/s; any finite values: templates that sweep through 0 Hz or beyond fs/2 are legal, the
 * definition is the sampled formula).  L = template length in samples (2 <= L <= 4096; the
 * "1 s" is L/fs).  Computes per template, on the device in float64, 1/||cos phi||^2 and
 * 1/||sin phi||^2 (0 if the norm is 0) and the fixed-point phase constants used to synthesise
 * the template inside the correlation kernels; template waveforms are never stored.
 * Synchronous (returns when the bank is ready).  *out_bank is written only on success. */
int bfly_make_bank(double fs_hz, int32_t L, int64_t n_templates,
                   const double *f0_hz, const double *f1_hzps,
                   int device, bfly_bank **out_bank);

/* The non-linear family (descending chirps that
 * settle towards a late-time frequency; the paper gives no waveform; reading N1 of DESIGN.md):
 * templates with a constant second frequency derivative f2 [Hz/s^2],
 *     f(t) = f0 + f1 t + f2 t^2 / 2,     phi_k = 2 pi (f0 t_k + f1 t_k^2 / 2 + f2 t_k^3 / 6),
 * which carry an exponentially settling chirp f_inf + D exp(-t / tc) over one template by its
 * frequency, slope and curvature at the template's first sample.  f2_hzps2: HOST, n_templates
 * float64, or NULL for all zero (then identical to bfly_make_bank).  Every other call works on
 * such a bank unchanged; bfly_butterfly_map bins by f0 as before. */
int bfly_make_bank3(double fs_hz, int32_t L, int64_t n_templates,
                    const double *f0_hz, const double *f1_hzps, const double *f2_hzps2,
                    int device, bfly_bank **out_bank);
/* f2 of templates [first, first + count) to a HOST float64 array.  Synchronous. */
int bfly_bank_get_f2(const bfly_bank *bank, int64_t first, int64_t count, double *f2_hzps2);

/* Convenience: inclusive uniform grids f0 = f0_lo + i (f0_hi - f0_lo)/(n_f0 - 1) (likewise
 * f1), evaluated in float64 exactly like numpy.linspace; template j = i_f0 * n_f1 + i_f1. */
int bfly_make_bank_grid(double fs_hz, int32_t L,
                        double f0_lo, double f0_hi, int32_t n_f0,
                        double f1_lo, double f1_hi, int32_t n_f1,
                        int device, bfly_bank **out_bank);

void bfly_free_bank(bfly_bank *bank);            /* NULL is allowed */
int64_t bfly_bank_size(const bfly_bank *bank);   /* number of templates; -1 if bank is NULL */

/* Template families.  BFLY_FAMILY_POLY: polynomial phase (f0, f1 [, f2]) -- bfly_make_bank,
 * bfly_make_bank3, bfly_make_bank_grid.  BFLY_FAMILY_SETTLE: exponentially settling chirps,
 * bfly_make_bank_settle below. */
enum { BFLY_FAMILY_POLY = 0, BFLY_FAMILY_SETTLE = 1 };

/* ---- A1 for the settling family (reading N2 of DESIGN.md) ---------------
 * PAPER.md:21-26 (sec. 1, Eq. 1: descending chirps of a spinning-down black hole-disk system that
 * "reach a late time plateau" f_GW = 600-700 Hz (M/10 Msun)^-1), PAPER.md:60 (Fig. 2, right) and
 * PAPER.md:54 ("trajectories of frequency f(t)"); the paper prints no waveform, the reading is
 *     f(t) = f_inf + D exp(-t / tc),   phi_k = 2 pi ( f_inf t_k + D tc (1 - exp(-t_k / tc)) ),
 * t_k = k/fs, k = 0 .. L-1: D = f(0) - f_inf [Hz] (D > 0 descends towards the plateau f_inf), tc > 0
 * the settling time [s].  f_inf_hz, delta_hz, tau_c_s: HOST, n_templates float64 each.  The rest of
 * the path is unchanged: every correlation form, bfly_tails, the maps.  The butterfly map bins a
 * template by its START frequency f_inf + D (reading C10: the frequency the signal has at the
 * start of the matched window); bfly_bank_get returns that as f0, with f1 = -D/tc and
 * bfly_bank_get_f2 = D/tc^2 (slope and curvature at the first sample).  Errors as bfly_make_bank;
 * BFLY_EINVAL also for tc <= 0 or a non-finite parameter. */
int bfly_make_bank_settle(double fs_hz, int32_t L, int64_t n_templates, const double *f_inf_hz,
                          const double *delta_hz, const double *tau_c_s, int device,
                          bfly_bank **out_bank);
/* The family of a bank (BFLY_FAMILY_*; -1 for a null bank), and the parameters of templates
 * [first, first + count) of a settling bank (HOST outputs, any may be NULL; BFLY_EINVAL for a
 * bank of the other family). */
int bfly_bank_family(const bfly_bank *bank);
int bfly_bank_get_settle(const bfly_bank *bank, int64_t first, int64_t count, double *f_inf_hz,
                         double *delta_hz, double *tau_c_s);

/* Copy bank parameters of templates [first, first + count) to HOST arrays (any may be NULL):
 * f0, f1 (float64) and the stored 1/||cos phi||^2, 1/||sin phi||^2 (float32).  Synchronous. */
int bfly_bank_get(const bfly_bank *bank, int64_t first, int64_t count,
                  double *f0_hz, double *f1_hzps, float *inv_nc2, float *inv_ns2);

/* Pre-size the workspace inside the bank for segments of up to max_n_samples samples, so that
 * later bfly_correlate calls allocate nothing.  Without it the first call with a longer segment
 * grows the workspace (a synchronising cudaMalloc).  Synchronous. */
int bfly_bank_reserve(bfly_bank *bank, int64_t max_n_samples);

/* ---- A2-A7: correlate one segment against the whole bank ---------------------------------
 * x_dev: DEVICE, n_samples fp32, read-only.  Lags searched: lag_begin <= tau < lag_end, which
 * must lie within the valid lags [0, n_samples - L + 1) (no zero padding, no circular wrap).
 * rho_max_dev[T] fp32 and arg_lag_dev[T] int32: DEVICE, overwritten; arg_lag is relative to
 * x_dev[0].  An empty lag range gives rho_max = 0, arg_lag = lag_begin.  n_samples < 2^31.
 * Asynchronous on `stream`; no host synchronisation; no allocation if the workspace is
 * already large enough (see bfly_bank_reserve).  One call at a time per bank (the workspace
 * is shared): a concurrent second call from another thread returns BFLY_EINVAL, and a call on
 * another stream than the previous one is ordered after it (Conventions above). */
int bfly_correlate(const bfly_bank *bank, const float *x_dev, int64_t n_samples,
                   int64_t lag_begin, int64_t lag_end,
                   float *rho_max_dev, int32_t *arg_lag_dev, void *stream);

/* ---- the same without any allocation -------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it): bfly_correlate in its default form (BFLY_FORM_FFT_TC: needs
 * L >= BFLY_TC_MIN_L, else BFLY_EUNSUPPORTED) with the per-call scratch -- data-block spectra,
 * per-lag normalisers, block scales: what bfly_correlate keeps in the bank's workspace -- in a
 * file-scope static device array of 1 MB + 256 B inside the library, which every GPU that loads
 * the library holds until the process exits.  Arguments, layouts, results (bit for bit) and error
 * behaviour as bfly_correlate (rows A2-A7), except:
 *  - n_samples <= BFLY_STATIC_MAX_SAMPLES (one 16-s segment at 4096 Hz, 16 overlap-save blocks);
 *    a longer segment returns BFLY_ERANGE and launches nothing;
 *  - the call allocates and frees nothing, on the host or the device, reads the bank's
 *    parameters only, does not touch its workspace and does not take its in-use flag;
 *  - ALL calls, on any bank and any stream of the same device, share the one array: two calls
 *    that overlap on the GPU race (serialise them on one stream or with events).  The array
 *    keeps the previous call's contents; every region a call reads it writes first, so nothing
 *    needs clearing. */
#define BFLY_STATIC_MAX_SAMPLES 65536
int bfly_correlate_static(const bfly_bank *bank, const float *x_dev, int64_t n_samples,
                          int64_t lag_begin, int64_t lag_end, float *rho_max_dev,
                          int32_t *arg_lag_dev, void *stream);

/* The same with an explicit correlation form (BFLY_FORM_*). */
int bfly_correlate_form(const bfly_bank *bank, int form, const float *x_dev, int64_t n_samples,
                        int64_t lag_begin, int64_t lag_end,
                        float *rho_max_dev, int32_t *arg_lag_dev, void *stream);

/* ---- several segments against the same bank in one call ---------------------------------------
 * PAPER.md:124 (Fig. 6: the same search on the two detectors H1 and L1, "simultaneous rho > kappa
 * sigma in H1 and L1"), PAPER.md:70 (the bank is applied segment after segment); DESIGN.md 6.1.
 * n_segments >= 1 segments of n_samples samples each; x_dev, rho_max_dev, arg_lag_dev: HOST arrays
 * of n_segments DEVICE pointers (layouts as bfly_correlate); the same lag range in every segment.
 * The results are those of n_segments calls of bfly_correlate, bit for bit; what changes is the
 * cost: up to four segments go through one launch of the default form, in which the template is
 * synthesised and transformed once per template for all of them (measured on 16-s segments:
 * 1.4 % less time per correlation at two segments, 4.0 % at four).  Segments whose lags past the last whole block
 * cannot be taken from a transform (n_lags mod 4096 in 1..4 with L > 4096 - that remainder), and
 * banks with L < BFLY_TC_MIN_L, are processed one call per segment.  Errors as bfly_correlate. */
int bfly_correlate_multi(const bfly_bank *bank, int32_t n_segments, const float *const *x_dev, int64_t n_samples,
                         int64_t lag_begin, int64_t lag_end, float *const *rho_max_dev,
                         int32_t *const *arg_lag_dev, void *stream);

/* ---- A8: threshold and accumulate into the butterfly map ---------------------------------
 * For every template with rho_max > kappa (strict, compared in fp32):
 *     tbin = (lag_origin + arg_lag) / samples_per_tbin        (integer division)
 *     fbin = floor((f0 - f_lo_hz) / df_hz)                    (float64)
 *     map_dev[tbin * n_fbins + fbin] += 1     if 0 <= tbin < n_tbins and 0 <= fbin < n_fbins
 * counters_dev[0] += number of hits, counters_dev[1] += hits that fell outside the map.
 * map_dev (uint32, row-major [n_tbins][n_fbins]) and counters_dev (2 x uint64) are DEVICE
 * buffers that are ACCUMULATED into (the caller zeroes them).  rho_max_dev / arg_lag_dev are
 * the outputs of bfly_correlate for the same bank.  lag_origin >= 0 is the absolute sample
 * index of x_dev[0] in a longer stream (0 for a single segment).  Asynchronous on `stream`. */
int bfly_butterfly_map(const bfly_bank *bank,
                       const float *rho_max_dev, const int32_t *arg_lag_dev,
                       float kappa, int64_t lag_origin, int32_t samples_per_tbin,
                       double f_lo_hz, double df_hz, int32_t n_fbins, int32_t n_tbins,
                       uint32_t *map_dev, uint64_t *counters_dev, void *stream);

/* ---- The paper's own reduction: tails of the output above kappa sigma ----------------------
 * PAPER.md:70 ("only tails of butterfly output rho exceeding kappa sigma ... are communicated to
 * the CPU"), PAPER.md:120 ("sigma is the standard deviation of the matched filtered output rho,
 * computed in a predictor step by Parseval's Theorem").  Readings S1-S3 of DESIGN.md:
 *     sigma_j^2 = (1 / (2 N)) sum_{tau < N} ( c~_j(tau)^2 + s~_j(tau)^2 ),   N = n_samples,
 * c~, s~ the CIRCULAR correlations of the whole segment x_dev[0 .. N) with the unit-norm
 * quadrature templates (what a length-N FFT correlation produces; evaluated from spectra by
 * Parseval's theorem, never in the time domain), and a hit is every valid lag
 * lag_begin <= tau < lag_end with
 *     rho_sigma = sqrt(c_j(tau)^2 + s_j(tau)^2) / sigma_j  >  kappa          (strict, fp32),
 * c, s the sums of bfly_correlate before the division by ||x_tau||.  sigma_j = 0 gives no hits.
 * Outputs (DEVICE, caller-owned): sigma_dev[T] fp32, overwritten; the hit list
 * hit_template_dev / hit_lag_dev / hit_rho_dev [capacity] in NO particular order (lags relative
 * to x_dev[0]); *n_hits_dev (uint64) is INCREMENTED by the number of hits found, which may
 * exceed capacity: hits are then stored at positions old count .. capacity - 1 only and the
 * caller sees the overflow from the count (the caller zeroes the counter before the first call
 * and may chain calls into one list).  Needs L >= BFLY_TC_MIN_L (runs on the tensor-core FFT
 * form); BFLY_EUNSUPPORTED otherwise.  Asynchronous on `stream`. */
int bfly_tails(const bfly_bank *bank, const float *x_dev, int64_t n_samples, int64_t lag_begin,
               int64_t lag_end, float kappa, float *sigma_dev, int64_t capacity,
               int32_t *hit_template_dev, int32_t *hit_lag_dev, float *hit_rho_dev,
               uint64_t *n_hits_dev, void *stream);

/* One count per hit of a bfly_tails list at (tbin of lag_origin + hit_lag, fbin of the hit
 * template's f0): the coordinates and accumulation rules of bfly_butterfly_map, but a template
 * may contribute many hits per segment (the paper's trajectory map).  n_hits is a
 * HOST value: the number of list entries to use (at most the list's capacity). */
int bfly_hits_map(const bfly_bank *bank, const int32_t *hit_template_dev, const int32_t *hit_lag_dev,
                  int64_t n_hits, int64_t lag_origin, int32_t samples_per_tbin, double f_lo_hz,
                  double df_hz, int32_t n_fbins, int32_t n_tbins, uint32_t *map_dev,
                  uint64_t *counters_dev, void *stream);

/* ---- Reading the output of two series: control, coincidence, pseudo-spectra ----------------
 * PAPER.md:68 (control "following time-randomisation of the H1 and L1 data ... maximal entropy,
 * keeping histograms the same"), PAPER.md:124 ("pseudo-spectra of simultaneous rho > kappa sigma
 * in H1 and L1 ... by independent counts and by simultaneous counts with frequency pairs within
 * Delta f = 50 Hz").  Readings T1-T3 of DESIGN.md.  These three calls need no bank; they run on
 * the CURRENT device, asynchronously on `stream`; all pointers are DEVICE, caller-owned.
 *
 * T1  out_dev[i] = x_dev[perm_dev[i]], i < n.  perm_dev (int32) is an INPUT: a permutation of
 *     0..n-1 drawn by the caller's seeded generator (the library draws no random numbers).  An
 *     index outside [0, n) writes 0 and sets *bad_dev (int32, may be NULL) to 1.  out_dev must
 *     not alias x_dev.  The control is then the same bfly_correlate / bfly_tails on out_dev. */
int bfly_time_randomize(const float *x_dev, const int32_t *perm_dev, int64_t n, float *out_dev,
                        int32_t *bad_dev, void *stream);

/* T2  Two count maps of the same geometry (uint32 [n_tbins][n_fbins], one count per hit, as
 *     bfly_butterfly_map / bfly_hits_map write them).  co1_dev[t][f] = map1_dev[t][f] if map2_dev
 *     has a non-zero bin at the same time bin t within half_width_bins frequency bins of f, else
 *     0; co2_dev likewise with the roles exchanged.  co1_dev / co2_dev are OVERWRITTEN and must
 *     not alias the inputs.  n_fbins <= 65536 (BFLY_ERANGE). */
int bfly_coincidence(const uint32_t *map1_dev, const uint32_t *map2_dev, int32_t n_tbins,
                     int32_t n_fbins, int32_t half_width_bins, uint32_t *co1_dev,
                     uint32_t *co2_dev, void *stream);

/* T3  spectrum_dev[f] += sum over t of map_dev[t][f]  (uint64 [n_fbins], ACCUMULATED into, so
 *     that blocks of a long run add up; the caller zeroes it). */
int bfly_pseudo_spectrum(const uint32_t *map_dev, int32_t n_tbins, int32_t n_fbins,
                         uint64_t *spectrum_dev, void *stream);

/* ---- A9 / end-to-end: the whole path on a HOST series ------------------------------------
 * Runs A2-A8 over a HOST series x_host[n_samples] (fp32), cut into chunks of chunk_samples
 * samples with an overlap of L samples (hop = chunk_samples - L): chunk c starts at sample
 * c * hop, searches its local lags [0, hop), the last chunk all the valid lags it has left,
 * so every valid lag of the series is searched exactly once; lag_origin = c * hop; the map
 * accumulates over chunks (one hit per template per chunk at most).  chunk_samples <= 0 or
 * >= n_samples means a single chunk.  Copies each chunk host->device, runs bfly_correlate and
 * bfly_butterfly_map on `stream`, and at the end copies to the HOST outputs (any may be NULL):
 * rho_max_host[T] / arg_lag_host[T] of the LAST chunk (arg_lag local to that chunk), map_host
 * [n_tbins * n_fbins] (overwritten with the run's counts) and counters_host[2].  Synchronous:
 * returns when the outputs are in host memory. */
int bfly_search_host(bfly_bank *bank, const float *x_host, int64_t n_samples,
                     int64_t chunk_samples, float kappa, int32_t samples_per_tbin,
                     double f_lo_hz, double df_hz, int32_t n_fbins, int32_t n_tbins,
                     float *rho_max_host, int32_t *arg_lag_host,
                     uint32_t *map_host, uint64_t *counters_host, void *stream);

/* Measurement aid (bench.py's roofline figure).  With timing enabled, bfly_correlate records a
 * CUDA event on `stream` immediately before and after the launch of its correlation-core
 * kernel (row A4-A7; the dominant kernel).  bfly_bank_core_ms waits for the stop event of the
 * most recent bfly_correlate call on this bank and returns the elapsed device time between the
 * two events in milliseconds (BFLY_EINVAL if timing is off or no call was made). */
int bfly_bank_set_timing(bfly_bank *bank, int enable);
int bfly_bank_core_ms(bfly_bank *bank, float *ms_out);

/* Diagnostic (tests only): the bare length-8192 transform of BFLY_FORM_FFT_TC,
 *     z[n] = sum_m y[m] exp(+2 pi i m n / 8192),
 * on one natural-order input.  y_dev, z_dev: DEVICE, 8192 interleaved complex fp32 each
 * (16384 floats), caller-owned.  full = 0 computes only n < 4096 (what the correlation uses;
 * z[4096..] is left untouched), full != 0 all 8192 outputs.  Inputs are rounded to fp16, so
 * |y| must stay within the fp16 range.  Asynchronous on `stream`. */
int bfly_debug_fft_tc(const float *y_dev, float *z_dev, int full, void *stream);

/* Diagnostic (tests and DESIGN.md 10 only): the same transform on the 5th-generation tensor cores
 * (tcgen05.mma kind::f16, DFT matrices resident in tensor memory, data through swizzled shared
 * memory; csrc/bfly_fft_tc5.cu), outputs n < 4096 only.  y_dev: DEVICE, 2 n_pairs transforms of
 * 8192 interleaved complex fp32; z_dev: DEVICE, 2 n_pairs x 4096 interleaved complex fp32,
 * overwritten.  One CTA; `reps` repeats every pair (timing: cycles_dev[0], optional DEVICE int64,
 * receives the SM clock cycles of the whole loop).  Asynchronous on `stream`. */
int bfly_debug_fft_tc5(const float *y_dev, float *z_dev, int32_t n_pairs, int32_t reps, int64_t *cycles_dev,
                       void *stream);

/* Measurement aid (bench.py's roofline denominators; "measured by a microbenchmark
 * on the box"): runs one microbenchmark kernel on every SM of the CURRENT device (two warm-up
 * launches, the third timed with CUDA events) and returns its rate.  Synchronous.
 *   BFLY_PEAK_FFMA   value_out[0] = fp32 flop/s of independent FFMA chains (2 flop each)
 *   BFLY_PEAK_FFMA2  the same with the packed two-lane FFMA2 of sm_100 (4 flop each)
 *   BFLY_PEAK_LDS    bytes/s of a conflict-free ld.shared.v4 stream
 *   BFLY_PEAK_HMMA   flop/s of independent mma.sync.m16n8k16 f16 -> f32 (4096 flop each)
 *   BFLY_PEAK_SHFL   warp shuffles/s
 *   BFLY_PEAK_L2     bytes/s of ld.global.v4 over a 480 KB set shared by all CTAs (L2-resident)
 *   BFLY_PEAK_UMMA   value_out must hold 2 doubles: [0] = flop per clock and SM of back-to-back
 *                    tcgen05.mma kind::f16 M = 128, K = 16 (variant bits 0-1: 1 = A, B from shared
 *                    memory, 2 = A from tensor memory, 0 = none; bit 2: N = 256 instead of 128),
 *                    [1] = clocks per iteration of 16 warps streaming beside it (bit 3: 32 KB of
 *                    st.shared.v4 + 32 KB of ld.shared.v4 per iteration; bit 4: 64 KB of
 *                    tcgen05.ld per iteration; bit 5: consecutive MMAs accumulate into two tiles
 *                    in turn; bit 6: N = 64)
 * `variant` is ignored by the others.  ms_out (optional): the timed launch in milliseconds. */
enum { BFLY_PEAK_FFMA = 0, BFLY_PEAK_FFMA2 = 1, BFLY_PEAK_LDS = 2, BFLY_PEAK_HMMA = 3,
       BFLY_PEAK_SHFL = 4, BFLY_PEAK_L2 = 5, BFLY_PEAK_UMMA = 6 };
int bfly_debug_peak(int which, int variant, int iters, double *value_out, double *ms_out);

/* Number of kernel launches the library has enqueued so far in this process (for bench.py's
 * gpu_launches claim). */
int64_t bfly_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* BFLY_H */
