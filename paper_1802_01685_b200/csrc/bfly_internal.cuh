// Internal declarations shared by the translation units of libbfly (not part of the C ABI).
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/bfly.h"

struct bfly_bank {
    int device;
    int sm_count;
    double fs;
    int32_t L;
    int64_t T;
    // per-template parameters (device, struct of arrays; A1)
    double *f0;      // Hz
    double *f1;      // Hz/s
    double *f2;      // Hz/s^2 (reading N1: the non-linear family; all zero for a linear bank)
    uint64_t *phA;   // f0/fs            in units of 2^-64 cycles per sample
    uint64_t *phB;   // f1/(2 fs^2)      in units of 2^-64 cycles per sample^2
    uint64_t *phC;   // f2/(6 fs^3)      in units of 2^-64 cycles per sample^3
    int has_f2;      // some template has f2 != 0 (selects the cubic-phase kernel variants)
    int family;      // BFLY_FAMILY_POLY: phA/phB/phC as above.  BFLY_FAMILY_SETTLE (reading N2):
                     // f(t) = f_inf + D exp(-t/tc); phA = f_inf/fs as above, phB = the bits of the
                     // double D tc [cycles], phC = the bits of the double 1/(fs tc) [1/sample];
                     // f0/f1/f2 hold the frequency, slope and curvature at the first sample
    double *s_finf, *s_delta, *s_tc;   // the settle family's own parameters (bfly_bank_get_settle)
    float *inc2;     // 1 / ||cos phi||^2 (0 if the norm is 0)
    float *ins2;     // 1 / ||sin phi||^2
    // workspace (grown by bfly_bank_reserve / on demand)
    float *rn2;               // 1 / n2[tau] for the lags of the current call
    int64_t rn2_cap;          // floats
    float2 *xspec;            // data-block spectra X_b, [block][FFT_B] complex, natural order
    int64_t xspec_cap;        // complex elements
    __half *xh;               // BFLY_FORM_FFT_TC: data-block spectra, fp16, operand layout
    int64_t xh_cap;           // halves (16384 per block)
    float *rn2p;              // BFLY_FORM_FFT_TC: per-lag normaliser in epilogue order
    int64_t rn2p_cap;         // floats (4096 per block)
    double *qs;               // BFLY_FORM_FFT_TC: per-block scale 2^(-2s) / S16^2
    int64_t qs_cap;
    double *racf;             // bfly_tails: circular autocorrelation of the segment, lags 0..L-1
    float *wspec;             // bfly_tails: its length-8192 transform W in the operand layout
    __half *ys;               // BFLY_FORM_DENSE_TC: eight shifted fp16 copies of the scaled series
    int64_t ys_cap;
    float *rn2s;              // BFLY_FORM_DENSE_TC: 1 / (n2 scale^2), padded to whole lag tiles
    int64_t rn2s_cap;
    unsigned int *maxbits;    // BFLY_FORM_DENSE_TC: bits of max |x| of the current call
    int64_t maxbits_cap;
    unsigned long long *packed;  // T packed (rho^2 bits, ~lag) words for the direct form
    float *x_stage;           // device copy of a host chunk (bfly_search_host)
    int64_t x_stage_cap;
    float *rho_multi;         // bfly_search_host with several chunks per launch: group x T each
    int32_t *arg_multi;
    int64_t rho_multi_cap, arg_multi_cap;
    float *rho_stage;         // T
    int32_t *arg_stage;       // T
    uint32_t *map_stage;
    int64_t map_stage_cap;
    unsigned long long *cnt_stage;  // 2
    // guards of the mutable workspace: `busy` makes a second host thread entering a
    // workspace-using call on the same bank fail with BFLY_EINVAL instead of racing; `ws_event`
    // (recorded at the end of every such call) orders the workspace between streams: a call on
    // another stream than the previous one first waits for it
    int busy;
    cudaEvent_t ws_event;
    cudaStream_t ws_stream;
    int ws_valid;
    // measurement aid (bfly_bank_set_timing)
    int timing;
    int timed;                  // a start/stop pair has been recorded
    cudaEvent_t ev_start, ev_stop;
};

namespace bfly {

void set_error(const char *fmt, ...);
int cuda_fail(cudaError_t e, const char *what);   // records the message, returns BFLY_ECUDA
void count_launch(int n = 1);

#define BFLY_CUDA(call)                                          \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return bfly::cuda_fail(e__, #call); \
    } while (0)

// One-time setup that must run once PER DEVICE (cudaFuncSetAttribute applies to the current
// device's copy of the function only), thread safe.  f() returns a BFLY_* status.
constexpr int MAX_DEVICES = 64;
struct PerDeviceOnce {
    std::mutex m;
    bool done[MAX_DEVICES] = {};
    template <class F>
    int run(int device, F &&f)
    {
        if (device < 0 || device >= MAX_DEVICES) { set_error("device %d out of range", device); return BFLY_EINVAL; }
        std::lock_guard<std::mutex> g(m);
        if (done[device]) return BFLY_OK;
        const int rc = f();
        if (rc == BFLY_OK) done[device] = true;
        return rc;
    }
};

// Every entry point runs on the bank's device and leaves the caller's current device as it was.
struct DeviceGuard {
    int prev = -1, dev;
    cudaError_t err;
    explicit DeviceGuard(int device) : dev(device)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        err = prev == device ? cudaSuccess : cudaSetDevice(device);
    }
    ~DeviceGuard() { if (prev >= 0 && prev != dev) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

// Exclusive use of a bank's workspace for the duration of one call (host side).
struct BankLock {
    bfly_bank *b;
    bool held;
    explicit BankLock(const bfly_bank *bank) : b(const_cast<bfly_bank *>(bank))
    {
        int expected = 0;
        held = __atomic_compare_exchange_n(&b->busy, &expected, 1, false, __ATOMIC_ACQUIRE, __ATOMIC_RELAXED);
    }
    ~BankLock() { if (held) __atomic_store_n(&b->busy, 0, __ATOMIC_RELEASE); }
    BankLock(const BankLock &) = delete;
    BankLock &operator=(const BankLock &) = delete;
};

// bfly_bank_set_timing: events around the correlation-core kernel on the caller's stream
inline void core_timer_start(const bfly_bank *b, cudaStream_t st)
{
    if (b->timing) cudaEventRecord(b->ev_start, st);
}
inline void core_timer_stop(const bfly_bank *b, cudaStream_t st)
{
    if (b->timing) {
        cudaEventRecord(b->ev_stop, st);
        const_cast<bfly_bank *>(b)->timed = 1;
    }
}

// FFT-form geometry: block length of the overlap-save FFT.
constexpr int FFT_LOG2B = 13;
constexpr int FFT_B = 1 << FFT_LOG2B;   // 8192
constexpr int FFT_MAX_L = FFT_B / 2;    // 4096

// launchers (each enqueues on `stream`, returns a BFLY_* status)
int launch_bank_params(bfly_bank *b, cudaStream_t stream);
int launch_bank_params_settle(bfly_bank *b, cudaStream_t stream);
int launch_sliding_norm(const float *x, int64_t n_samples, int32_t L, int64_t lag_begin,
                        int64_t n_lags, float *rn2, cudaStream_t stream);
int launch_direct(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                  int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream);
int launch_fft(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
               int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream);
int launch_map(const bfly_bank *b, const float *rho_max, const int32_t *arg_lag, float kappa,
               int64_t lag_origin, int32_t samples_per_tbin, double f_lo, double df,
               int32_t n_fbins, int32_t n_tbins, uint32_t *map, unsigned long long *counters,
               cudaStream_t stream);
int64_t fft_blocks_needed(int32_t L, int64_t n_lags);
int launch_fft_tc(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                  int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream);
int launch_fft_tc_static(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin, int64_t lag_end,
                         float *rho_max, int32_t *arg_lag, cudaStream_t stream);
int64_t tc_blocks_needed(int64_t n_lags);
bool tc_multi_supported(int32_t L, int64_t n_lags);
int launch_fft_tc_multi(const bfly_bank *b, int n_seg, const float *const *x, int64_t n_samples, int64_t lag_begin,
                        int64_t lag_end, float *const *rho_max, int32_t *const *arg_lag, cudaStream_t stream);
void tc_plan(int64_t n_lags, int64_t *n_blocks, int32_t *n_tail);
int launch_fft_tc5(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                   int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream);
int launch_tails_tc(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                    int64_t lag_end, float kappa, float *sigma, int64_t capacity,
                    int32_t *hit_template, int32_t *hit_lag, float *hit_rho,
                    unsigned long long *n_hits, cudaStream_t stream);
int launch_hits_map(const bfly_bank *b, const int32_t *hit_template, const int32_t *hit_lag,
                    int64_t n_hits, int64_t lag_origin, int32_t samples_per_tbin, double f_lo,
                    double df, int32_t n_fbins, int32_t n_tbins, uint32_t *map,
                    unsigned long long *counters, cudaStream_t stream);
int launch_time_randomize(const float *x, const int32_t *perm, int64_t n, float *out, int *bad,
                          cudaStream_t stream);
int launch_coincidence(const uint32_t *m1, const uint32_t *m2, int32_t n_tbins, int32_t n_fbins,
                       int32_t w, uint32_t *c1, uint32_t *c2, cudaStream_t stream);
int launch_pseudo_spectrum(const uint32_t *m, int32_t n_tbins, int32_t n_fbins,
                           unsigned long long *spec, cudaStream_t stream);
int launch_dense_tc(bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin, int64_t lag_end,
                    float *rho_max, int32_t *arg_lag, cudaStream_t stream);
int launch_debug_fft_tc(const float2 *y, float2 *z, int full, cudaStream_t stream);
int launch_debug_fft_tc5(const float2 *y, float2 *z, int n_pairs, int reps, long long *cycles_dev, cudaStream_t stream);

// Template phase in cycles, as a 64-bit fixed-point fraction:
// phi_k/2pi mod 1 = (A k + B k^2 + C k^3) 2^-64 (Horner, modulo 2^64: the wrap is the mod 1).
__device__ __forceinline__ uint64_t template_phase(uint64_t A, uint64_t B, uint64_t C, uint64_t k)
{
    return ((C * k + B) * k + A) * k;
}
// The settling family (reading N2): phi_k/2pi = f_inf k/fs + D tc (1 - exp(-k/(fs tc))).
// The linear term is exact fixed point (A k mod 2^64); the exponential term is evaluated in float64
// (-expm1 keeps full precision for k << fs tc; |D tc| of a few thousand cycles leaves an absolute
// error of ~1e-12 cycle), reduced modulo one cycle and added as a 2^-64 fraction.
__device__ __forceinline__ uint64_t settle_phase(uint64_t A, double Dtc, double inv_fstc, uint64_t k)
{
    double v = Dtc * (-expm1(-inv_fstc * (double)k));
    v -= floor(v);                                           // [0, 1)
    return A * k + __double2ull_rz(v * 18446744073709551616.0);
}
__device__ __forceinline__ uint64_t family_phase(int family, uint64_t A, uint64_t B, uint64_t C, uint64_t k)
{
    if (family == BFLY_FAMILY_SETTLE)
        return settle_phase(A, __longlong_as_double((long long)B), __longlong_as_double((long long)C), k);
    return template_phase(A, B, C, k);
}
__device__ __forceinline__ void template_sincos(int family, uint64_t A, uint64_t B, uint64_t C, uint32_t k,
                                                float *s, float *c)
{
    uint64_t ph = family_phase(family, A, B, C, k);
    // top 32 bits as a signed fraction of a half-turn: angle = pi * v, v in [-1, 1)
    float v = (float)(int32_t)(uint32_t)(ph >> 32) * 4.656612873077393e-10f;  // 2^-31
    sincospif(v, s, c);
}

}  // namespace bfly
