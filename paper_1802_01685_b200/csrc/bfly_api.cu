// C ABI entry points of libbfly: argument validation, bank and workspace management.
// See include/bfly.h for the contract of every call.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <atomic>
#include <new>
#include <vector>

#include "bfly_internal.cuh"

namespace bfly {

static thread_local char g_err[512] = "";
static std::atomic<int64_t> g_launches{0};

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char *what)
{
    set_error("%s: %s", what, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? BFLY_ENOMEM : BFLY_ECUDA;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static int select_device(int device, int *sm_count)
{
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n <= 0) {
        set_error("no CUDA device (%s); there is no CPU fallback", cudaGetErrorString(e));
        return BFLY_EUNSUPPORTED;
    }
    if (device < 0 || device >= n) {
        set_error("device %d out of range (0..%d)", device, n - 1);
        return BFLY_EINVAL;
    }
    cudaDeviceProp p;
    BFLY_CUDA(cudaGetDeviceProperties(&p, device));
    if (p.major != 10) {
        set_error("device %d is sm_%d%d; this library is built for sm_100a only", device, p.major,
                  p.minor);
        return BFLY_EUNSUPPORTED;
    }
    *sm_count = p.multiProcessorCount;
    return BFLY_OK;
}

// Workspace hand-over between streams: a call on another stream than the previous workspace-using
// call first waits for that call's work (the workspace is one set of buffers per bank).
static int ws_begin(bfly_bank *b, cudaStream_t st)
{
    if (b->ws_valid && b->ws_stream != st) BFLY_CUDA(cudaStreamWaitEvent(st, b->ws_event, 0));
    return BFLY_OK;
}
static int ws_end(bfly_bank *b, cudaStream_t st)
{
    BFLY_CUDA(cudaEventRecord(b->ws_event, st));
    b->ws_stream = st;
    b->ws_valid = 1;
    return BFLY_OK;
}

#define BFLY_ENTER(bank_)                                                                  \
    DeviceGuard dev_guard__((bank_)->device);                                              \
    if (dev_guard__.err != cudaSuccess) return cuda_fail(dev_guard__.err, "cudaSetDevice")
#define BFLY_LOCK(bank_)                                                                   \
    BankLock bank_lock__(bank_);                                                           \
    if (!bank_lock__.held) {                                                               \
        set_error("the bank is in use by another call (one call at a time per bank)");     \
        return BFLY_EINVAL;                                                                \
    }

template <typename T>
static int grow(T **ptr, int64_t *cap, int64_t need)
{
    if (need <= *cap) return BFLY_OK;
    if (*ptr) {
        BFLY_CUDA(cudaFree(*ptr));
        *ptr = nullptr;
        *cap = 0;
    }
    BFLY_CUDA(cudaMalloc((void **)ptr, sizeof(T) * (size_t)need));
    *cap = need;
    return BFLY_OK;
}

static int reserve_for(bfly_bank *b, int64_t n_samples)
{
    if (n_samples < b->L) return BFLY_OK;
    const int64_t n_lags = n_samples - b->L + 1;
    int rc = grow(&b->rn2, &b->rn2_cap, n_lags);
    if (rc) return rc;
    if ((rc = grow(&b->xspec, &b->xspec_cap, fft_blocks_needed(b->L, n_lags) * FFT_B))) return rc;
    const int64_t nb = tc_blocks_needed(n_lags);
    if ((rc = grow(&b->xh, &b->xh_cap, nb * 2 * FFT_B))) return rc;
    if ((rc = grow(&b->rn2p, &b->rn2p_cap, nb * (FFT_B / 2)))) return rc;
    return grow(&b->qs, &b->qs_cap, nb);
}

// the same for n_seg equal-length segments in one launch (launch_fft_tc_multi)
static int reserve_for_multi(bfly_bank *b, int64_t n_samples, int n_seg)
{
    int rc = reserve_for(b, n_samples);
    if (rc || n_samples < b->L) return rc;
    const int64_t n_lags = n_samples - b->L + 1, nb = tc_blocks_needed(n_lags);
    if ((rc = grow(&b->rn2, &b->rn2_cap, n_seg * n_lags))) return rc;
    if ((rc = grow(&b->xh, &b->xh_cap, n_seg * nb * 2 * FFT_B))) return rc;
    if ((rc = grow(&b->rn2p, &b->rn2p_cap, n_seg * nb * (FFT_B / 2)))) return rc;
    return grow(&b->qs, &b->qs_cap, n_seg * nb);
}

}  // namespace bfly

using namespace bfly;

extern "C" {

const char *bfly_strerror(int status)
{
    switch (status) {
        case BFLY_OK: return "ok";
        case BFLY_EINVAL: return "invalid argument";
        case BFLY_ENOMEM: return "out of memory";
        case BFLY_ECUDA: return "CUDA error";
        case BFLY_EUNSUPPORTED: return "unsupported device or form (sm_100a required, no CPU fallback)";
        case BFLY_ERANGE: return "size out of the supported range";
        default: return "unknown status";
    }
}

const char *bfly_last_error(void) { return g_err; }

int64_t bfly_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

void bfly_free_bank(bfly_bank *b)
{
    if (!b) return;
    DeviceGuard guard(b->device);
    cudaFree(b->f0); cudaFree(b->f1); cudaFree(b->f2); cudaFree(b->phA); cudaFree(b->phB); cudaFree(b->phC);
    cudaFree(b->inc2); cudaFree(b->ins2); cudaFree(b->rn2); cudaFree(b->xspec);
    cudaFree(b->xh); cudaFree(b->rn2p); cudaFree(b->qs);
    cudaFree(b->ys); cudaFree(b->rn2s); cudaFree(b->maxbits); cudaFree(b->racf); cudaFree(b->wspec);
    cudaFree(b->s_finf); cudaFree(b->s_delta); cudaFree(b->s_tc);
    cudaFree(b->packed); cudaFree(b->x_stage); cudaFree(b->rho_stage); cudaFree(b->arg_stage);
    cudaFree(b->rho_multi); cudaFree(b->arg_multi);
    cudaFree(b->map_stage); cudaFree(b->cnt_stage);
    if (b->ws_event) cudaEventDestroy(b->ws_event);
    if (b->ev_start) cudaEventDestroy(b->ev_start);
    if (b->ev_stop) cudaEventDestroy(b->ev_stop);
    delete b;
}

int64_t bfly_bank_size(const bfly_bank *b) { return b ? b->T : -1; }

int bfly_make_bank(double fs_hz, int32_t L, int64_t n_templates, const double *f0_hz,
                   const double *f1_hzps, int device, bfly_bank **out_bank)
{
    return bfly_make_bank3(fs_hz, L, n_templates, f0_hz, f1_hzps, nullptr, device, out_bank);
}

int bfly_make_bank3(double fs_hz, int32_t L, int64_t n_templates, const double *f0_hz,
                    const double *f1_hzps, const double *f2_hzps2, int device, bfly_bank **out_bank)
{
    if (!out_bank || !f0_hz || !f1_hzps) { set_error("null pointer"); return BFLY_EINVAL; }
    if (!(fs_hz > 0.0) || !std::isfinite(fs_hz)) { set_error("fs must be finite and > 0"); return BFLY_EINVAL; }
    if (L < 2) { set_error("L must be >= 2"); return BFLY_EINVAL; }
    if (L > FFT_MAX_L) { set_error("L = %d exceeds the supported maximum %d", L, FFT_MAX_L); return BFLY_ERANGE; }
    if (n_templates < 1) { set_error("n_templates must be >= 1"); return BFLY_EINVAL; }
    for (int64_t j = 0; j < n_templates; ++j)
        if (!std::isfinite(f0_hz[j]) || !std::isfinite(f1_hzps[j]) || (f2_hzps2 && !std::isfinite(f2_hzps2[j]))) {
            set_error("template %lld has a non-finite f0, f1 or f2", (long long)j);
            return BFLY_EINVAL;
        }
    int sms = 0;
    int rc = select_device(device, &sms);
    if (rc) return rc;
    DeviceGuard guard(device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
    bfly_bank *b = new (std::nothrow) bfly_bank();
    if (!b) { set_error("host allocation failed"); return BFLY_ENOMEM; }
    memset(b, 0, sizeof(*b));
    b->device = device; b->sm_count = sms; b->fs = fs_hz; b->L = L; b->T = n_templates;
    const size_t T = (size_t)n_templates;
    cudaError_t e;
#define BANK_TRY(call) if ((e = (call)) != cudaSuccess) { rc = cuda_fail(e, #call); bfly_free_bank(b); return rc; }
    BANK_TRY(cudaEventCreateWithFlags(&b->ws_event, cudaEventDisableTiming));
    BANK_TRY(cudaMalloc((void **)&b->f0, T * sizeof(double)));
    BANK_TRY(cudaMalloc((void **)&b->f1, T * sizeof(double)));
    BANK_TRY(cudaMalloc((void **)&b->phA, T * sizeof(uint64_t)));
    BANK_TRY(cudaMalloc((void **)&b->phB, T * sizeof(uint64_t)));
    BANK_TRY(cudaMalloc((void **)&b->f2, T * sizeof(double)));
    BANK_TRY(cudaMalloc((void **)&b->phC, T * sizeof(uint64_t)));
    BANK_TRY(cudaMalloc((void **)&b->inc2, T * sizeof(float)));
    BANK_TRY(cudaMalloc((void **)&b->ins2, T * sizeof(float)));
    BANK_TRY(cudaMalloc((void **)&b->packed, T * sizeof(unsigned long long)));
    BANK_TRY(cudaMalloc((void **)&b->rho_stage, T * sizeof(float)));
    BANK_TRY(cudaMalloc((void **)&b->arg_stage, T * sizeof(int32_t)));
    BANK_TRY(cudaMalloc((void **)&b->cnt_stage, 2 * sizeof(unsigned long long)));
    BANK_TRY(cudaMemcpy(b->f0, f0_hz, T * sizeof(double), cudaMemcpyHostToDevice));
    BANK_TRY(cudaMemcpy(b->f1, f1_hzps, T * sizeof(double), cudaMemcpyHostToDevice));
    if (f2_hzps2) {
        BANK_TRY(cudaMemcpy(b->f2, f2_hzps2, T * sizeof(double), cudaMemcpyHostToDevice));
        for (int64_t j = 0; j < n_templates && !b->has_f2; ++j) b->has_f2 = f2_hzps2[j] != 0.0;
    }
    else { BANK_TRY(cudaMemset(b->f2, 0, T * sizeof(double))); }
#undef BANK_TRY
    rc = launch_bank_params(b, 0);
    if (rc == BFLY_OK) {
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) rc = cuda_fail(e, "bank parameter kernel");
    }
    if (rc) { bfly_free_bank(b); return rc; }
    *out_bank = b;
    return BFLY_OK;
}

int bfly_bank_family(const bfly_bank *b) { return b ? b->family : -1; }

int bfly_make_bank_settle(double fs_hz, int32_t L, int64_t n_templates, const double *f_inf_hz,
                          const double *delta_hz, const double *tau_c_s, int device, bfly_bank **out_bank)
{
    if (!out_bank || !f_inf_hz || !delta_hz || !tau_c_s) { set_error("null pointer"); return BFLY_EINVAL; }
    if (!(fs_hz > 0.0) || !std::isfinite(fs_hz)) { set_error("fs must be finite and > 0"); return BFLY_EINVAL; }
    if (L < 2) { set_error("L must be >= 2"); return BFLY_EINVAL; }
    if (L > FFT_MAX_L) { set_error("L = %d exceeds the supported maximum %d", L, FFT_MAX_L); return BFLY_ERANGE; }
    if (n_templates < 1) { set_error("n_templates must be >= 1"); return BFLY_EINVAL; }
    std::vector<double> f0, f1, f2;
    try { f0.resize((size_t)n_templates); f1.resize((size_t)n_templates); f2.resize((size_t)n_templates); }
    catch (...) { set_error("host allocation failed"); return BFLY_ENOMEM; }
    for (int64_t j = 0; j < n_templates; ++j) {
        const double fi = f_inf_hz[j], d = delta_hz[j], tc = tau_c_s[j];
        if (!std::isfinite(fi) || !std::isfinite(d) || !std::isfinite(tc) || !(tc > 0.0) ||
            !std::isfinite(d * tc) || !std::isfinite(1.0 / (fs_hz * tc))) {
            set_error("template %lld: f_inf, D must be finite and tc finite and > 0", (long long)j);
            return BFLY_EINVAL;
        }
        f0[(size_t)j] = fi + d;              // frequency, slope and curvature at the first sample
        f1[(size_t)j] = -d / tc;
        f2[(size_t)j] = d / (tc * tc);
    }
    // the polynomial bank of the first-sample Taylor coefficients carries f0/f1/f2 (map frequency,
    // bfly_bank_get); its phase constants and norms are then replaced by the settling family's
    bfly_bank *b = nullptr;
    int rc = bfly_make_bank3(fs_hz, L, n_templates, f0.data(), f1.data(), f2.data(), device, &b);
    if (rc) return rc;
    DeviceGuard guard(device);
    const size_t bytes = (size_t)n_templates * sizeof(double);
    cudaError_t e;
#define SETTLE_TRY(call) if ((e = (call)) != cudaSuccess) { rc = cuda_fail(e, #call); bfly_free_bank(b); return rc; }
    SETTLE_TRY(cudaMalloc((void **)&b->s_finf, bytes));
    SETTLE_TRY(cudaMalloc((void **)&b->s_delta, bytes));
    SETTLE_TRY(cudaMalloc((void **)&b->s_tc, bytes));
    SETTLE_TRY(cudaMemcpy(b->s_finf, f_inf_hz, bytes, cudaMemcpyHostToDevice));
    SETTLE_TRY(cudaMemcpy(b->s_delta, delta_hz, bytes, cudaMemcpyHostToDevice));
    SETTLE_TRY(cudaMemcpy(b->s_tc, tau_c_s, bytes, cudaMemcpyHostToDevice));
#undef SETTLE_TRY
    b->family = BFLY_FAMILY_SETTLE;
    b->has_f2 = 0;
    rc = launch_bank_params_settle(b, 0);
    if (rc == BFLY_OK) {
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) rc = cuda_fail(e, "settle bank parameter kernel");
    }
    if (rc) { bfly_free_bank(b); return rc; }
    *out_bank = b;
    return BFLY_OK;
}

int bfly_bank_get_settle(const bfly_bank *b, int64_t first, int64_t count, double *f_inf_hz,
                         double *delta_hz, double *tau_c_s)
{
    if (!b) { set_error("null bank"); return BFLY_EINVAL; }
    if (b->family != BFLY_FAMILY_SETTLE) { set_error("not a settling-family bank"); return BFLY_EINVAL; }
    if (first < 0 || count < 0 || first + count > b->T) { set_error("template range outside the bank"); return BFLY_EINVAL; }
    BFLY_ENTER(b);
    const size_t n = (size_t)count * sizeof(double);
    if (f_inf_hz) BFLY_CUDA(cudaMemcpy(f_inf_hz, b->s_finf + first, n, cudaMemcpyDeviceToHost));
    if (delta_hz) BFLY_CUDA(cudaMemcpy(delta_hz, b->s_delta + first, n, cudaMemcpyDeviceToHost));
    if (tau_c_s) BFLY_CUDA(cudaMemcpy(tau_c_s, b->s_tc + first, n, cudaMemcpyDeviceToHost));
    return BFLY_OK;
}

int bfly_make_bank_grid(double fs_hz, int32_t L, double f0_lo, double f0_hi, int32_t n_f0,
                        double f1_lo, double f1_hi, int32_t n_f1, int device, bfly_bank **out_bank)
{
    if (n_f0 < 1 || n_f1 < 1) { set_error("grid sizes must be >= 1"); return BFLY_EINVAL; }
    if (!std::isfinite(f0_lo) || !std::isfinite(f0_hi) || !std::isfinite(f1_lo) || !std::isfinite(f1_hi)) {
        set_error("grid bounds must be finite"); return BFLY_EINVAL;
    }
    const int64_t T = (int64_t)n_f0 * n_f1;
    std::vector<double> f0, f1;
    try { f0.resize((size_t)T); f1.resize((size_t)T); }
    catch (...) { set_error("host allocation failed"); return BFLY_ENOMEM; }
    // numpy.linspace: start + i * step with step = (stop - start) / (n - 1); last point = stop
    const double s0 = n_f0 > 1 ? (f0_hi - f0_lo) / (double)(n_f0 - 1) : 0.0;
    const double s1 = n_f1 > 1 ? (f1_hi - f1_lo) / (double)(n_f1 - 1) : 0.0;
    for (int32_t i = 0; i < n_f0; ++i) {
        const double a = (n_f0 > 1 && i == n_f0 - 1) ? f0_hi : f0_lo + (double)i * s0;
        for (int32_t k = 0; k < n_f1; ++k) {
            const double c = (n_f1 > 1 && k == n_f1 - 1) ? f1_hi : f1_lo + (double)k * s1;
            f0[(size_t)i * n_f1 + k] = a;
            f1[(size_t)i * n_f1 + k] = c;
        }
    }
    return bfly_make_bank(fs_hz, L, T, f0.data(), f1.data(), device, out_bank);
}

int bfly_bank_get(const bfly_bank *b, int64_t first, int64_t count, double *f0_hz,
                  double *f1_hzps, float *inv_nc2, float *inv_ns2)
{
    if (!b) { set_error("null bank"); return BFLY_EINVAL; }
    if (first < 0 || count < 0 || first + count > b->T) { set_error("template range outside the bank"); return BFLY_EINVAL; }
    BFLY_ENTER(b);
    const size_t n = (size_t)count;
    if (f0_hz) BFLY_CUDA(cudaMemcpy(f0_hz, b->f0 + first, n * sizeof(double), cudaMemcpyDeviceToHost));
    if (f1_hzps) BFLY_CUDA(cudaMemcpy(f1_hzps, b->f1 + first, n * sizeof(double), cudaMemcpyDeviceToHost));
    if (inv_nc2) BFLY_CUDA(cudaMemcpy(inv_nc2, b->inc2 + first, n * sizeof(float), cudaMemcpyDeviceToHost));
    if (inv_ns2) BFLY_CUDA(cudaMemcpy(inv_ns2, b->ins2 + first, n * sizeof(float), cudaMemcpyDeviceToHost));
    return BFLY_OK;
}

int bfly_bank_get_f2(const bfly_bank *b, int64_t first, int64_t count, double *f2_hzps2)
{
    if (!b || !f2_hzps2) { set_error("null pointer"); return BFLY_EINVAL; }
    if (first < 0 || count < 0 || first + count > b->T) { set_error("template range outside the bank"); return BFLY_EINVAL; }
    BFLY_ENTER(b);
    BFLY_CUDA(cudaMemcpy(f2_hzps2, b->f2 + first, (size_t)count * sizeof(double), cudaMemcpyDeviceToHost));
    return BFLY_OK;
}

int bfly_bank_reserve(bfly_bank *b, int64_t max_n_samples)
{
    if (!b) { set_error("null bank"); return BFLY_EINVAL; }
    if (max_n_samples < b->L) { set_error("max_n_samples < L"); return BFLY_EINVAL; }
    if (max_n_samples >= (1LL << 31)) { set_error("segment too long"); return BFLY_ERANGE; }
    BFLY_ENTER(b);
    BFLY_LOCK(b);
    if (b->ws_valid) BFLY_CUDA(cudaEventSynchronize(b->ws_event));   // buffers may be freed below
    return reserve_for(b, max_n_samples);
}

int bfly_bank_set_timing(bfly_bank *b, int enable)
{
    if (!b) { set_error("null bank"); return BFLY_EINVAL; }
    BFLY_ENTER(b);
    if (enable && !b->ev_start) {
        BFLY_CUDA(cudaEventCreate(&b->ev_start));
        BFLY_CUDA(cudaEventCreate(&b->ev_stop));
    }
    b->timing = enable ? 1 : 0;
    b->timed = 0;
    return BFLY_OK;
}

int bfly_bank_core_ms(bfly_bank *b, float *ms_out)
{
    if (!b || !ms_out) { set_error("null pointer"); return BFLY_EINVAL; }
    if (!b->timing || !b->timed) { set_error("no timed bfly_correlate call on this bank"); return BFLY_EINVAL; }
    BFLY_ENTER(b);
    BFLY_CUDA(cudaEventSynchronize(b->ev_stop));
    BFLY_CUDA(cudaEventElapsedTime(ms_out, b->ev_start, b->ev_stop));
    return BFLY_OK;
}

// Argument checks of bfly_correlate_form (before any device work); resolves BFLY_FORM_DEFAULT.
static int correlate_check(const bfly_bank *bank, int *form_io, const float *x_dev, int64_t n_samples,
                           int64_t lag_begin, int64_t lag_end, const float *rho_max_dev,
                           const int32_t *arg_lag_dev)
{
    int form = *form_io;
    if (!bank || !x_dev || !rho_max_dev || !arg_lag_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_samples < bank->L) { set_error("n_samples < L"); return BFLY_EINVAL; }
    if (n_samples >= (1LL << 31)) { set_error("segment too long (n_samples must be < 2^31)"); return BFLY_ERANGE; }
    if (lag_begin < 0 || lag_end < lag_begin || lag_end > n_samples - bank->L + 1) {
        set_error("lag range [%lld, %lld) outside the valid lags [0, %lld)", (long long)lag_begin,
                  (long long)lag_end, (long long)(n_samples - bank->L + 1));
        return BFLY_EINVAL;
    }
    // the tensor-core form needs templates long enough for its fp16 rounding errors to average
    // out; shorter ones go to the fp32 FFT form
    if (form == BFLY_FORM_DEFAULT) form = bank->L >= BFLY_TC_MIN_L ? BFLY_FORM_FFT_TC : BFLY_FORM_FFT;
    if ((form == BFLY_FORM_FFT_TC || form == BFLY_FORM_DENSE_TC || form == BFLY_FORM_FFT_TC5) && bank->L < BFLY_TC_MIN_L) {
        set_error("the fp16-operand forms need L >= %d (L = %d)", BFLY_TC_MIN_L, bank->L);
        return BFLY_EUNSUPPORTED;
    }
    if (form != BFLY_FORM_FFT && form != BFLY_FORM_DIRECT && form != BFLY_FORM_FFT_TC && form != BFLY_FORM_DENSE_TC &&
        form != BFLY_FORM_FFT_TC5) { set_error("unknown form %d", form); return BFLY_EUNSUPPORTED; }
    *form_io = form;
    return BFLY_OK;
}

// bfly_correlate_form with the arguments checked, the device selected and the bank locked
static int correlate_locked(const bfly_bank *bank, int form, const float *x_dev, int64_t n_samples,
                            int64_t lag_begin, int64_t lag_end, float *rho_max_dev,
                            int32_t *arg_lag_dev, void *stream)
{
    bfly_bank *b = const_cast<bfly_bank *>(bank);   // the workspace is mutable state of the bank
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ws_begin(b, st);
    if (rc) return rc;
    if ((rc = reserve_for(b, n_samples))) return rc;
    rc = launch_sliding_norm(x_dev, n_samples, b->L, lag_begin, lag_end - lag_begin, b->rn2, st);
    if (rc) return rc;
    if (form == BFLY_FORM_DIRECT)
        rc = launch_direct(b, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev, st);
    else if (form == BFLY_FORM_DENSE_TC)
        rc = launch_dense_tc(b, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev, st);
    else if (form == BFLY_FORM_FFT)
        rc = launch_fft(b, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev, st);
    else if (form == BFLY_FORM_FFT_TC5)
        rc = launch_fft_tc5(b, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev, st);
    else
        rc = launch_fft_tc(b, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev, st);
    if (rc) return rc;
    return ws_end(b, st);
}

// n_seg <= 4 segments of equal length, the same lag range in each, arguments checked, bank locked:
// one launch of the default form when every lag comes from a transform, else one call per segment
static int correlate_multi_locked(const bfly_bank *bank, int n_seg, const float *const *x_dev, int64_t n_samples,
                                  int64_t lag_begin, int64_t lag_end, float *const *rho_max_dev,
                                  int32_t *const *arg_lag_dev, void *stream)
{
    bfly_bank *b = const_cast<bfly_bank *>(bank);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n_lags = lag_end - lag_begin;
    if (n_seg < 2 || !tc_multi_supported(b->L, n_lags)) {
        const int form = b->L >= BFLY_TC_MIN_L ? BFLY_FORM_FFT_TC : BFLY_FORM_FFT;
        for (int sg = 0; sg < n_seg; ++sg) {
            const int rc = correlate_locked(bank, form, x_dev[sg], n_samples, lag_begin, lag_end, rho_max_dev[sg],
                                            arg_lag_dev[sg], stream);
            if (rc) return rc;
        }
        return BFLY_OK;
    }
    int rc = ws_begin(b, st);
    if (rc) return rc;
    if ((rc = reserve_for_multi(b, n_samples, n_seg))) return rc;
    for (int sg = 0; sg < n_seg; ++sg)
        if ((rc = launch_sliding_norm(x_dev[sg], n_samples, b->L, lag_begin, n_lags, b->rn2 + (int64_t)sg * n_lags, st)))
            return rc;
    if ((rc = launch_fft_tc_multi(b, n_seg, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev, st))) return rc;
    return ws_end(b, st);
}

int bfly_correlate_multi(const bfly_bank *bank, int32_t n_segments, const float *const *x_dev, int64_t n_samples,
                         int64_t lag_begin, int64_t lag_end, float *const *rho_max_dev,
                         int32_t *const *arg_lag_dev, void *stream)
{
    if (!bank || !x_dev || !rho_max_dev || !arg_lag_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_segments < 1) { set_error("n_segments must be >= 1"); return BFLY_EINVAL; }
    for (int32_t sg = 0; sg < n_segments; ++sg) {
        int form = BFLY_FORM_DEFAULT;
        const int rc = correlate_check(bank, &form, x_dev[sg], n_samples, lag_begin, lag_end, rho_max_dev[sg], arg_lag_dev[sg]);
        if (rc) return rc;
    }
    BFLY_ENTER(bank);
    BFLY_LOCK(bank);
    for (int32_t s0 = 0; s0 < n_segments; s0 += 4) {
        const int g = n_segments - s0 < 4 ? n_segments - s0 : 4;
        const int rc = correlate_multi_locked(bank, g, x_dev + s0, n_samples, lag_begin, lag_end, rho_max_dev + s0,
                                              arg_lag_dev + s0, stream);
        if (rc) return rc;
    }
    return BFLY_OK;
}

int bfly_correlate_form(const bfly_bank *bank, int form, const float *x_dev, int64_t n_samples,
                        int64_t lag_begin, int64_t lag_end, float *rho_max_dev,
                        int32_t *arg_lag_dev, void *stream)
{
    int rc = correlate_check(bank, &form, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev);
    if (rc) return rc;
    BFLY_ENTER(bank);
    BFLY_LOCK(bank);
    return correlate_locked(bank, form, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev,
                            stream);
}

int bfly_tails(const bfly_bank *bank, const float *x_dev, int64_t n_samples, int64_t lag_begin,
               int64_t lag_end, float kappa, float *sigma_dev, int64_t capacity,
               int32_t *hit_template_dev, int32_t *hit_lag_dev, float *hit_rho_dev,
               uint64_t *n_hits_dev, void *stream)
{
    if (!bank || !x_dev || !sigma_dev || !n_hits_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (capacity < 0 || (capacity > 0 && (!hit_template_dev || !hit_lag_dev || !hit_rho_dev))) {
        set_error("hit list arrays missing for capacity %lld", (long long)capacity);
        return BFLY_EINVAL;
    }
    if (!std::isfinite(kappa) || !(kappa > 0.0f)) { set_error("kappa must be finite and > 0"); return BFLY_EINVAL; }
    if (n_samples < bank->L) { set_error("n_samples < L"); return BFLY_EINVAL; }
    if (n_samples >= (1LL << 31)) { set_error("segment too long (n_samples must be < 2^31)"); return BFLY_ERANGE; }
    if (lag_begin < 0 || lag_end < lag_begin || lag_end > n_samples - bank->L + 1) {
        set_error("lag range [%lld, %lld) outside the valid lags [0, %lld)", (long long)lag_begin,
                  (long long)lag_end, (long long)(n_samples - bank->L + 1));
        return BFLY_EINVAL;
    }
    if (bank->L < BFLY_TC_MIN_L) {
        set_error("bfly_tails needs L >= %d (L = %d)", BFLY_TC_MIN_L, bank->L);
        return BFLY_EUNSUPPORTED;
    }
    bfly_bank *b = const_cast<bfly_bank *>(bank);
    BFLY_ENTER(b);
    BFLY_LOCK(b);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ws_begin(b, st);
    if (rc) return rc;
    if ((rc = reserve_for(b, n_samples))) return rc;
    if (!b->racf) BFLY_CUDA(cudaMalloc((void **)&b->racf, sizeof(double) * FFT_MAX_L));
    if (!b->wspec) BFLY_CUDA(cudaMalloc((void **)&b->wspec, sizeof(float) * FFT_B));
    // rn2 serves the direct tail lags of the kernel's geometry in the other mode; not needed here
    rc = launch_tails_tc(b, x_dev, n_samples, lag_begin, lag_end, kappa, sigma_dev, capacity,
                         hit_template_dev, hit_lag_dev, hit_rho_dev,
                         (unsigned long long *)n_hits_dev, st);
    if (rc) return rc;
    return ws_end(b, st);
}

int bfly_hits_map(const bfly_bank *bank, const int32_t *hit_template_dev, const int32_t *hit_lag_dev,
                  int64_t n_hits, int64_t lag_origin, int32_t samples_per_tbin, double f_lo_hz,
                  double df_hz, int32_t n_fbins, int32_t n_tbins, uint32_t *map_dev,
                  uint64_t *counters_dev, void *stream)
{
    if (!bank || !map_dev || !counters_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_hits < 0 || (n_hits > 0 && (!hit_template_dev || !hit_lag_dev))) { set_error("bad hit list"); return BFLY_EINVAL; }
    if (!(df_hz > 0.0) || !std::isfinite(df_hz) || !std::isfinite(f_lo_hz)) { set_error("df must be finite and > 0, f_lo finite"); return BFLY_EINVAL; }
    if (samples_per_tbin <= 0 || n_fbins <= 0 || n_tbins <= 0 || lag_origin < 0) { set_error("bad map geometry"); return BFLY_EINVAL; }
    BFLY_ENTER(bank);
    return launch_hits_map(bank, hit_template_dev, hit_lag_dev, n_hits, lag_origin, samples_per_tbin,
                           f_lo_hz, df_hz, n_fbins, n_tbins, map_dev, (unsigned long long *)counters_dev,
                           (cudaStream_t)stream);
}

static int current_device_ok()
{
    int dev = 0;
    BFLY_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp p;
    BFLY_CUDA(cudaGetDeviceProperties(&p, dev));
    if (p.major != 10) { set_error("device %d is sm_%d%d; this library is built for sm_100a only", dev, p.major, p.minor); return BFLY_EUNSUPPORTED; }
    return BFLY_OK;
}

int bfly_time_randomize(const float *x_dev, const int32_t *perm_dev, int64_t n, float *out_dev,
                        int32_t *bad_dev, void *stream)
{
    if (!x_dev || !perm_dev || !out_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n < 0 || n >= (1LL << 31)) { set_error("n must be in [0, 2^31)"); return BFLY_EINVAL; }
    if (x_dev == out_dev) { set_error("out_dev must not alias x_dev"); return BFLY_EINVAL; }
    int rc = current_device_ok();
    if (rc) return rc;
    return launch_time_randomize(x_dev, perm_dev, n, out_dev, bad_dev, (cudaStream_t)stream);
}

int bfly_coincidence(const uint32_t *map1_dev, const uint32_t *map2_dev, int32_t n_tbins,
                     int32_t n_fbins, int32_t half_width_bins, uint32_t *co1_dev,
                     uint32_t *co2_dev, void *stream)
{
    if (!map1_dev || !map2_dev || !co1_dev || !co2_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_tbins <= 0 || n_fbins <= 0 || half_width_bins < 0) { set_error("bad map geometry or window"); return BFLY_EINVAL; }
    if (co1_dev == map1_dev || co1_dev == map2_dev || co2_dev == map1_dev || co2_dev == map2_dev || co1_dev == co2_dev) {
        set_error("outputs must not alias the inputs or each other");
        return BFLY_EINVAL;
    }
    int rc = current_device_ok();
    if (rc) return rc;
    return launch_coincidence(map1_dev, map2_dev, n_tbins, n_fbins, half_width_bins, co1_dev, co2_dev,
                              (cudaStream_t)stream);
}

int bfly_pseudo_spectrum(const uint32_t *map_dev, int32_t n_tbins, int32_t n_fbins,
                         uint64_t *spectrum_dev, void *stream)
{
    if (!map_dev || !spectrum_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_tbins <= 0 || n_fbins <= 0) { set_error("bad map geometry"); return BFLY_EINVAL; }
    int rc = current_device_ok();
    if (rc) return rc;
    return launch_pseudo_spectrum(map_dev, n_tbins, n_fbins, (unsigned long long *)spectrum_dev,
                                  (cudaStream_t)stream);
}

int bfly_debug_fft_tc(const float *y_dev, float *z_dev, int full, void *stream)
{
    if (!y_dev || !z_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    return launch_debug_fft_tc(reinterpret_cast<const float2 *>(y_dev),
                               reinterpret_cast<float2 *>(z_dev), full, (cudaStream_t)stream);
}

int bfly_debug_fft_tc5(const float *y_dev, float *z_dev, int32_t n_pairs, int32_t reps, int64_t *cycles_dev,
                       void *stream)
{
    if (!y_dev || !z_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_pairs < 1 || reps < 1) { set_error("n_pairs and reps must be >= 1"); return BFLY_EINVAL; }
    int rc = current_device_ok();
    if (rc) return rc;
    return launch_debug_fft_tc5(reinterpret_cast<const float2 *>(y_dev), reinterpret_cast<float2 *>(z_dev),
                                n_pairs, reps, reinterpret_cast<long long *>(cycles_dev), (cudaStream_t)stream);
}

int bfly_correlate(const bfly_bank *bank, const float *x_dev, int64_t n_samples, int64_t lag_begin,
                   int64_t lag_end, float *rho_max_dev, int32_t *arg_lag_dev, void *stream)
{
    return bfly_correlate_form(bank, BFLY_FORM_DEFAULT, x_dev, n_samples, lag_begin, lag_end,
                               rho_max_dev, arg_lag_dev, stream);
}

// The default form with its scratch in a static device array: allocates nothing (no cudaMalloc, no
// cudaFree, no allocating library call), touches no state of the bank, takes no bank lock.
int bfly_correlate_static(const bfly_bank *bank, const float *x_dev, int64_t n_samples, int64_t lag_begin,
                          int64_t lag_end, float *rho_max_dev, int32_t *arg_lag_dev, void *stream)
{
    int form = BFLY_FORM_FFT_TC;
    int rc = correlate_check(bank, &form, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev);
    if (rc) return rc;
    if (n_samples > BFLY_STATIC_MAX_SAMPLES) {
        set_error("bfly_correlate_static: n_samples = %lld exceeds BFLY_STATIC_MAX_SAMPLES = %d (the static scratch "
                  "array holds one segment of that size; use bfly_correlate)", (long long)n_samples,
                  (int)BFLY_STATIC_MAX_SAMPLES);
        return BFLY_ERANGE;
    }
    BFLY_ENTER(bank);
    return launch_fft_tc_static(bank, x_dev, n_samples, lag_begin, lag_end, rho_max_dev, arg_lag_dev,
                                (cudaStream_t)stream);
}

int bfly_butterfly_map(const bfly_bank *bank, const float *rho_max_dev, const int32_t *arg_lag_dev,
                       float kappa, int64_t lag_origin, int32_t samples_per_tbin, double f_lo_hz,
                       double df_hz, int32_t n_fbins, int32_t n_tbins, uint32_t *map_dev,
                       uint64_t *counters_dev, void *stream)
{
    if (!bank || !rho_max_dev || !arg_lag_dev || !map_dev || !counters_dev) { set_error("null pointer"); return BFLY_EINVAL; }
    if (!std::isfinite(kappa)) { set_error("kappa must be finite"); return BFLY_EINVAL; }
    if (!(df_hz > 0.0) || !std::isfinite(df_hz) || !std::isfinite(f_lo_hz)) { set_error("df must be finite and > 0, f_lo finite"); return BFLY_EINVAL; }
    if (samples_per_tbin <= 0 || n_fbins <= 0 || n_tbins <= 0 || lag_origin < 0) { set_error("bad map geometry"); return BFLY_EINVAL; }
    BFLY_ENTER(bank);
    return launch_map(bank, rho_max_dev, arg_lag_dev, kappa, lag_origin, samples_per_tbin, f_lo_hz,
                      df_hz, n_fbins, n_tbins, map_dev, (unsigned long long *)counters_dev,
                      (cudaStream_t)stream);
}

int bfly_search_host(bfly_bank *b, const float *x_host, int64_t n_samples, int64_t chunk_samples,
                     float kappa, int32_t samples_per_tbin, double f_lo_hz, double df_hz,
                     int32_t n_fbins, int32_t n_tbins, float *rho_max_host, int32_t *arg_lag_host,
                     uint32_t *map_host, uint64_t *counters_host, void *stream)
{
    if (!b || !x_host) { set_error("null pointer"); return BFLY_EINVAL; }
    if (n_samples < b->L) { set_error("n_samples < L"); return BFLY_EINVAL; }
    if (!std::isfinite(kappa) || !(df_hz > 0.0) || !std::isfinite(df_hz) || !std::isfinite(f_lo_hz) ||
        samples_per_tbin <= 0 || n_fbins <= 0 || n_tbins <= 0) { set_error("bad threshold or map geometry"); return BFLY_EINVAL; }
    if (chunk_samples <= 0 || chunk_samples > n_samples) chunk_samples = n_samples;
    if (chunk_samples <= b->L && chunk_samples < n_samples) { set_error("chunk_samples must exceed L"); return BFLY_EINVAL; }
    if (chunk_samples >= (1LL << 31)) { set_error("chunk too long"); return BFLY_ERANGE; }
    BFLY_ENTER(b);
    BFLY_LOCK(b);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ws_begin(b, st);
    if (rc) return rc;
    if ((rc = reserve_for(b, chunk_samples))) return rc;
    if ((rc = grow(&b->x_stage, &b->x_stage_cap, chunk_samples))) return rc;
    const int64_t cells = (int64_t)n_fbins * n_tbins;
    if ((rc = grow(&b->map_stage, &b->map_stage_cap, cells))) return rc;
    BFLY_CUDA(cudaMemsetAsync(b->map_stage, 0, sizeof(uint32_t) * (size_t)cells, st));
    BFLY_CUDA(cudaMemsetAsync(b->cnt_stage, 0, 2 * sizeof(unsigned long long), st));
    const int64_t total_lags = n_samples - b->L + 1;
    // a single chunk takes every valid lag; otherwise hop = chunk - L (reading C11)
    const int64_t hop = (chunk_samples >= n_samples) ? total_lags : chunk_samples - b->L;
    // Consecutive chunks of equal length and equal lag range go through one launch, up to four at
    // a time (bfly_correlate_multi: synthesis and the transform of g once per template for all of
    // them); results and map are those of chunk-by-chunk calls, bit for bit.
    const int64_t n_chunks = (total_lags + hop - 1) / hop;
    const int max_group = n_chunks >= 3 ? (n_chunks - 1 < 4 ? (int)(n_chunks - 1) : 4) : 1;   // (the last chunk is ragged)
    if (max_group > 1) {
        if ((rc = grow(&b->x_stage, &b->x_stage_cap, (int64_t)max_group * chunk_samples))) return rc;
        if ((rc = grow(&b->rho_multi, &b->rho_multi_cap, (int64_t)max_group * b->T))) return rc;
        if ((rc = grow(&b->arg_multi, &b->arg_multi_cap, (int64_t)max_group * b->T))) return rc;
        if ((rc = reserve_for_multi(b, chunk_samples, max_group))) return rc;
    }
    const float *last_rho = b->rho_stage;
    const int32_t *last_arg = b->arg_stage;
    int64_t start = 0;
    bool done = false;
    while (!done && start < total_lags) {
        int64_t starts[4], n0 = 0, lag_end0 = 0;
        int g = 0;
        for (; g < max_group && !done && start < total_lags; ++g) {
            const int64_t n = (chunk_samples < n_samples - start) ? chunk_samples : n_samples - start;
            const int64_t lags_here = n - b->L + 1;
            const bool last = start + hop >= total_lags;
            const int64_t lag_end = last ? lags_here : (hop < lags_here ? hop : lags_here);
            if (g == 0) { n0 = n; lag_end0 = lag_end; }
            else if (n != n0 || lag_end != lag_end0) break;      // another shape: next group
            starts[g] = start;
            if (last) done = true;
            start += hop;
        }
        float *rho_p[4];
        int32_t *arg_p[4];
        const float *x_p[4];
        for (int i = 0; i < g; ++i) {
            float *xs = b->x_stage + (int64_t)i * chunk_samples;
            BFLY_CUDA(cudaMemcpyAsync(xs, x_host + starts[i], sizeof(float) * (size_t)n0, cudaMemcpyHostToDevice, st));
            x_p[i] = xs;
            rho_p[i] = g > 1 ? b->rho_multi + (int64_t)i * b->T : b->rho_stage;
            arg_p[i] = g > 1 ? b->arg_multi + (int64_t)i * b->T : b->arg_stage;
        }
        int form = BFLY_FORM_DEFAULT;
        rc = correlate_check(b, &form, x_p[0], n0, 0, lag_end0, rho_p[0], arg_p[0]);
        if (rc) return rc;
        rc = correlate_multi_locked(b, g, x_p, n0, 0, lag_end0, rho_p, arg_p, st);
        if (rc) return rc;
        for (int i = 0; i < g; ++i) {
            rc = launch_map(b, rho_p[i], arg_p[i], kappa, starts[i], samples_per_tbin, f_lo_hz, df_hz,
                            n_fbins, n_tbins, b->map_stage, b->cnt_stage, st);
            if (rc) return rc;
        }
        last_rho = rho_p[g - 1];
        last_arg = arg_p[g - 1];
    }
    const size_t T = (size_t)b->T;
    if (rho_max_host) BFLY_CUDA(cudaMemcpyAsync(rho_max_host, last_rho, T * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (arg_lag_host) BFLY_CUDA(cudaMemcpyAsync(arg_lag_host, last_arg, T * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (map_host) BFLY_CUDA(cudaMemcpyAsync(map_host, b->map_stage, sizeof(uint32_t) * (size_t)cells, cudaMemcpyDeviceToHost, st));
    if (counters_host) BFLY_CUDA(cudaMemcpyAsync(counters_host, b->cnt_stage, 2 * sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
    BFLY_CUDA(cudaStreamSynchronize(st));
    return BFLY_OK;
}

}  // extern "C"
