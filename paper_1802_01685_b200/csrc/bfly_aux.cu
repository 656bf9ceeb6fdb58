// Small kernels around the correlation core: bank parameters (A1), sliding data norm (A2),
// threshold + butterfly map (A8).  None of them is on the critical path.
#include <cmath>

#include "bfly_internal.cuh"

namespace bfly {

// ---------------------------------------------------------------------------- A1
// One warp per template: fixed-point phase constants and 1/||cos phi||^2, 1/||sin phi||^2 in
// float64 (BASELINE.json configs[0]: "each unit-L2-normalized"; reading C2: separately).
__global__ void __launch_bounds__(256) bank_params_kernel(int64_t T, int32_t L, double fs,
                                                          const double *__restrict__ f0,
                                                          const double *__restrict__ f1,
                                                          const double *__restrict__ f2,
                                                          uint64_t *__restrict__ phA,
                                                          uint64_t *__restrict__ phB,
                                                          uint64_t *__restrict__ phC,
                                                          float *__restrict__ inc2,
                                                          float *__restrict__ ins2)
{
    const int lane = threadIdx.x & 31;
    const int64_t j = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (j >= T) return;
    // cycles per sample and per sample^2, reduced mod 1, as 2^-64 fixed point
    double a = f0[j] / fs;
    double b = 0.5 * f1[j] / (fs * fs);
    double c3 = f2[j] / (6.0 * fs * fs * fs);        // cycles per sample^3 (reading N1)
    c3 -= floor(c3 + 0.5);
    a -= floor(a);                       // [0, 1]  (1.0 only by rounding of a tiny negative a)
    if (a >= 1.0) a = 0.0;
    b -= floor(b + 0.5);                 // [-0.5, 0.5)
    // scaling by 2^64 is exact; a < 1 and |b| <= 0.5 keep both conversions in range
    const uint64_t A = __double2ull_rn(a * 18446744073709551616.0);
    const uint64_t B = (uint64_t)__double2ll_rn(b * 18446744073709551616.0);
    const uint64_t C = (uint64_t)__double2ll_rn(c3 * 18446744073709551616.0);
    double sc = 0.0, ss = 0.0;
    for (int32_t k = lane; k < L; k += 32) {
        const uint64_t ph = template_phase(A, B, C, (uint64_t)k);
        // signed fraction of a turn in [-0.5, 0.5): angle = 2 pi * fr
        const double fr = (double)(int64_t)ph * 5.421010862427522e-20;   // 2^-64
        double s, c;
        sincospi(2.0 * fr, &s, &c);
        sc += c * c;
        ss += s * s;
    }
    for (int o = 16; o > 0; o >>= 1) {
        sc += __shfl_xor_sync(0xffffffffu, sc, o);
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
    }
    if (lane == 0) {
        phA[j] = A;
        phB[j] = B;
        phC[j] = C;
        inc2[j] = sc > 0.0 ? (float)(1.0 / sc) : 0.0f;
        ins2[j] = ss > 0.0 ? (float)(1.0 / ss) : 0.0f;
    }
}

// The same for the settling family (reading N2): phA = f_inf/fs as 2^-64 fixed point, phB / phC =
// the bits of the doubles D tc and 1/(fs tc); norms from the same phase function the kernels use.
__global__ void __launch_bounds__(256) bank_params_settle_kernel(int64_t T, int32_t L, double fs,
                                                                 const double *__restrict__ f_inf,
                                                                 const double *__restrict__ delta,
                                                                 const double *__restrict__ tc,
                                                                 uint64_t *__restrict__ phA,
                                                                 uint64_t *__restrict__ phB,
                                                                 uint64_t *__restrict__ phC,
                                                                 float *__restrict__ inc2,
                                                                 float *__restrict__ ins2)
{
    const int lane = threadIdx.x & 31;
    const int64_t j = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (j >= T) return;
    double a = f_inf[j] / fs;
    a -= floor(a);
    if (a >= 1.0) a = 0.0;
    const uint64_t A = __double2ull_rn(a * 18446744073709551616.0);
    const double Dtc = delta[j] * tc[j], inv = 1.0 / (fs * tc[j]);
    double sc = 0.0, ss = 0.0;
    for (int32_t k = lane; k < L; k += 32) {
        const uint64_t ph = settle_phase(A, Dtc, inv, (uint64_t)k);
        const double fr = (double)(int64_t)ph * 5.421010862427522e-20;   // 2^-64
        double s, c;
        sincospi(2.0 * fr, &s, &c);
        sc += c * c;
        ss += s * s;
    }
    for (int o = 16; o > 0; o >>= 1) {
        sc += __shfl_xor_sync(0xffffffffu, sc, o);
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
    }
    if (lane == 0) {
        phA[j] = A;
        phB[j] = (uint64_t)__double_as_longlong(Dtc);
        phC[j] = (uint64_t)__double_as_longlong(inv);
        inc2[j] = sc > 0.0 ? (float)(1.0 / sc) : 0.0f;
        ins2[j] = ss > 0.0 ? (float)(1.0 / ss) : 0.0f;
    }
}

int launch_bank_params_settle(bfly_bank *b, cudaStream_t stream)
{
    const int warps = 8;
    const int64_t blocks = (b->T + warps - 1) / warps;
    if (blocks >= (1LL << 31)) { set_error("bank too large"); return BFLY_ERANGE; }
    bank_params_settle_kernel<<<(unsigned)blocks, warps * 32, 0, stream>>>(
        b->T, b->L, b->fs, b->s_finf, b->s_delta, b->s_tc, b->phA, b->phB, b->phC, b->inc2, b->ins2);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

int launch_bank_params(bfly_bank *b, cudaStream_t stream)
{
    const int warps = 8;
    const int64_t blocks = (b->T + warps - 1) / warps;
    if (blocks >= (1LL << 31)) { set_error("bank too large"); return BFLY_ERANGE; }
    bank_params_kernel<<<(unsigned)blocks, warps * 32, 0, stream>>>(b->T, b->L, b->fs, b->f0, b->f1,
                                                                    b->f2, b->phA, b->phB, b->phC,
                                                                    b->inc2, b->ins2);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

// ---------------------------------------------------------------------------- A2
// rn2[i] = 1 / sum_k x[lag_begin + i + k]^2 (0 if the window is all zero), each lag summed on
// its own in float64 (north_star: "normalized by the sliding data norm"; reading C6).
__global__ void __launch_bounds__(256) sliding_norm_kernel(const float *__restrict__ x, int32_t L,
                                                           int64_t lag_begin, int64_t n_lags,
                                                           float *__restrict__ rn2)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_lags) return;
    const float *p = x + lag_begin + i;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int32_t k = 0;
    for (; k + 4 <= L; k += 4) {
        const double v0 = (double)__ldg(p + k), v1 = (double)__ldg(p + k + 1);
        const double v2 = (double)__ldg(p + k + 2), v3 = (double)__ldg(p + k + 3);
        a0 = fma(v0, v0, a0); a1 = fma(v1, v1, a1); a2 = fma(v2, v2, a2); a3 = fma(v3, v3, a3);
    }
    for (; k < L; ++k) { const double v = (double)__ldg(p + k); a0 = fma(v, v, a0); }
    const double n2 = (a0 + a1) + (a2 + a3);
    rn2[i] = n2 > 0.0 ? (float)(1.0 / n2) : 0.0f;
}

int launch_sliding_norm(const float *x, int64_t n_samples, int32_t L, int64_t lag_begin,
                        int64_t n_lags, float *rn2, cudaStream_t stream)
{
    (void)n_samples;
    if (n_lags <= 0) return BFLY_OK;
    const int64_t blocks = (n_lags + 255) / 256;
    sliding_norm_kernel<<<(unsigned)blocks, 256, 0, stream>>>(x, L, lag_begin, n_lags, rn2);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

// ---------------------------------------------------------------------------- A8
// Threshold and count (only rho exceeding the threshold is kept;
// chirp-based spectrogram).  Reading C9 (strict >, fp32) and C10 (time = start of
// the matched window, frequency = f0).  Integer atomics: the result is order independent.
__global__ void __launch_bounds__(256) map_kernel(int64_t T, const double *__restrict__ f0,
                                                  const float *__restrict__ rho_max,
                                                  const int32_t *__restrict__ arg_lag, float kappa,
                                                  int64_t lag_origin, int32_t samples_per_tbin,
                                                  double f_lo, double df, int32_t n_fbins,
                                                  int32_t n_tbins, uint32_t *__restrict__ map,
                                                  unsigned long long *__restrict__ counters)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool hit = false, dropped = false;
    if (j < T && rho_max[j] > kappa) {
        hit = true;
        const int64_t tbin = (lag_origin + (int64_t)arg_lag[j]) / samples_per_tbin;
        const double fb = floor((f0[j] - f_lo) / df);
        if (tbin >= 0 && tbin < n_tbins && fb >= 0.0 && fb < (double)n_fbins)
            atomicAdd(&map[tbin * (int64_t)n_fbins + (int64_t)fb], 1u);
        else
            dropped = true;
    }
    // one counter update per warp
    const unsigned mh = __ballot_sync(0xffffffffu, hit);
    const unsigned md = __ballot_sync(0xffffffffu, dropped);
    if ((threadIdx.x & 31) == 0) {
        if (mh) atomicAdd(&counters[0], (unsigned long long)__popc(mh));
        if (md) atomicAdd(&counters[1], (unsigned long long)__popc(md));
    }
}

int launch_map(const bfly_bank *b, const float *rho_max, const int32_t *arg_lag, float kappa,
               int64_t lag_origin, int32_t samples_per_tbin, double f_lo, double df,
               int32_t n_fbins, int32_t n_tbins, uint32_t *map, unsigned long long *counters,
               cudaStream_t stream)
{
    const int64_t blocks = (b->T + 255) / 256;
    map_kernel<<<(unsigned)blocks, 256, 0, stream>>>(b->T, b->f0, rho_max, arg_lag, kappa, lag_origin,
                                                     samples_per_tbin, f_lo, df, n_fbins, n_tbins,
                                                     map, counters);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

// The map of a hit list (bfly_tails): one count per hit at (time bin of the hit's lag, frequency
// bin of its template's f0) -- the same coordinates as map_kernel (reading C10), but a template
// may contribute many hits per segment: the paper's trajectory map.
__global__ void __launch_bounds__(256) hits_map_kernel(int64_t n_hits, int64_t T, const double *__restrict__ f0,
                                                       const int32_t *__restrict__ hit_template,
                                                       const int32_t *__restrict__ hit_lag,
                                                       int64_t lag_origin, int32_t samples_per_tbin,
                                                       double f_lo, double df, int32_t n_fbins,
                                                       int32_t n_tbins, uint32_t *__restrict__ map,
                                                       unsigned long long *__restrict__ counters)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool hit = false, dropped = false;
    if (i < n_hits) {
        hit = true;
        const int64_t j = hit_template[i];
        const int64_t tbin = (lag_origin + (int64_t)hit_lag[i]) / samples_per_tbin;
        const double fb = (j >= 0 && j < T) ? floor((f0[j] - f_lo) / df) : -1.0;
        if (tbin >= 0 && tbin < n_tbins && fb >= 0.0 && fb < (double)n_fbins)
            atomicAdd(&map[tbin * (int64_t)n_fbins + (int64_t)fb], 1u);
        else
            dropped = true;
    }
    const unsigned mh = __ballot_sync(0xffffffffu, hit);
    const unsigned md = __ballot_sync(0xffffffffu, dropped);
    if ((threadIdx.x & 31) == 0) {
        if (mh) atomicAdd(&counters[0], (unsigned long long)__popc(mh));
        if (md) atomicAdd(&counters[1], (unsigned long long)__popc(md));
    }
}

int launch_hits_map(const bfly_bank *b, const int32_t *hit_template, const int32_t *hit_lag,
                    int64_t n_hits, int64_t lag_origin, int32_t samples_per_tbin, double f_lo,
                    double df, int32_t n_fbins, int32_t n_tbins, uint32_t *map,
                    unsigned long long *counters, cudaStream_t stream)
{
    if (n_hits == 0) return BFLY_OK;
    hits_map_kernel<<<(unsigned)((n_hits + 255) / 256), 256, 0, stream>>>(
        n_hits, b->T, b->f0, hit_template, hit_lag, lag_origin, samples_per_tbin, f_lo, df, n_fbins,
        n_tbins, map, counters);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

}  // namespace bfly
