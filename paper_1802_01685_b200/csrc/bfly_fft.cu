// BFLY_FORM_FFT: hand-written batched overlap-save FFT correlate with the fused epilogue
// (rows A3-A7 of DESIGN.md; the paper's own correlation method: "FFT ...
// complex-to-complex single precision", here entirely in registers and shared memory).
//
// Mathematics.  With g[k] = cos(phi_k) - i sin(phi_k) (k < L, zero-padded to B) and a data block
// xb[n] = x[o_b + n], n < B,
//     z_b(tau') = sum_k xb[tau' + k] g[k] = c(tau') - i s(tau')      exact for tau' <= B - L,
// and with F+ the unnormalised length-B transform Y[m] = sum_n y[n] exp(+2 pi i m n / B):
//     z_b = F+( X_b . G ),   G = F+(g),   X_b = conj(F+(xb)) / B.
// X_b is computed once per call by data_spectra_kernel; the correlation kernel keeps G in
// registers, so per (template, block) the only memory traffic is one read of X_b from L2.
//
// The length-8192 transform is 16 x 32 x 16, three passes of register-resident radix-2 DIF
// butterflies, 512 threads x 16 points (16 warps per SM, 128 registers per thread):
//     n = 512 n1 + 16 n2 + n3   ->   m = m1 + 16 m2 + 512 m3        (n2, m2 < 32; others < 16)
//     pass 1: thread t = 16 n2 + n3: 16-point over n1, times w_8192^(m1 t)      -> buf0
//     pass 2: (n3, m1) x role:       32-point over n2 split over a thread pair: role 0 takes
//             the sums a+b (even m2), role 1 the rotated differences (odd m2); each then runs a
//             16-point transform; times w_512^(m2 n3)                            buf0 -> buf1
//     pass 3: thread t = m1 + 16 m2: 16-point over n3                            <- buf1
// Shared-memory layout idx(n3, r, m1) = n3 * 513 + r * 16 + m1 (r = n2, then m2): every access
// of every pass is bank-conflict free; the two buffers ping-pong, so a transform needs two
// __syncthreads; and a thread's 16 outputs m = t + 512 s are exactly its 16 inputs of the next
// transform, so G never leaves the registers.
#include "bfly_fft32.cuh"

namespace bfly {

namespace {

using namespace fft32;


// X_b = conj(F+(xb)) / B for every data block of the call, natural order.
__global__ void __launch_bounds__(NT, 1)
data_spectra_kernel(const float *__restrict__ x, int64_t n_samples, int64_t lag_begin, int32_t V,
                    float2 *__restrict__ xspec)
{
    extern __shared__ float2 smem[];
    const Smem sm = carve(smem);
    const int t = threadIdx.x;
    fill_tables(sm, t);
    const int64_t off = lag_begin + (int64_t)blockIdx.x * V;
    float2 v[PTS];
#pragma unroll
    for (int s = 0; s < PTS; ++s) {
        const int64_t g = off + t + NT * s;
        v[s] = make_float2(g < n_samples ? __ldg(x + g) : 0.0f, 0.0f);
    }
    fft8192(v, sm, t);
    float2 *out = xspec + (int64_t)blockIdx.x * FFT_B + t;
    const float sc = 1.0f / (float)FFT_B;
#pragma unroll
    for (int s = 0; s < PTS; ++s) out[NT * s] = make_float2(v[s].x * sc, -v[s].y * sc);
}

// One CTA per template at a time (persistent, strided over the bank): G = F+(g) in registers,
// then per data block z = F+(X_b . G) and the fused epilogue (A5-A7).
// SV = ceil(V / 512): output slots s >= SV never hold a valid lag (tau' = t + 512 s >= V), so their
// butterflies in the last pass and their epilogue are dead code (SV = 9 at L = 4096).
template <int SV>
__global__ void __launch_bounds__(NT, 1)
fft_correlate_kernel(int64_t T, int32_t L, int family, const uint64_t *__restrict__ phA,
                     const uint64_t *__restrict__ phB, const uint64_t *__restrict__ phC,
                     const float *__restrict__ inc2,
                     const float *__restrict__ ins2, const float2 *__restrict__ xspec,
                     const float *__restrict__ rn2, int64_t lag_begin, int64_t n_lags, int32_t V,
                     int32_t n_blocks, float *__restrict__ rho_max, int32_t *__restrict__ arg_lag)
{
    extern __shared__ float2 smem[];
    const Smem sm = carve(smem);
    __shared__ unsigned long long red[NT / 32];
    const int t = threadIdx.x;
    fill_tables(sm, t);

    for (int64_t j = blockIdx.x; j < T; j += gridDim.x) {
        // ---- A3: synthesise g[n] = exp(-i phi_n), n = t + 512 s < L, and transform it
        const uint64_t A = phA[j], Bq = phB[j], Cq = phC[j];
        float2 G[PTS];
#pragma unroll
        for (int s = 0; s < PTS; ++s) {
            const int n = t + NT * s;
            float sn = 0.0f, cs = 0.0f;
            if (n < L) template_sincos(family, A, Bq, Cq, (uint32_t)n, &sn, &cs);
            G[s] = make_float2(cs, -sn);
        }
        fft8192(G, sm, t);
        const float ic = inc2[j], is = ins2[j];

        float best = -1.0f;                    // rho^2 >= 0: the first valid lag always wins
        int32_t best_i = 0;                    // lag index relative to lag_begin
        for (int32_t b = 0; b < n_blocks; ++b) {
            // ---- A4: z = F+(X_b . G)
            const float2 *xb = xspec + (int64_t)b * FFT_B + t;
            float2 v[PTS];
#pragma unroll
            for (int s = 0; s < PTS; ++s) v[s] = __ldg(xb + NT * s);
#pragma unroll
            for (int s = 0; s < PTS; ++s) v[s] = cmul(v[s], G[s]);
            fft8192(v, sm, t);
            // ---- A5-A7: tau' = t + 512 s; valid while tau' < V and the lag exists
            const int64_t i0 = (int64_t)b * V;
            const int64_t left = n_lags - i0;
            const int32_t vb = left < V ? (int32_t)left : V;
            const float *r = rn2 + i0 + t;
#pragma unroll
            for (int s = 0; s < SV; ++s) {
                const int tp = t + NT * s;
                if (tp < vb) {
                    const float q = fmaf(v[s].x * v[s].x, ic, v[s].y * v[s].y * is) * __ldg(r + NT * s);
                    if (q > best) { best = q; best_i = (int32_t)i0 + tp; }
                }
            }
        }
        // ---- A7: CTA-wide max with ties to the smallest lag
        unsigned long long p = 0ull;
        if (best >= 0.0f)
            p = ((unsigned long long)__float_as_uint(best) << 32) |
                (unsigned long long)(0xFFFFFFFFu - (uint32_t)best_i);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long q = __shfl_xor_sync(0xffffffffu, p, o);
            p = q > p ? q : p;
        }
        if ((t & 31) == 0) red[t >> 5] = p;
        __syncthreads();
        if (t == 0) {
#pragma unroll
            for (int w = 1; w < NT / 32; ++w) p = red[w] > p ? red[w] : p;
            if (p == 0ull) {                    // no valid lag at all (empty range)
                rho_max[j] = 0.0f;
                arg_lag[j] = (int32_t)lag_begin;
            } else {
                rho_max[j] = sqrtf(__uint_as_float((uint32_t)(p >> 32)));
                arg_lag[j] = (int32_t)(lag_begin + (int64_t)(0xFFFFFFFFu - (uint32_t)(p & 0xFFFFFFFFull)));
            }
        }
        __syncthreads();                        // red[] is reused by the next template
    }
}



}  // namespace

int64_t fft_blocks_needed(int32_t L, int64_t n_lags)
{
    const int64_t V = FFT_B - L + 1;
    return n_lags > 0 ? (n_lags + V - 1) / V : 0;
}

int launch_fft(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
               int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream)
{
    static PerDeviceOnce once;           // function attributes are per device
    const int rc_attr = once.run(b->device, []() -> int {
        BFLY_CUDA(cudaFuncSetAttribute(data_spectra_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(fft_correlate_kernel<9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(fft_correlate_kernel<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(fft_correlate_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM));
        return BFLY_OK;
    });
    if (rc_attr) return rc_attr;
    const int64_t n_lags = lag_end - lag_begin;
    const int32_t V = FFT_B - b->L + 1;
    const int64_t n_blocks = fft_blocks_needed(b->L, n_lags);
    if (n_blocks * FFT_B > b->xspec_cap) { set_error("FFT workspace too small (internal)"); return BFLY_EINVAL; }
    if (n_lags >= (1LL << 31)) { set_error("too many lags"); return BFLY_ERANGE; }
    if (n_blocks > 0) {
        data_spectra_kernel<<<(unsigned)n_blocks, NT, FFT_SMEM, stream>>>(x, n_samples, lag_begin, V, b->xspec);
        count_launch();
        BFLY_CUDA(cudaGetLastError());
    }
    const int64_t ctas = b->T < (int64_t)b->sm_count ? b->T : (int64_t)b->sm_count;
    core_timer_start(b, stream);
    const int sv = (V + NT - 1) / NT;
#define BFLY_FFT_LAUNCH(SV_)                                                                        \
    fft_correlate_kernel<SV_><<<(unsigned)ctas, NT, FFT_SMEM, stream>>>(                             \
        b->T, b->L, b->family, b->phA, b->phB, b->phC, b->inc2, b->ins2, b->xspec, b->rn2, lag_begin, n_lags, V, \
        (int32_t)n_blocks, rho_max, arg_lag)
    if (sv <= 9) BFLY_FFT_LAUNCH(9);
    else if (sv <= 13) BFLY_FFT_LAUNCH(13);
    else BFLY_FFT_LAUNCH(16);
#undef BFLY_FFT_LAUNCH
    core_timer_stop(b, stream);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

}  // namespace bfly
