// BFLY_FORM_DIRECT: fp32 CUDA-core time-domain correlation with the fused epilogue.
//
// A slow, simple second implementation of rows A3-A7 used as a cross-check of the
// FFT form at sizes the CPU oracle cannot reach.  Templates are synthesised into shared memory
// from the fixed-point phase constants (A3); the sums c, s run on the FP32 pipe (A4); the
// epilogue takes c^2/||hc||^2 + s^2/||hs||^2 over the sliding norm (A5, A6), reduces max/argmax
// over the tile's lags with warp shuffles and merges lag tiles with a packed 64-bit atomicMax
// (value bits high, inverted lag low, so that equal values resolve to the smallest lag) (A7).
#include "bfly_internal.cuh"

namespace bfly {

namespace {
constexpr int DT_J = 16;     // templates per CTA
constexpr int DT_LAGS = 512; // lags per CTA (2 per thread)
constexpr int DT_K = 64;     // template samples per chunk
constexpr int DT_THREADS = 256;

__global__ void __launch_bounds__(DT_THREADS)
direct_kernel(int64_t T, int32_t L, int family, const uint64_t *__restrict__ phA,
              const uint64_t *__restrict__ phB, const uint64_t *__restrict__ phC,
              const float *__restrict__ inc2,
              const float *__restrict__ ins2, const float *__restrict__ x, int64_t n_samples,
              int64_t lag_begin, int64_t n_lags, const float *__restrict__ rn2,
              int64_t n_lag_tiles, unsigned long long *__restrict__ packed)
{
    extern __shared__ float smem[];
    float *xs = smem;                               // DT_LAGS + L (+ pad)
    float *hc = xs + ((DT_LAGS + L + 3) & ~3);      // [DT_J][DT_K]
    float *hs = hc + DT_J * DT_K;

    const int64_t tile = blockIdx.x;
    const int64_t jt = tile / n_lag_tiles;
    const int64_t lt = tile - jt * n_lag_tiles;
    const int64_t j0 = jt * DT_J;
    const int64_t i0 = lt * DT_LAGS;                // first lag index (relative to lag_begin)
    const int tid = threadIdx.x;

    // data window x[lag_begin + i0 .. + DT_LAGS + L - 1), zero beyond the series
    for (int i = tid; i < DT_LAGS + L; i += DT_THREADS) {
        const int64_t g = lag_begin + i0 + i;
        xs[i] = g < n_samples ? __ldg(x + g) : 0.0f;
    }

    float ac[2][DT_J], as[2][DT_J];
#pragma unroll
    for (int j = 0; j < DT_J; ++j) { ac[0][j] = ac[1][j] = as[0][j] = as[1][j] = 0.0f; }

    for (int k0 = 0; k0 < L; k0 += DT_K) {
        __syncthreads();
        // synthesise DT_J x DT_K template samples (A3)
        for (int e = tid; e < DT_J * DT_K; e += DT_THREADS) {
            const int j = e / DT_K, kk = e - j * DT_K;
            const int k = k0 + kk;
            float s = 0.0f, c = 0.0f;
            if (k < L && j0 + j < T) template_sincos(family, phA[j0 + j], phB[j0 + j], phC[j0 + j], (uint32_t)k, &s, &c);
            hc[e] = c;
            hs[e] = s;
        }
        __syncthreads();
        const float *x0 = xs + tid + k0;
        const float *x1 = x0 + DT_THREADS;
#pragma unroll 4
        for (int kk = 0; kk < DT_K; kk += 4) {
            const float a0 = x0[kk], a1 = x0[kk + 1], a2 = x0[kk + 2], a3 = x0[kk + 3];
            const float b0 = x1[kk], b1 = x1[kk + 1], b2 = x1[kk + 2], b3 = x1[kk + 3];
#pragma unroll
            for (int j = 0; j < DT_J; ++j) {
                const float4 c4 = *reinterpret_cast<const float4 *>(hc + j * DT_K + kk);
                const float4 s4 = *reinterpret_cast<const float4 *>(hs + j * DT_K + kk);
                ac[0][j] = fmaf(a0, c4.x, ac[0][j]); ac[0][j] = fmaf(a1, c4.y, ac[0][j]);
                ac[0][j] = fmaf(a2, c4.z, ac[0][j]); ac[0][j] = fmaf(a3, c4.w, ac[0][j]);
                as[0][j] = fmaf(a0, s4.x, as[0][j]); as[0][j] = fmaf(a1, s4.y, as[0][j]);
                as[0][j] = fmaf(a2, s4.z, as[0][j]); as[0][j] = fmaf(a3, s4.w, as[0][j]);
                ac[1][j] = fmaf(b0, c4.x, ac[1][j]); ac[1][j] = fmaf(b1, c4.y, ac[1][j]);
                ac[1][j] = fmaf(b2, c4.z, ac[1][j]); ac[1][j] = fmaf(b3, c4.w, ac[1][j]);
                as[1][j] = fmaf(b0, s4.x, as[1][j]); as[1][j] = fmaf(b1, s4.y, as[1][j]);
                as[1][j] = fmaf(b2, s4.z, as[1][j]); as[1][j] = fmaf(b3, s4.w, as[1][j]);
            }
        }
    }

    // epilogue (A5-A7)
    const int64_t ia = i0 + tid, ib = ia + DT_THREADS;
    const float ra = ia < n_lags ? __ldg(rn2 + ia) : 0.0f;
    const float rb = ib < n_lags ? __ldg(rn2 + ib) : 0.0f;
#pragma unroll
    for (int j = 0; j < DT_J; ++j) {
        const bool live = (j0 + j < T);
        const float ic = live ? inc2[j0 + j] : 0.0f, is = live ? ins2[j0 + j] : 0.0f;
        const float qa = fmaf(ac[0][j] * ac[0][j], ic, as[0][j] * as[0][j] * is) * ra;
        const float qb = fmaf(ac[1][j] * ac[1][j], ic, as[1][j] * as[1][j] * is) * rb;
        unsigned long long pa = 0ull, pb = 0ull;
        if (ia < n_lags)
            pa = ((unsigned long long)__float_as_uint(qa) << 32) |
                 (unsigned long long)(0xFFFFFFFFu - (uint32_t)(lag_begin + ia));
        if (ib < n_lags)
            pb = ((unsigned long long)__float_as_uint(qb) << 32) |
                 (unsigned long long)(0xFFFFFFFFu - (uint32_t)(lag_begin + ib));
        unsigned long long p = pa > pb ? pa : pb;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long q = __shfl_xor_sync(0xffffffffu, p, o);
            p = q > p ? q : p;
        }
        if ((tid & 31) == 0 && live && p != 0ull) atomicMax(packed + j0 + j, p);
    }
}

__global__ void __launch_bounds__(256)
unpack_kernel(int64_t T, const unsigned long long *__restrict__ packed, int64_t lag_begin,
              float *__restrict__ rho_max, int32_t *__restrict__ arg_lag)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= T) return;
    const unsigned long long p = packed[j];
    if (p == 0ull) {            // empty lag range
        rho_max[j] = 0.0f;
        arg_lag[j] = (int32_t)lag_begin;
        return;
    }
    rho_max[j] = sqrtf(__uint_as_float((uint32_t)(p >> 32)));
    arg_lag[j] = (int32_t)(0xFFFFFFFFu - (uint32_t)(p & 0xFFFFFFFFull));
}
}  // namespace

int launch_direct(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                  int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream)
{
    const int64_t n_lags = lag_end - lag_begin;
    BFLY_CUDA(cudaMemsetAsync(b->packed, 0, sizeof(unsigned long long) * (size_t)b->T, stream));
    if (n_lags > 0) {
        const int64_t n_lag_tiles = (n_lags + DT_LAGS - 1) / DT_LAGS;
        const int64_t n_j_tiles = (b->T + DT_J - 1) / DT_J;
        const int64_t tiles = n_lag_tiles * n_j_tiles;
        if (tiles >= (1LL << 31)) { set_error("direct form: too many tiles (%lld)", (long long)tiles); return BFLY_ERANGE; }
        const size_t smem = sizeof(float) * (size_t)(((DT_LAGS + b->L + 3) & ~3) + 2 * DT_J * DT_K);
        core_timer_start(b, stream);
        direct_kernel<<<(unsigned)tiles, DT_THREADS, smem, stream>>>(
            b->T, b->L, b->family, b->phA, b->phB, b->phC, b->inc2, b->ins2, x, n_samples, lag_begin, n_lags, b->rn2,
            n_lag_tiles, b->packed);
        core_timer_stop(b, stream);
        count_launch();
        BFLY_CUDA(cudaGetLastError());
    }
    unpack_kernel<<<(unsigned)((b->T + 255) / 256), 256, 0, stream>>>(b->T, b->packed, lag_begin,
                                                                      rho_max, arg_lag);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

}  // namespace bfly
