// The paper's way of reading the output of two series (readings T1-T3 of
// DESIGN.md): time-randomised control, simultaneous hits in two series with
// frequencies within a window, and pseudo-spectra (Fig. 6).  Integer and gather
// work only: results are exact and order independent.  All three are HBM-bound streams.
#include "bfly_internal.cuh"

namespace bfly {

namespace {

// T1: out[i] = x[perm[i]]; an index outside [0, n) writes 0 and raises the flag.
__global__ void __launch_bounds__(256)
time_randomize_kernel(const float *__restrict__ x, const int32_t *__restrict__ perm, int64_t n,
                      float *__restrict__ out, int *__restrict__ bad)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t p = perm[i];
    if (p < 0 || p >= n) { out[i] = 0.0f; if (bad) *bad = 1; return; }
    out[i] = __ldg(x + p);
}

// T2: one CTA per time bin.  Presence bits of both rows in shared memory; a frequency bin has a
// partner when the other row has a set bit within +- w bins.
constexpr int CO_MAX_WORDS = 2048;           // up to 65536 frequency bins per row
__global__ void __launch_bounds__(256)
coincidence_kernel(const uint32_t *__restrict__ m1, const uint32_t *__restrict__ m2, int32_t n_fbins,
                   int32_t w, uint32_t *__restrict__ c1, uint32_t *__restrict__ c2)
{
    __shared__ uint32_t p1[CO_MAX_WORDS], p2[CO_MAX_WORDS];
    const int64_t row = (int64_t)blockIdx.x * n_fbins;
    const int n_words = (n_fbins + 31) >> 5;
    for (int k = threadIdx.x; k < n_words; k += blockDim.x) { p1[k] = 0u; p2[k] = 0u; }
    __syncthreads();
    for (int f = threadIdx.x; f < n_fbins; f += blockDim.x) {
        if (m1[row + f]) atomicOr(&p1[f >> 5], 1u << (f & 31));
        if (m2[row + f]) atomicOr(&p2[f >> 5], 1u << (f & 31));
    }
    __syncthreads();
    auto any_in = [&](const uint32_t *p, int lo, int hi) {      // any set bit in [lo, hi]
        for (int k = lo >> 5; k <= hi >> 5; ++k) {
            uint32_t mask = 0xFFFFFFFFu;
            if (k == lo >> 5) mask &= 0xFFFFFFFFu << (lo & 31);
            if (k == hi >> 5) mask &= 0xFFFFFFFFu >> (31 - (hi & 31));
            if (p[k] & mask) return true;
        }
        return false;
    };
    for (int f = threadIdx.x; f < n_fbins; f += blockDim.x) {
        const int lo = max(f - w, 0), hi = (int)min((int64_t)f + w, (int64_t)n_fbins - 1);
        const uint32_t a = m1[row + f], b = m2[row + f];
        c1[row + f] = (a && any_in(p2, lo, hi)) ? a : 0u;
        c2[row + f] = (b && any_in(p1, lo, hi)) ? b : 0u;
    }
}

// T3: column sums.  blockIdx.y takes a slab of 256 time bins; consecutive threads read
// consecutive frequency bins (coalesced); one 64-bit atomic per thread and slab.
__global__ void __launch_bounds__(256)
pseudo_spectrum_kernel(const uint32_t *__restrict__ m, int32_t n_tbins, int32_t n_fbins,
                       unsigned long long *__restrict__ spec)
{
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_fbins) return;
    const int t0 = blockIdx.y * 256, t1 = min(t0 + 256, n_tbins);
    unsigned long long s = 0ull;
    for (int t = t0; t < t1; ++t) s += m[(int64_t)t * n_fbins + f];
    if (s) atomicAdd(&spec[f], s);
}

}  // namespace

int launch_time_randomize(const float *x, const int32_t *perm, int64_t n, float *out, int *bad,
                          cudaStream_t stream)
{
    if (n == 0) return BFLY_OK;
    time_randomize_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(x, perm, n, out, bad);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

int launch_coincidence(const uint32_t *m1, const uint32_t *m2, int32_t n_tbins, int32_t n_fbins,
                       int32_t w, uint32_t *c1, uint32_t *c2, cudaStream_t stream)
{
    if (n_fbins > CO_MAX_WORDS * 32) { set_error("more than %d frequency bins", CO_MAX_WORDS * 32); return BFLY_ERANGE; }
    coincidence_kernel<<<(unsigned)n_tbins, 256, 0, stream>>>(m1, m2, n_fbins, w, c1, c2);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

int launch_pseudo_spectrum(const uint32_t *m, int32_t n_tbins, int32_t n_fbins,
                           unsigned long long *spec, cudaStream_t stream)
{
    dim3 grid((unsigned)((n_fbins + 255) / 256), (unsigned)((n_tbins + 255) / 256));
    pseudo_spectrum_kernel<<<grid, 256, 0, stream>>>(m, n_tbins, n_fbins, spec);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

}  // namespace bfly
