// TEMPORARY STUB (replaced by the FFT form): routes to the direct form so that the boundary,
// the tests and the bench can be exercised end to end.
#include "bfly_internal.cuh"
namespace bfly {
int64_t fft_blocks_needed(int32_t L, int64_t n_lags)
{
    const int64_t V = FFT_B - L + 1;
    return n_lags > 0 ? (n_lags + V - 1) / V : 0;
}
int launch_fft(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
               int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream)
{
    return launch_direct(b, x, n_samples, lag_begin, lag_end, rho_max, arg_lag, stream);
}
}
