// fp32 length-8192 FFT in registers and shared memory (512 threads x 16 points): the transform of
// BFLY_FORM_FFT (bfly_fft.cu), also used to compute the data-block spectra of BFLY_FORM_FFT_TC.
// See bfly_fft.cu for the index maps and the shared-memory layout.
#pragma once
#include "bfly_internal.cuh"

namespace bfly {
namespace fft32 {

constexpr int NT = 512;            // threads per CTA
constexpr int PTS = 16;            // points per thread
constexpr int ROW = 513;           // padded row (n3) stride of a work buffer, in complex
constexpr int WORK = 16 * ROW;     // complex elements of one work buffer
constexpr int TW1 = 15 * NT;       // pass 1 -> 2 twiddles w_8192^(m1 t), m1 = 1..15
constexpr int TW2 = 512;           // pass 2 -> 3 twiddles w_512^k
static_assert(NT * PTS == FFT_B, "geometry");

struct Smem {                      // carved from dynamic shared memory
    float2 *buf0, *buf1, *tw1, *tw2;
};
__device__ __forceinline__ Smem carve(float2 *base)
{
    return Smem{base, base + WORK, base + 2 * WORK, base + 2 * WORK + TW1};
}

// cos(2 pi k / 32), k = 0..8
__device__ __forceinline__ constexpr float cos32(int k)
{
    return k == 0 ? 1.0f
         : k == 1 ? 0.98078528040323044913f
         : k == 2 ? 0.92387953251128675613f
         : k == 3 ? 0.83146961230254523708f
         : k == 4 ? 0.70710678118654752440f
         : k == 5 ? 0.55557023301960222474f
         : k == 6 ? 0.38268343236508977173f
         : k == 7 ? 0.19509032201612826785f
         : 0.0f;
}
// exp(+2 pi i k / 32) for 0 <= k < 16
__device__ __forceinline__ constexpr float tw32_re(int k) { return k <= 8 ? cos32(k) : -cos32(16 - k); }
__device__ __forceinline__ constexpr float tw32_im(int k) { return k <= 8 ? cos32(8 - k) : cos32(k - 8); }

__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

template <int N> __device__ __forceinline__ constexpr int bitrev(int m)
{
    int r = 0;
    for (int b = 1; b < N; b <<= 1) { r = (r << 1) | (m & 1); m >>= 1; }
    return r;
}

// In-register radix-2 decimation-in-frequency transform Y[m] = sum_n a[n] exp(+2 pi i m n / N);
// on return a[bitrev(m)] holds Y[m].  Fully unrolled: every index and twiddle is a constant.
template <int N> __device__ __forceinline__ void fft_dif(float2 (&a)[N])
{
#pragma unroll
    for (int span = N / 2; span >= 1; span >>= 1) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
            if ((i & span) == 0) {
                const int j = i + span;
                const int k = (i & (span - 1)) * (16 / span);   // twiddle exp(2 pi i k / 32)
                const float2 u = a[i], v = a[j];
                a[i] = make_float2(u.x + v.x, u.y + v.y);
                const float dx = u.x - v.x, dy = u.y - v.y;
                if (k == 0) {
                    a[j] = make_float2(dx, dy);
                } else if (k == 8) {            // times +i
                    a[j] = make_float2(-dy, dx);
                } else if (k == 4) {            // times (1 + i)/sqrt 2
                    a[j] = make_float2((dx - dy) * cos32(4), (dx + dy) * cos32(4));
                } else if (k == 12) {           // times (-1 + i)/sqrt 2
                    a[j] = make_float2((-dx - dy) * cos32(4), (dx - dy) * cos32(4));
                } else {
                    const float c = tw32_re(k), s = tw32_im(k);
                    a[j] = make_float2(fmaf(dx, c, -dy * s), fmaf(dx, s, dy * c));
                }
            }
        }
    }
}

// The three passes.  In: v[s] = y[t + 512 s].  Out: v[s] = Y[t + 512 s].
__device__ __forceinline__ void fft8192(float2 (&v)[PTS], const Smem &sm, const int t)
{
    // ---- pass 1: 16-point over n1, twiddle w_8192^(m1 t), store at (n3, n2, m1) of buf0
    fft_dif<16>(v);
    {
        float2 *dst = sm.buf0 + (t & 15) * ROW + (t >> 4) * 16;
        const float2 *tw = sm.tw1 + t;
        dst[0] = v[0];
#pragma unroll
        for (int m1 = 1; m1 < 16; ++m1) dst[m1] = cmul(v[bitrev<16>(m1)], tw[(m1 - 1) * NT]);
    }
    __syncthreads();
    // ---- pass 2: 32-point over n2 as (radix-2 stage split over two threads) + 16-point
    {
        const int q = t & 255, role = t >> 8, n3 = q >> 4, m1 = q & 15;
        const float2 *src = sm.buf0 + n3 * ROW + m1;
        float2 c[16];
        if (role == 0) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const float2 a = src[i * 16], b = src[(i + 16) * 16];
                c[i] = make_float2(a.x + b.x, a.y + b.y);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const float2 a = src[i * 16], b = src[(i + 16) * 16];
                const float dx = a.x - b.x, dy = a.y - b.y;
                if (i == 0) c[i] = make_float2(dx, dy);
                else if (i == 8) c[i] = make_float2(-dy, dx);
                else c[i] = make_float2(fmaf(dx, tw32_re(i), -dy * tw32_im(i)), fmaf(dx, tw32_im(i), dy * tw32_re(i)));
            }
        }
        fft_dif<16>(c);
        float2 *dst = sm.buf1 + n3 * ROW + role * 16 + m1;          // m2 = 2 k + role
        const float2 *tw = sm.tw2 + role * n3;                      // (2 k + role) n3 < 512
#pragma unroll
        for (int k = 0; k < 16; ++k) dst[k * 32] = cmul(c[bitrev<16>(k)], tw[2 * k * n3]);
    }
    __syncthreads();
    // ---- pass 3: 16-point over n3; output m = t + 512 m3 lands in slot m3
    {
        const float2 *src = sm.buf1 + t;
        float2 a[16];
#pragma unroll
        for (int n3 = 0; n3 < 16; ++n3) a[n3] = src[n3 * ROW];
        fft_dif<16>(a);
#pragma unroll
        for (int m3 = 0; m3 < 16; ++m3) v[m3] = a[bitrev<16>(m3)];
    }
}

// Twiddle tables, once per CTA (the kernels are persistent).
__device__ __forceinline__ void fill_tables(const Smem &sm, int t)
{
    float s, c;
    sincospif((float)t * (1.0f / 256.0f), &s, &c);
    sm.tw2[t] = make_float2(c, s);
#pragma unroll 1
    for (int m1 = 1; m1 < 16; ++m1) {
        sincospif((float)(m1 * t) * (1.0f / 4096.0f), &s, &c);
        sm.tw1[(m1 - 1) * NT + t] = make_float2(c, s);
    }
    __syncthreads();
}

constexpr size_t FFT_SMEM = sizeof(float2) * (size_t)(2 * WORK + TW1 + TW2);

}  // namespace fft32
}  // namespace bfly
