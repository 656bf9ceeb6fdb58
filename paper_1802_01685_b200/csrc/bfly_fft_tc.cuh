// BFLY_FORM_FFT_TC: device code of the tensor-core FFT (see bfly_fft_tc.cu for the whole story).
//
// Length-8192 transform z[n] = sum_m Y[m] exp(+2 pi i m n / 8192) as four passes of small DFTs
// executed by mma.sync.m16n8k16 (fp16 operands, fp32 accumulate) on real-embedded DFT matrices:
//     m = 1024 a + 128 b + 16 c + d'          a, b, c < 8,  d' < 16        (input index)
//     n = alpha + 8 beta + 64 gamma + 512 delta   alpha, beta, gamma < 8, delta < 16 (output)
//     pass A: 8-point DFT over a  -> alpha, times w_64^(b alpha)
//     pass B: 8-point DFT over b  -> beta,  times w_8192^((alpha + 8 beta)(16 c + d'))
//     -- exchange through shared memory --
//     pass C: 8-point DFT over c  -> gamma, times w_128^(d' gamma)
//     pass D: 16-point DFT over d' -> delta (only delta < 8, i.e. n < 4096, unless FULL)
// A complex r-point DFT on 8 columns is the real product [[Wr, -Wi], [Wi, Wr]] x [Xr; Xi]: for
// r = 8 exactly one m16n8k16 MMA (64 complex points per MMA), for r = 16 with 8 outputs two.
// Passes A -> B and C -> D chain in registers with no data movement: the accumulator fragment of
// one MMA (rows = output index, two adjacent columns per thread) is, after the twiddle and the
// fp16 pack, exactly the B-operand fragment of the next MMA that contracts over those columns.
//
// Fragment conventions (PTX ISA, mma.m16n8k16 .f16): lane = 4 g + t;
//     A (16x16 row):  a0 (row g, k 2t..2t+1)  a1 (row g+8, k 2t..)  a2 (row g, k 2t+8..)  a3 (row g+8, k 2t+8..)
//     B (16x8 col):   b0 (k 2t..2t+1, col g)  b1 (k 2t+8..2t+9, col g)
//     D (16x8):       d0 (row g, col 2t) d1 (row g, col 2t+1) d2 (row g+8, col 2t) d3 (row g+8, col 2t+1)
// Embedding: rows/k 0..7 = real parts, 8..15 = imaginary parts, so a3 == a0 and a thread's D holds
// the two complex numbers (d0, d2) and (d1, d3).
//
// Accuracy.  DFT matrices are scaled by S8 / S16 so that every entry is (nearly) an fp16 number
// (S8 / sqrt 2 is within 2.6e-7, relative, of one; the three irrational entries of W16 within
// 2.9e-5); the scale is taken out again in the fp32 twiddles and in the epilogue.  Twiddles are
// applied in fp32 (packed FMUL2 / FFMA2) on the fp32 accumulators; data are rounded to fp16 once
// per pass.
#pragma once

#include <cuda_fp16.h>

#include "bfly_internal.cuh"

namespace bfly {
namespace tc {

constexpr int NT = 512;                    // threads per CTA (16 warps)
constexpr int TCV = 4096;                  // lags produced per block (delta < 8)
constexpr float S8 = 1.3603515625f;        // fp16 number with S8 / sqrt(2) ~ fp16 number
constexpr float S16 = 1.8603515625f;       // same for cos(pi/8), sqrt(1/2), sin(pi/8)
constexpr int EXCH_WORDS = 8192;           // one exchange buffer: 8192 complex as 2 x fp16
constexpr int MAX_TAIL = 4;                // lags past the last whole block done by direct sums

__device__ __forceinline__ uint32_t pack_h2(float lo, float hi)
{
    __half2 v = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&v);
}
__device__ __forceinline__ __half2 as_h2(uint32_t w) { return *reinterpret_cast<__half2 *>(&w); }
__device__ __forceinline__ uint32_t as_u32(__half2 v) { return *reinterpret_cast<uint32_t *>(&v); }

// Two complex numbers held by component: r = (Re p0, Re p1), i = (Im p0, Im p1).  That is how a
// thread's MMA accumulator arrives ((d0, d1) and (d2, d3) are aligned register pairs), so the
// twiddle multiply is four packed fp32 instructions (FMUL2 / FFMA2, sm_100) for two points.
struct cpair { float2 r, i; };
__device__ __forceinline__ cpair cmul2(const float (&d)[4], const cpair &w)
{
    const float2 dr = make_float2(d[0], d[1]), di = make_float2(d[2], d[3]);
    cpair p;
    p.r = __ffma2_rn(make_float2(-di.x, -di.y), w.i, __fmul2_rn(dr, w.r));
    p.i = __ffma2_rn(di, w.r, __fmul2_rn(dr, w.i));
    return p;
}
__device__ __forceinline__ cpair make_cpair(float2 p0, float2 p1)
{
    cpair c;
    c.r = make_float2(p0.x, p1.x);
    c.i = make_float2(p0.y, p1.y);
    return c;
}

// The same two complex numbers in fp16: r = (Re p0, Re p1), i = (Im p0, Im p1) as half2 words --
// the accumulator fragment of an fp16-accumulate MMA and, unchanged, the B fragment of the next.
struct hpair { uint32_t r, i; };
__device__ __forceinline__ hpair cmul2(const uint32_t (&d)[2], const hpair &w)
{
    const __half2 dr = as_h2(d[0]), di = as_h2(d[1]), wr = as_h2(w.r), wi = as_h2(w.i);
    hpair p;
    p.r = as_u32(__hfma2(__hneg2(di), wi, __hmul2(dr, wr)));
    p.i = as_u32(__hfma2(di, wr, __hmul2(dr, wi)));
    return p;
}
__device__ __forceinline__ hpair make_hpair(float2 p0, float2 p1)
{
    hpair c;
    c.r = pack_h2(p0.x, p1.x);
    c.i = pack_h2(p0.y, p1.y);
    return c;
}
template <bool HALF> struct TwT { typedef cpair type; };
template <> struct TwT<true> { typedef hpair type; };
template <bool HALF> __device__ __forceinline__ typename TwT<HALF>::type make_tw(float2 p0, float2 p1);
template <> __device__ __forceinline__ cpair make_tw<false>(float2 p0, float2 p1) { return make_cpair(p0, p1); }
template <> __device__ __forceinline__ hpair make_tw<true>(float2 p0, float2 p1) { return make_hpair(p0, p1); }

// D = A x B (+ C); A = (a0, a1, a2, a0)
__device__ __forceinline__ void mma_z(float (&d)[4], const uint32_t (&a)[3], uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%4}, {%7,%8}, {%9,%9,%9,%9};"
        : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(b0), "r"(b1), "f"(0.0f));
}
__device__ __forceinline__ void mma_acc(float (&d)[4], const uint32_t (&a)[3], uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%4}, {%7,%8}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(b0), "r"(b1));
}

// fp16-accumulate variant: d0 = (row g, cols 2t, 2t+1), d1 = (row g + 8, ..) as half2 words
__device__ __forceinline__ void mma_h(uint32_t (&d)[2], const uint32_t (&a)[3], uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f16.f16.f16.f16 {%0,%1}, {%2,%3,%4,%2}, {%5,%6}, {%7,%7};"
        : "=r"(d[0]), "=r"(d[1])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(b0), "r"(b1), "r"(0u));
}

// Per-thread constants of the transform (registers for the whole kernel).  HALF selects the
// all-fp16 inner passes (fp16-accumulate MMAs, half2 twiddles: no fp32 <-> fp16 conversions
// between passes A .. C; pass D and the epilogue stay fp32).
template <bool HALF>
struct ConstsT {
    uint32_t w8[3];          // A fragment of S8 * W8 (real-embedded)
    uint32_t w16[2][3];      // A fragments of S16 * W16, rows delta < 8, k-step h (d' = 8 h + ..)
    typedef typename TwT<HALF>::type tw_t;
    tw_t twAB;               // e = 0, 1: w_64^(g (2t+e)) / S8:            alpha = g, b = 2t + e
    tw_t twBig[8];           // [ci*2+h], e = 0, 1: w_8192^((2t+e + 8g)(16 c + d')) / S8
    tw_t twC[2];             // [h], e = 0, 1: w_128^((8h + 2t + e) g) / S8:  gamma = g
    uint32_t st_off[4];      // [2 e + p]: byte offset of this thread's chunk (U = 2t + e + 8g, chunk0 + p) in an exchange buffer
};

// exp(+2 pi i num / den) * scale, num reduced mod den first (den a power of two <= 8192)
__device__ __forceinline__ float2 root(int num, int den, float scale)
{
    float s, c;
    sincospif((float)(num & (den - 1)) * (2.0f / (float)den), &s, &c);
    return make_float2(c * scale, s * scale);
}

// A fragment (a0, a1, a2) of the real-embedded r-point DFT rows `row0 + g`, input points k0 + 2t, +1
__device__ __forceinline__ void dft_frag(uint32_t (&a)[3], int r, float scale, int row, int k)
{
    const float2 w0 = root(row * k, r, scale), w1 = root(row * (k + 1), r, scale);
    a[0] = pack_h2(w0.x, w1.x);
    a[1] = pack_h2(w0.y, w1.y);
    a[2] = pack_h2(-w0.y, -w1.y);
}

// Byte-free addressing of an exchange buffer, in 16-byte chunks: unit U = alpha + 8 beta owns 32
// chunks; chunk (d' & 7) * 4 + (c >> 1) holds {Re(d'<8), Im(d'<8), Re(d'>=8), Im(d'>=8)} of the
// c pair as four fp16x2 words.  The XOR makes both the stores (lanes differ in U) and the loads
// (lanes differ in chunk) bank-conflict free.
__device__ __forceinline__ int exch_chunk(int U, int chunk) { return U * 32 + (chunk ^ ((U >> 1) & 7)); }

// Warp w handles, before the exchange, the eight 64-point sub-transforms ("units") with
// c = 4 (w >> 3) + ci, d' = (w & 7) + 8 h  (unit index u = 2 ci + h), and after it the four
// units with alpha + 8 beta = 4 w + i.
template <bool HALF>
__device__ __forceinline__ void make_consts(ConstsT<HALF> &k, int tid)
{
    const int w = tid >> 5, g = (tid >> 2) & 7, t = tid & 3;
    dft_frag(k.w8, 8, S8, g, 2 * t);
    dft_frag(k.w16[0], 16, S16, g, 2 * t);
    dft_frag(k.w16[1], 16, S16, g, 8 + 2 * t);
    const float r8 = 1.0f / S8;
    k.twAB = make_tw<HALF>(root(g * (2 * t), 64, r8), root(g * (2 * t + 1), 64, r8));
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int c = 4 * (w >> 3) + (u >> 1), dp = (w & 7) + 8 * (u & 1);
        k.twBig[u] = make_tw<HALF>(root((2 * t + 8 * g) * (16 * c + dp), 8192, r8),
                                root((2 * t + 1 + 8 * g) * (16 * c + dp), 8192, r8));
    }
    {
        const int chunk0 = (w & 7) * 4 + 2 * (w >> 3);
#pragma unroll
        for (int e = 0; e < 2; ++e)
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                k.st_off[2 * e + p] = 16u * (uint32_t)exch_chunk(2 * t + e + 8 * g, chunk0 + p);
                asm volatile("" : "+r"(k.st_off[2 * e + p]));      // held as byte offsets: STS [R + UR], no LEA per store
            }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h)
        k.twC[h] = make_tw<HALF>(root((8 * h + 2 * t) * g, 128, r8), root((8 * h + 2 * t + 1) * g, 128, r8));
}

// Passes A and B of the eight units of this warp.  In: yr[u], yi[u] = B fragments (fp16x2 pairs
// over a = 2t, 2t+1; column b = g).  Out: stored to the exchange buffer.
// BYTE_OFF: store through the precomputed byte offsets k.st_off (STS [R + UR], no LEA per store)
// instead of chunk indices.  Measured at config 4: the max / argmax kernel is 0.3 % slower with
// it, the kappa-sigma tails kernel (higher register pressure) 2.5 % faster: used there only.
template <bool BYTE_OFF = false>
__device__ __forceinline__ void chain1(const ConstsT<false> &k, const uint32_t (&yr)[8],
                                       const uint32_t (&yi)[8], uint4 *exch, int tid)
{
    const int w = tid >> 5, g = (tid >> 2) & 7, t = tid & 3;
    cpair v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        float d[4];
        mma_z(d, k.w8, yr[u], yi[u]);                 // alpha = g; b = 2t, 2t+1
        const cpair p = cmul2(d, k.twAB);
        float f[4];
        mma_z(f, k.w8, pack_h2(p.r.x, p.r.y), pack_h2(p.i.x, p.i.y));   // beta = g; alpha = 2t, 2t+1
        v[u] = cmul2(f, k.twBig[u]);
    }
    const int chunk0 = (w & 7) * 4 + 2 * (w >> 3);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int U = 2 * t + e + 8 * g;
#pragma unroll
        for (int p = 0; p < 2; ++p) {                 // c pair (4 cq + 2 p, + 1): units 4p + h, 4p + 2 + h
            uint4 q;
            q.x = e ? pack_h2(v[4 * p].r.y, v[4 * p + 2].r.y) : pack_h2(v[4 * p].r.x, v[4 * p + 2].r.x);
            q.y = e ? pack_h2(v[4 * p].i.y, v[4 * p + 2].i.y) : pack_h2(v[4 * p].i.x, v[4 * p + 2].i.x);
            q.z = e ? pack_h2(v[4 * p + 1].r.y, v[4 * p + 3].r.y) : pack_h2(v[4 * p + 1].r.x, v[4 * p + 3].r.x);
            q.w = e ? pack_h2(v[4 * p + 1].i.y, v[4 * p + 3].i.y) : pack_h2(v[4 * p + 1].i.x, v[4 * p + 3].i.x);
            if (BYTE_OFF) *reinterpret_cast<uint4 *>(reinterpret_cast<unsigned char *>(exch) + k.st_off[2 * e + p]) = q;
            else exch[exch_chunk(U, chunk0 + p)] = q;
        }
    }
}

template <bool BYTE_OFF = false>     // (ignored by the all-fp16 variant)
__device__ __forceinline__ void chain1(const ConstsT<true> &k, const uint32_t (&yr)[8],
                                       const uint32_t (&yi)[8], uint4 *exch, int tid)
{
    const int w = tid >> 5, g = (tid >> 2) & 7, t = tid & 3;
    hpair v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        uint32_t d[2], f[2];
        mma_h(d, k.w8, yr[u], yi[u]);                 // alpha = g; b = 2t, 2t+1
        const hpair p = cmul2(d, k.twAB);
        mma_h(f, k.w8, p.r, p.i);                     // beta = g; alpha = 2t, 2t+1
        v[u] = cmul2(f, k.twBig[u]);
    }
    const int chunk0 = (w & 7) * 4 + 2 * (w >> 3);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int U = 2 * t + e + 8 * g;
        const uint32_t sel = e ? 0x7632u : 0x5410u;   // the e-th halves of two words
#pragma unroll
        for (int p = 0; p < 2; ++p) {                 // c pair (4 cq + 2 p, + 1): units 4p + h, 4p + 2 + h
            uint4 q;
            q.x = __byte_perm(v[4 * p].r, v[4 * p + 2].r, sel);
            q.y = __byte_perm(v[4 * p].i, v[4 * p + 2].i, sel);
            q.z = __byte_perm(v[4 * p + 1].r, v[4 * p + 3].r, sel);
            q.w = __byte_perm(v[4 * p + 1].i, v[4 * p + 3].i, sel);
            exch[exch_chunk(U, chunk0 + p)] = q;
        }
    }
}

// Passes C and D of unit U = 4 w + i.  Out (times S16): z = the two outputs (delta = g,
// gamma = 2t + e), e = 0, 1, by component; with FULL also zu = (delta = 8 + g, ..) using the
// extra A fragments w16u.
// Pass C of one unit in either arithmetic: the four B-fragment words of pass D.
__device__ __forceinline__ void pass_c(const ConstsT<false> &k, const uint4 &q, uint32_t (&o)[4])
{
    float d0[4], d1[4];
    mma_z(d0, k.w8, q.x, q.y);                        // gamma = g; d' = 2t, 2t+1
    mma_z(d1, k.w8, q.z, q.w);                        // gamma = g; d' = 8 + 2t, + 1
    const cpair a = cmul2(d0, k.twC[0]);
    const cpair b = cmul2(d1, k.twC[1]);
    o[0] = pack_h2(a.r.x, a.r.y); o[1] = pack_h2(a.i.x, a.i.y);
    o[2] = pack_h2(b.r.x, b.r.y); o[3] = pack_h2(b.i.x, b.i.y);
}
__device__ __forceinline__ void pass_c(const ConstsT<true> &k, const uint4 &q, uint32_t (&o)[4])
{
    uint32_t d0[2], d1[2];
    mma_h(d0, k.w8, q.x, q.y);
    mma_h(d1, k.w8, q.z, q.w);
    const hpair a = cmul2(d0, k.twC[0]);
    const hpair b = cmul2(d1, k.twC[1]);
    o[0] = a.r; o[1] = a.i; o[2] = b.r; o[3] = b.i;
}

template <bool FULL, bool HALF>
__device__ __forceinline__ void chain2(const ConstsT<HALF> &k, const uint4 *exch, int U, int lane,
                                       cpair &z, cpair &zu, const uint32_t (&w16u)[2][3])
{
    const uint4 q = exch[exch_chunk(U, lane)];
    uint32_t o[4];
    pass_c(k, q, o);
    float f[4];
    mma_z(f, k.w16[0], o[0], o[1]);
    mma_acc(f, k.w16[1], o[2], o[3]);
    z.r = make_float2(f[0], f[1]);
    z.i = make_float2(f[2], f[3]);
    if (FULL) {
        float h[4];
        mma_z(h, w16u[0], o[0], o[1]);
        mma_acc(h, w16u[1], o[2], o[3]);
        zu.r = make_float2(h[0], h[1]);
        zu.i = make_float2(h[2], h[3]);
    }
}

// Where input element m = 1024 a + 128 b + 16 c + d' lives: (thread, 32-bit word, half) of the
// per-thread operand layout [chunk ci][thread][4 words {Re h0, Im h0, Re h1, Im h1}] used for
// the data spectra in global memory and for G in shared memory.
__device__ __forceinline__ void operand_slot(int m, int &word, int &half)
{
    const int a = m >> 10, b = (m >> 7) & 7, c = (m >> 4) & 7, dp = m & 15;
    const int tid = ((c >> 2) * 8 + (dp & 7)) * 32 + b * 4 + (a >> 1);
    word = ((c & 3) * NT + tid) * 4 + (dp >> 3) * 2;     // + 1 for the imaginary part
    half = a & 1;
}

}  // namespace tc
}  // namespace bfly
