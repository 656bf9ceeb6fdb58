// BFLY_FORM_FFT_TC: batched overlap-save FFT correlate whose butterflies run on the tensor cores
// (rows A3-A7 of DESIGN.md; the paper's method is FFT correlation).
//
// Same mathematics as bfly_fft.cu: with g[k] = exp(-i phi_k) zero-padded to B = 8192,
//     z_b = F+( X_b . G ),  G = F+(g),  X_b = conj(F+(x_b)) / B,   c = Re z, s = -Im z,
// but each block yields V = 4096 lags (outputs n < 4096 of the transform; the rows delta >= 8 of
// the last pass are never computed), and the transform is the four-pass tensor-core FFT of
// bfly_fft_tc.cuh.  Per (template, block): 4 x 16-byte loads of X_b per thread (fp16, stored by
// tc_spectra_kernel in the operand layout of the first pass), X_b . G in packed fp16, 512
// mma.sync, one trip through shared memory, fp32 epilogue.  G lives in shared memory in the
// same operand layout.  Lags past the last whole block (n_lags mod 4096 <= MAX_TAIL, e.g. the
// 61441st lag of a 16-s segment) are direct fp32 sums taken while the template is synthesised.
//
// Data scaling: every block of x is multiplied by a power of two that puts its rms in [1, 2)
// (rho is scale invariant), so all intermediates sit well inside the fp16 range; the factor is
// folded, in float64, into the per-lag normaliser tc_norm_kernel writes.
#include <type_traits>

#include "bfly_fft32.cuh"
#include "bfly_fft_tc.cuh"

namespace bfly {

namespace {

using namespace tc;

// Arithmetic of passes A .. C (bfly_fft_tc.cuh): true = all-fp16 (fp16-accumulate MMAs, half2
// twiddles), false = fp32 accumulators and twiddles, fp16 operands only.  Measured at config 4:
// all-fp16 is 1.13x faster (1.34 s against 1.51 s per step) with 2.2x the error (rms |d rho|
// 2.4e-5 against 1.1e-5, maximum over a few hundred templates 9.7e-5 against 3.6e-5) and loses
// the noise-free rho = 1 case to the 2e-4 tolerance, so the fp32 variant is the one built.
#ifndef BFLY_TC_HALF
#define BFLY_TC_HALF 0
#endif
constexpr bool TC_HALF = BFLY_TC_HALF != 0;

typedef ConstsT<TC_HALF> Consts;

// ------------------------------------------------------------------------------------------
// Data-block spectra: X_b = conj(F+(x_b 2^s)) / B by the fp32 transform of bfly_fft32.cuh,
// rounded to fp16 and scattered into the operand layout.  qs[b] = 2^(-2s) / S16^2.
__global__ void __launch_bounds__(fft32::NT, 1)
tc_spectra_kernel(const float *__restrict__ x, int64_t n_samples, int64_t lag_begin,
                  __half *__restrict__ xh, double *__restrict__ qs)
{
    extern __shared__ float2 smem[];
    __shared__ float esum[fft32::NT / 32];
    const fft32::Smem sm = fft32::carve(smem);
    const int t = threadIdx.x;
    fft32::fill_tables(sm, t);
    const int64_t off = lag_begin + (int64_t)blockIdx.x * TCV;
    float2 v[fft32::PTS];
    float e = 0.0f;
#pragma unroll
    for (int s = 0; s < fft32::PTS; ++s) {
        const int64_t gi = off + t + fft32::NT * s;
        const float xv = gi < n_samples ? __ldg(x + gi) : 0.0f;
        v[s] = make_float2(xv, 0.0f);
        e = fmaf(xv, xv, e);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((t & 31) == 0) esum[t >> 5] = e;
    __syncthreads();
    float tot = 0.0f;
#pragma unroll
    for (int w = 0; w < fft32::NT / 32; ++w) tot += esum[w];      // same order in every thread
    float sc = 1.0f;
    if (tot > 0.0f && isfinite(tot)) {
        int ex;
        frexpf(sqrtf(tot * (1.0f / (float)FFT_B)), &ex);          // rms = m 2^ex, m in [0.5, 1)
        sc = ldexpf(1.0f, 1 - ex);
    }
#pragma unroll
    for (int s = 0; s < fft32::PTS; ++s) v[s].x *= sc;
    fft32::fft8192(v, sm, t);
    __half *out = xh + (int64_t)blockIdx.x * (2 * EXCH_WORDS);
    const float nb = 1.0f / (float)FFT_B;
#pragma unroll
    for (int s = 0; s < fft32::PTS; ++s) {
        int word, half;
        operand_slot(t + fft32::NT * s, word, half);
        out[2 * word + half] = __float2half_rn(v[s].x * nb);
        out[2 * (word + 1) + half] = __float2half_rn(-v[s].y * nb);
    }
    if (t == 0) qs[blockIdx.x] = 1.0 / ((double)sc * (double)sc * (double)S16 * (double)S16);
}

// Per-lag normaliser in the order the epilogue reads it: rn2p[b][thread][2 i + e] belongs to lag
// b 4096 + (4 w + i) + 64 (2t + e) + 512 g and holds qs[b] / n2 (0 if the window is all zero,
// -inf past the last lag so that such a slot never wins the maximum).  float64 sums as in A2.
__global__ void __launch_bounds__(256)
tc_norm_kernel(const float *__restrict__ x, int32_t L, int64_t lag_begin, int64_t n_fft_lags,
               const double *__restrict__ qs, float *__restrict__ rn2p, int64_t n_slots, int tails)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_slots) return;
    const int slot = (int)(idx & 7), tid = (int)((idx >> 3) & (NT - 1));
    const int64_t b = idx >> 12;
    const int w = tid >> 5, g = (tid >> 2) & 7, t = tid & 3;
    const int n = (4 * w + (slot >> 1)) + 64 * (2 * t + (slot & 1)) + 512 * g;
    const int64_t i = b * TCV + n;
    if (tails) {       // kappa-sigma tails: the block's scale alone, 0 past the last lag (never a hit)
        rn2p[idx] = i < n_fft_lags ? (float)qs[b] : 0.0f;
        return;
    }
    if (i >= n_fft_lags) { rn2p[idx] = -INFINITY; return; }
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
    rn2p[idx] = n2 > 0.0 ? (float)(qs[b] / n2) : 0.0f;
}

// ------------------------------------------------------------------------------------------
// The predictor step of the kappa-sigma tails (sigma "computed in a predictor step by
// Parseval's Theorem"; readings S1-S3 of DESIGN.md).  With R[d] the circular autocorrelation of
// the N-sample segment, sum_tau |z~(tau)|^2 of the circular correlation z~ of the segment with a
// template g of L <= B/2 samples is sum_d R[d] A_g[d] = (1/B) sum_m |G[m]|^2 W[m], where A_g is the
// template's autocorrelation, G its length-B spectrum (the one the correlate kernel computes
// anyway) and W the length-B transform of R restricted to |d| < L: one dot product per template.
__global__ void __launch_bounds__(256)
tc_autocorr_kernel(const float *__restrict__ x, int64_t n_samples, double *__restrict__ racf)
{
    __shared__ double part[8];
    const int64_t d = blockIdx.x;
    double a = 0.0;
    for (int64_t n = threadIdx.x; n < n_samples; n += 256) {
        int64_t m = n + d;
        if (m >= n_samples) m -= n_samples;
        a = fma((double)__ldg(x + n), (double)__ldg(x + m), a);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += part[w];
        racf[d] = t;
    }
}

// W[m] = sum_{|d| < L} R[|d|] exp(2 pi i m d / B) (real), written where the correlate kernel's
// threads find it next to G: float index word + half of operand_slot(m).
__global__ void __launch_bounds__(fft32::NT, 1)
tc_wspec_kernel(const double *__restrict__ racf, int32_t L, float *__restrict__ wspec)
{
    extern __shared__ float2 smem[];
    const fft32::Smem sm = fft32::carve(smem);
    const int t = threadIdx.x;
    fft32::fill_tables(sm, t);
    float2 v[fft32::PTS];
#pragma unroll
    for (int s = 0; s < fft32::PTS; ++s) {
        const int d = t + fft32::NT * s;
        float r = 0.0f;
        if (d < L) r = (float)racf[d];
        else if (FFT_B - d < L) r = (float)racf[FFT_B - d];
        v[s] = make_float2(r, 0.0f);
    }
    fft32::fft8192(v, sm, t);
#pragma unroll
    for (int s = 0; s < fft32::PTS; ++s) {
        int word, half;
        operand_slot(t + fft32::NT * s, word, half);
        wspec[word + half] = v[s].x;
    }
}

// ------------------------------------------------------------------------------------------
// Shared memory of tc_correlate_kernel (208 KB of the SM's 227 KB; one CTA per SM).
struct TcSmem {
    uint4 *exch;               // three exchange buffers, cycled by the block pipeline
    uint4 *gs;                 // G in the operand layout, fp16
    uint4 *xs;                 // two staging slots for X_b (filled by cp.async.bulk)
    float *xt;                 // x[first tail lag ..], L + MAX_TAIL - 1 samples at xt_slot(n) (direct tail lags)
    uint32_t *w16u;            // [2][3][32]: A fragments of W16 rows 8..15 (G transform only)
    float *tail;               // [2][16 warps][2 MAX_TAIL] partial sums of the direct tail lags
    unsigned long long *red;   // [2][16]
    float *icv;                // [2]: inc2 of the template whose maxima sit in red[parity] (for write_out)
    unsigned char *par;        // [2][32]: {phA, phB, phC, inc2, ins2} of the template after this one
    unsigned long long *bar;   // mbarriers: [0..2] exchange buffer full, [3..4] X_b slot filled
};
constexpr int N_EXCH = 3;
constexpr int OUT_TID = 12 * 32;                             // the thread that combines and writes a template's outputs
constexpr int COPY_TID = 15 * 32;                                        // the thread that issues the bulk copies and the parameter prefetch
constexpr size_t OFF_GS = (size_t)N_EXCH * EXCH_WORDS * 4;
constexpr size_t OFF_XS = OFF_GS + EXCH_WORDS * 4;
constexpr size_t OFF_XT = OFF_XS + 2 * EXCH_WORDS * 4;
constexpr size_t OFF_W16U = OFF_XT + (FFT_MAX_L + 32) * 4;
constexpr size_t OFF_TAIL = OFF_W16U + 2 * 3 * 32 * 4;
constexpr size_t OFF_RED = OFF_TAIL + 2 * 16 * 2 * MAX_TAIL * 4;   // tail[] is double buffered by template parity
constexpr size_t OFF_BAR = OFF_RED + 2 * 4 * 16 * 8;          // red[parity][segment][warp]
constexpr size_t OFF_PAR = OFF_BAR + 8 * 8;                   // two slots of prefetched bank parameters
constexpr size_t OFF_ICV = OFF_PAR + 2 * 32;                 // 1 / ||cos phi||^2 of the two templates in flight
constexpr size_t TC_SMEM = OFF_ICV + 16;
__device__ __forceinline__ TcSmem carve_tc(unsigned char *base)
{
    TcSmem s;
    s.exch = reinterpret_cast<uint4 *>(base);
    s.gs = reinterpret_cast<uint4 *>(base + OFF_GS);
    s.xs = reinterpret_cast<uint4 *>(base + OFF_XS);
    s.xt = reinterpret_cast<float *>(base + OFF_XT);
    s.w16u = reinterpret_cast<uint32_t *>(base + OFF_W16U);
    s.tail = reinterpret_cast<float *>(base + OFF_TAIL);
    s.red = reinterpret_cast<unsigned long long *>(base + OFF_RED);
    s.bar = reinterpret_cast<unsigned long long *>(base + OFF_BAR);
    s.par = base + OFF_PAR;
    s.icv = reinterpret_cast<float *>(base + OFF_ICV);
    return s;
}

// cos and sin of the template phase at sample n from the top 32 bits of the fixed-point phase
// (A n + B n^2) 2^-64 cycles: the two products are taken modulo 2^64 and only their high words
// kept (error < 2^-31 cycle), the angle goes to the SFU (sin.approx / cos.approx: absolute error
// ~ 2^-21 on [-pi, pi], far below the fp16 rounding of g that follows).
__device__ __forceinline__ void synth_sincos(uint32_t Ahi, uint32_t Alo, uint32_t Bhi, uint32_t Blo,
                                             uint32_t n, float *s, float *c)
{
    const uint32_t n2 = n * n;                                   // n < 2^12
    const uint32_t ph = n * Ahi + __umulhi(n, Alo) + n2 * Bhi + __umulhi(n2, Blo);
    const float ang = (float)(int32_t)ph * 1.4629180792671596e-9f;   // pi 2^-31: angle in [-pi, pi)
    *s = __sinf(ang);
    *c = __cosf(ang);
}

// Where thread `th`'s 16-byte operand chunk of G sits inside a 512-chunk row of sm.gs: bit 3 of the
// thread index folded into bit 1 and bit 4 into bit 0.  The lanes of a warp that store G
// (transform output order) differ in bits 0, 2, 3, 4, 8 of the owning thread's index -- and the
// lanes of a half-warp in bits 2, 3, 4, 8 only --, so without the folds they hit 4 (2) of the 8
// 16-byte bank groups: ncu showed 16 wavefronts per 8-byte store with no fold, 8 with the first
// fold alone, 4 is the minimum (every lane writes the same half of its chunk).  The readers' lanes
// differ in bits 0-4, of which the folds keep bits 0-2 a permutation: still conflict free.
__device__ __forceinline__ int gs_slot(int th) { return th ^ ((th >> 2) & 2) ^ ((th >> 4) & 1); }

// (q & m8) | rank as ONE lop3 (LUT 0xEA = (a & b) | c); the compiler left to itself emits two
__device__ __forceinline__ float rank_key(float q, uint32_t m8, uint32_t rank)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r) : "r"(__float_as_uint(q)), "r"(m8), "r"(rank));
    return __uint_as_float(r);
}

// Index of tail-window sample n in sm.xt: a thread's lanes differ in bits 7-9 (g) and 11-12 (t)
// of n; folding those into the bank bits makes the reads conflict free.
__device__ __forceinline__ int xt_slot(int n) { return n ^ ((n >> 7) & 7) ^ (((n >> 11) & 3) << 3); }

// mbarrier / bulk-copy wrappers (PTX ISA: "mbarrier", "cp.async.bulk")
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}
// (No proxy fence: the destination slot was only READ through the generic proxy, and those reads
// are ordered before this copy by the mbarrier the issuing thread has waited on -- the
// consumer-release / producer-acquire pattern of every TMA pipeline.  fence.proxy.async is for
// generic WRITES that the async proxy must see; here it cost warp 0 a MEMBAR.ALL.CTA per block.)
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, void *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}

// cp.async (LDGSTS) of 8 / 4 bytes: the bank parameters of the CTA's next template travel to shared
// memory while the current template runs, so that no template starts with a DRAM round trip
__device__ __forceinline__ void cp_async8(void *dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void *dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr(dst)), "l"(src) : "memory");
}

// One CTA per SM, persistent, strided over the bank; one template at a time.  Per template: g is
// synthesised and transformed to G (two __syncthreads), then the blocks run as a software
// pipeline: passes A, B of block b + 1 are issued between the wait for the exchange buffer of
// block b and passes C, D of block b, so the only synchronisation inside the block loop is a
// split-phase mbarrier (one arrival per warp) that is normally already complete when waited on.
// Three exchange buffers make that safe: a warp writing buffer (b + 1) mod 3 has passed
// "full(b)", so every warp has finished passes A, B of block b and hence passes C, D of block
// b - 2, the previous user of that buffer.  X_b is staged by one 32 KB cp.async.bulk per block,
// two blocks ahead, into two slots (the sequence of blocks simply continues across templates).
// TAILS = true is the paper's own reduction instead of max / argmax (bfly_tails; readings S1-S3):
// per template sigma by the Parseval predictor above, then every valid lag whose magnitude
// exceeds kappa sigma is appended to a hit list (one atomic per hit; hits are rare by design).
struct TailArgs {
    const float4 *wspec;       // W in the operand layout (tc_wspec_kernel)
    double sig_norm;           // 1 / (2 N B): sum_m |G|^2 W -> sigma^2 ||cos phi||^2 (gs holds G itself)
    float kappa;
    float *sigma;              // [T]
    long long capacity;
    int32_t *hit_template, *hit_lag;
    float *hit_rho;
    unsigned long long *n_hits;
};

// Several data segments of equal length against the same bank in one launch (bfly_correlate_multi:
// the two detectors of PAPER.md:124, or consecutive chunks of a stream): the blocks of segment s
// are blocks s n_blocks .. (s + 1) n_blocks - 1 of xh / rn2p / qs; synthesis and the transform of g
// are done once per template, max / argmax per (template, segment).
constexpr int MAX_SEG = 4;
struct SegArgs {
    int32_t n_seg;
    const float *rn2[MAX_SEG];     // 1 / n2 of the segment's lags (tail lags)
    int64_t lag_begin[MAX_SEG];    // added to the block-relative lag of the maximum
    float *rho_max[MAX_SEG];
    int32_t *arg_lag[MAX_SEG];
};

// FAM: 0 = linear chirps (32-bit phase arithmetic), 1 = cubic phase (reading N1, 64-bit Horner),
// 2 = exponentially settling chirps (reading N2: phB / phC carry the doubles D tc and 1/(fs tc)).
// MULTI: several segments per launch (SegArgs; max / argmax mode only).  A separate instantiation,
// so that the single-segment kernel -- the headline path -- is compiled exactly as without it.
template <bool TAILS, int FAM, bool MULTI>
__global__ void __launch_bounds__(NT, 1)
tc_correlate_kernel(int64_t T, int32_t L, const uint64_t *__restrict__ phA,
                    const uint64_t *__restrict__ phB, const uint64_t *__restrict__ phC,
                    const float *__restrict__ inc2,
                    const float *__restrict__ ins2, const uint4 *__restrict__ xh,
                    const float4 *__restrict__ rn2p, const float *__restrict__ x,
                    const float *__restrict__ rn2, int64_t lag_begin,
                    int32_t n_blocks, int32_t n_tail, int32_t n_ftail, const double *__restrict__ qs,
                    float *__restrict__ rho_max, int32_t *__restrict__ arg_lag, const SegArgs sa, const TailArgs ta)
{
    // single segment: rn2, lag_begin, rho_max, arg_lag; MULTI: the same per segment in sa (the direct
    // tail sums and the tails mode are single-segment)
    const int32_t n_seg = MULTI ? sa.n_seg : 1;
    // n_tail: lags past the last block taken as direct sums during synthesis; n_ftail: such lags
    // taken from the transform of the last block instead (launch_tc_common decides; one of the two is 0)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const TcSmem sm = carve_tc(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, t = lane & 3;
    Consts k;
    make_consts(k, tid);
    if (w == 0) {
        uint32_t a[3];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            dft_frag(a, 16, S16, 8 + g, 8 * h + 2 * t);
#pragma unroll
            for (int q = 0; q < 3; ++q) sm.w16u[(h * 3 + q) * 32 + lane] = a[q];
        }
    }
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < N_EXCH; ++i) mbar_init(sm.bar + i, NT / 32);
        mbar_init(sm.bar + 3, 1);
        mbar_init(sm.bar + 4, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (n_tail > 0)
        for (int i = tid; i < L + n_tail - 1; i += NT)
            sm.xt[xt_slot(i)] = __ldg(x + lag_begin + (int64_t)n_blocks * TCV + i);
    __syncthreads();

    constexpr uint32_t XB_BYTES = EXCH_WORDS * 4;
    const uint32_t nowu[2][3] = {{0, 0, 0}, {0, 0, 0}};
    // templates of this CTA and the running sequence of its blocks (COPY_TID issues the copies)
    const int64_t my_templates = blockIdx.x < T ? (T - 1 - blockIdx.x) / gridDim.x + 1 : 0;
    const int32_t seq_blocks = MULTI ? n_blocks * n_seg : n_blocks;   // blocks per template, all segments
    const uint64_t total_blocks = (uint64_t)my_templates * (uint64_t)seq_blocks;
    uint64_t issued = 0;                               // COPY_TID: X_b copies issued so far
    int32_t next_b = 0;                                // COPY_TID: block index of copy `issued`
    if (tid == COPY_TID)
        for (; issued < 2 && issued < total_blocks; ++issued) {
            mbar_expect_tx(sm.bar + 3 + (int)issued, XB_BYTES);
            bulk_load(sm.xs + issued * (EXCH_WORDS / 4), xh + (int64_t)next_b * (EXCH_WORDS / 4), XB_BYTES,
                      sm.bar + 3 + (int)issued);
            next_b = next_b + 1 == seq_blocks ? 0 : next_b + 1;
        }
    uint32_t m8 = 0xFFFFFFF8u;                         // in a register, so that (q & m8) | rank is one LOP3
    asm volatile("" : "+r"(m8));
    int gs_tid = gs_slot(tid);                         // held in a register: recomputing it costs the block loop two instructions
    asm volatile("" : "+r"(gs_tid));
    uint32_t xcnt = 0;                                 // blocks consumed: slot = xcnt & 1, parity = (xcnt >> 1) & 1
    int wb = 0, rb = 0;                                // exchange buffer written next / read next
    uint32_t fpar = 0;                                 // bit i: parity to wait for on "full(i)"

    auto prefetch_params = [&](int64_t jn, int slot) {            // COPY_TID only
        unsigned char *d = sm.par + 32 * slot;
        cp_async8(d, phA + jn);
        cp_async8(d + 8, phB + jn);
        if (FAM != 0) cp_async8(d + 16, phC + jn);
        cp_async4(d + 24, inc2 + jn);
        cp_async4(d + 28, ins2 + jn);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (tid == COPY_TID && blockIdx.x < T) {
        prefetch_params(blockIdx.x, 0);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    // OUT_TID: combine the warps' maxima of a finished template (red[slot]) and write its outputs
    auto write_out = [&](int64_t jo, int slot) {
        if (!MULTI) {
            const unsigned long long *red = sm.red + 16 * slot;
            unsigned long long p = red[0];
#pragma unroll
            for (int ww = 1; ww < 16; ++ww) p = red[ww] > p ? red[ww] : p;
            if (p == 0ull) {                            // rho = 0 at every lag (or no lag at all)
                rho_max[jo] = 0.0f;
                arg_lag[jo] = (int32_t)lag_begin;
            } else {
                const float ico = sm.icv[slot];
                rho_max[jo] = sqrtf(__uint_as_float((uint32_t)(p >> 32)) * ico);
                arg_lag[jo] = (int32_t)(lag_begin + (int64_t)(0xFFFFFFFFu - (uint32_t)(p & 0xFFFFFFFFull)));
            }
            return;
        }
        const float ico = sm.icv[slot];
        for (int sg = 0; sg < n_seg; ++sg) {
            const unsigned long long *red = sm.red + 16 * (MAX_SEG * slot + sg);
            unsigned long long p = red[0];
#pragma unroll
            for (int ww = 1; ww < 16; ++ww) p = red[ww] > p ? red[ww] : p;
            if (p == 0ull) {                            // rho = 0 at every lag (or no lag at all)
                sa.rho_max[sg][jo] = 0.0f;
                sa.arg_lag[sg][jo] = (int32_t)sa.lag_begin[sg];
            } else {
                sa.rho_max[sg][jo] = sqrtf(__uint_as_float((uint32_t)(p >> 32)) * ico);
                sa.arg_lag[sg][jo] = (int32_t)(sa.lag_begin[sg] + (int64_t)(0xFFFFFFFFu - (uint32_t)(p & 0xFFFFFFFFull)));
            }
        }
    };
    // No CTA-wide barrier separates one template from the next: the first barrier of a template
    // (after its synthesis) is where every warp is known to have left the previous one.  Until
    // then a warp of template j + 1 writes only red[], tail[] (both double buffered by template
    // parity) and the exchange buffer `wb`, whose last reader was block n_blocks - 3 of template j
    // (finished by every warp: the writer has passed full(n_blocks - 1)).  The next template's
    // parameters are published by the arrival of COPY_TID in the front half of the last block.
    int ps = 0;                                                  // parameter slot / red[] / tail[] half of this template
    int64_t j = blockIdx.x;
    for (; j < T; j += gridDim.x, ps ^= 1) {
        // ---- A3: synthesise g[n] = cos phi_n - i r sin phi_n, r = ||cos phi|| / ||sin phi||,
        //      n = 1024 a + 128 g + 16 c + d' < L, as the operand fragments of pass A (so that
        //      |z|^2 / ||cos phi||^2 is the quadrature sum); direct sums for the tail lags
        const unsigned char *pp = sm.par + 32 * ps;
        const uint64_t A = *reinterpret_cast<const uint64_t *>(pp), Bq = *reinterpret_cast<const uint64_t *>(pp + 8);
        const uint64_t Cq = FAM != 0 ? *reinterpret_cast<const uint64_t *>(pp + 16) : 0ull;
        const uint32_t Ahi = (uint32_t)(A >> 32), Alo = (uint32_t)A;
        const uint32_t Bhi = (uint32_t)(Bq >> 32), Blo = (uint32_t)Bq;
        const float ic = *reinterpret_cast<const float *>(pp + 24);
        // ic > 0 (cos phi_0 = 1); fast division and square root: r enters g before its fp16 rounding
        const float rq = __fsqrt_rn(__fdividef(*reinterpret_cast<const float *>(pp + 28), ic));
        // The index arithmetic of the per-template code below depends on the thread only, so the
        // compiler would hoist it out of the template loop and hold its results in registers all
        // through the block loop -- which is at the 128-register limit and then recomputes its OWN
        // addresses on every block (measured: +24 instructions per block).  An opaque copy of the
        // thread index keeps that arithmetic here, where it costs a few dozen cheap instructions
        // per template.
        int ptid = tid;
        asm volatile("" : "+r"(ptid));
        const int pl = ptid & 31, pw = ptid >> 5, pg = pl >> 2, pt = pl & 3;
        {
            // The samples n >= 4096 are zero padding, so only the lanes t < 2 own non-zero operand
            // words; the work is split over all four lanes of a group: lane t synthesises, for the
            // owner lane t & 1, the units u = 4 (t >> 1) .. + 3, and the owners fetch the upper
            // four units from lane + 2 by shuffle.
            uint32_t yr[8], yi[8];
            float tc_[MAX_TAIL], ts_[MAX_TAIL];
#pragma unroll
            for (int r = 0; r < MAX_TAIL; ++r) tc_[r] = ts_[r] = 0.0f;
            const int to = pt & 1, uh = pt >> 1;
            uint32_t pr[4], pi[4];
            // (templates of the full 4096 samples -- every config but one -- need no n < L test: a
            // uniform branch picks the instantiation without it)
            auto synth = [&](auto checked) {
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
                const int c = 4 * (pw >> 3) + 2 * uh + (kk >> 1), dp = (pw & 7) + 8 * (kk & 1);
                float cs[2], sn[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int n = 1024 * (2 * to + e) + 128 * pg + 16 * c + dp;
                    cs[e] = sn[e] = 0.0f;
                    if (!decltype(checked)::value || n < L) {
                        if (FAM == 0) {              // linear chirp
                            synth_sincos(Ahi, Alo, Bhi, Blo, (uint32_t)n, &sn[e], &cs[e]);
                        } else {                     // N1: cubic phase, full 64-bit Horner; N2: settling
                            const uint64_t p64 = FAM == 1 ? template_phase(A, Bq, Cq, (uint64_t)n)
                                                          : settle_phase(A, __longlong_as_double((long long)Bq),
                                                                         __longlong_as_double((long long)Cq), (uint64_t)n);
                            const uint32_t ph = (uint32_t)(p64 >> 32);
                            const float ang = (float)(int32_t)ph * 1.4629180792671596e-9f;
                            sn[e] = __sinf(ang);
                            cs[e] = __cosf(ang);
                        }
                        sn[e] *= rq;
                        if (n_tail > 0) {
                            const float xv = sm.xt[xt_slot(n)];
                            tc_[0] = fmaf(xv, cs[e], tc_[0]);
                            ts_[0] = fmaf(xv, sn[e], ts_[0]);
                            if (n_tail > 1) {
#pragma unroll
                                for (int r = 1; r < MAX_TAIL; ++r) {
                                    const float xr = r < n_tail ? sm.xt[xt_slot(n + r)] : 0.0f;
                                    tc_[r] = fmaf(xr, cs[e], tc_[r]);
                                    ts_[r] = fmaf(xr, sn[e], ts_[r]);
                                }
                            }
                        }
                    }
                }
                pr[kk] = pack_h2(cs[0], cs[1]);
                pi[kk] = pack_h2(-sn[0], -sn[1]);
            }
            };
            if (L == FFT_MAX_L) synth(std::false_type{});
            else synth(std::true_type{});
            const bool owner = pt < 2;
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
                const uint32_t ur = __shfl_down_sync(0xffffffffu, pr[kk], 2);
                const uint32_t ui = __shfl_down_sync(0xffffffffu, pi[kk], 2);
                yr[kk] = owner ? pr[kk] : 0u;
                yi[kk] = owner ? pi[kk] : 0u;
                yr[4 + kk] = owner ? ur : 0u;
                yi[4 + kk] = owner ? ui : 0u;
            }
            if (n_tail > 0) {
#pragma unroll
                for (int r = 0; r < MAX_TAIL; ++r) {
                    if (r >= n_tail) break;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        tc_[r] += __shfl_xor_sync(0xffffffffu, tc_[r], o);
                        ts_[r] += __shfl_xor_sync(0xffffffffu, ts_[r], o);
                    }
                    if (pl == 0) {
                        float *tl = sm.tail + ps * (16 * 2 * MAX_TAIL);
                        tl[(pw * MAX_TAIL + r) * 2] = tc_[r];
                        tl[(pw * MAX_TAIL + r) * 2 + 1] = ts_[r];
                    }
                }
            }
            chain1<TAILS>(k, yr, yi, sm.exch + wb * (EXCH_WORDS / 4), tid);
        }
        __syncthreads();                                // every warp has left the previous template
        // (the per-template chores are spread over warps 0, 8 and 12 so that no warp trails the others
        // into the next barrier: COPY_TID (lane 0 of warp 15: the highest warp index is favoured by the issue arbiter and so has
        // slack for the extra work; measured -0.3 % against warp 0) owns the copies, OUT_TID the outputs,
        // warp 8 the tail lags)
        if (tid == OUT_TID && !TAILS && j != (int64_t)blockIdx.x) write_out(j - gridDim.x, ps ^ 1);
        if (tid == COPY_TID && j + gridDim.x < T) prefetch_params(j + gridDim.x, ps ^ 1);
        // ---- G = F+(g): all 16 rows of the last pass; G / S16 -> fp16 -> operand layout
        {
            uint32_t w16u[2][3];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < 3; ++q) w16u[h][q] = sm.w16u[(h * 3 + q) * 32 + lane];
            // output m = U + 64 (2t + e) + 512 g + 4096 up (U = 4w + i) lives in operand_slot(m):
            // thread ((e 8 + (U & 7)) 32 + (t + 4 (g & 1)) 4 + (g >> 2) + 2 up), word pair
            // (U >> 3) & 1 of chunk U >> 4, half (g >> 1) & 1.  The lanes g and g ^ 2 hold the two
            // halves of the same words: they exchange by shuffle, the lane with bit 1 of g clear
            // writes the e = 0 words, the other the e = 1 words, {Re, Im} as one 8-byte store.
            uint32_t *gw = reinterpret_cast<uint32_t *>(sm.gs);
            const float2 r16 = make_float2(1.0f / S16, 1.0f / S16);
            const int gb1 = (pg >> 1) & 1;
            const uint32_t sel = gb1 ? 0x3276u : 0x5410u;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                cpair z, zu;
                chain2<true, TC_HALF>(k, sm.exch + wb * (EXCH_WORDS / 4), 4 * w + i, lane, z, zu, w16u);
                const int U = 4 * pw + i;
                const float2 a0 = __fmul2_rn(z.r, r16), b0 = __fmul2_rn(z.i, r16);
                const float2 a1 = __fmul2_rn(zu.r, r16), b1 = __fmul2_rn(zu.i, r16);
                const uint32_t R0 = pack_h2(a0.x, a0.y), I0 = pack_h2(b0.x, b0.y);     // (e = 0, e = 1)
                const uint32_t R1 = pack_h2(a1.x, a1.y), I1 = pack_h2(b1.x, b1.y);
                const uint32_t oR0 = __shfl_xor_sync(0xffffffffu, R0, 8), oI0 = __shfl_xor_sync(0xffffffffu, I0, 8);
                const uint32_t oR1 = __shfl_xor_sync(0xffffffffu, R1, 8), oI1 = __shfl_xor_sync(0xffffffffu, I1, 8);
                const int tid0 = (gb1 * 8 + (U & 7)) * 32 + (pt + 4 * (pg & 1)) * 4 + (pg >> 2);
                const int word0 = ((U >> 4) * NT + gs_slot(tid0)) * 4 + ((U >> 3) & 1) * 2;
                *reinterpret_cast<uint2 *>(gw + word0) = make_uint2(__byte_perm(R0, oR0, sel), __byte_perm(I0, oI0, sel));
                *reinterpret_cast<uint2 *>(gw + (word0 ^ 8)) = make_uint2(__byte_perm(R1, oR1, sel), __byte_perm(I1, oI1, sel));   // thread tid0 + 2
            }
        }
        // ---- the segments of this template (one pass; more with bfly_correlate_multi).  The barrier
        //      at the head of a pass is "G is in place" for the first and the segment boundary for the
        //      others (ptxas needs a barrier between the divergent end of a pass and the block loop
        //      to keep that loop on the uniform datapath).
        int sg = 0;
        float thr = 0.0f, rsig2 = 0.0f;               // TAILS: kappa^2 sigma^2 / inc2 and inc2 / sigma^2
        do {
        __syncthreads();
        if (TAILS) {
            float acc = 0.0f;
#pragma unroll
            for (int ci = 0; ci < 4; ++ci) {
                const uint4 gq = sm.gs[ci * NT + gs_slot(tid)];
                const float4 wv = __ldg(ta.wspec + ci * NT + tid);
                const float2 r0 = __half22float2(as_h2(gq.x)), i0 = __half22float2(as_h2(gq.y));
                const float2 r1 = __half22float2(as_h2(gq.z)), i1 = __half22float2(as_h2(gq.w));
                acc = fmaf(fmaf(r0.x, r0.x, i0.x * i0.x), wv.x, acc);
                acc = fmaf(fmaf(r0.y, r0.y, i0.y * i0.y), wv.y, acc);
                acc = fmaf(fmaf(r1.x, r1.x, i1.x * i1.x), wv.z, acc);
                acc = fmaf(fmaf(r1.y, r1.y, i1.y * i1.y), wv.w, acc);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            float *part = reinterpret_cast<float *>(sm.red);
            if (lane == 0) part[w] = acc;
            __syncthreads();
            double tot = 0.0;
#pragma unroll
            for (int ww = 0; ww < 16; ++ww) tot += (double)part[ww];      // same order in every thread
            const float s2c = (float)(tot * ta.sig_norm);                 // sigma^2 ||cos phi||^2 (>= 0 up to rounding)
            const float sig2 = fmaxf(s2c * ic, 0.0f);
            if (tid == 0) ta.sigma[j] = sqrtf(sig2);
            thr = ta.kappa * ta.kappa * fmaxf(s2c, 0.0f);
            rsig2 = sig2 > 0.0f ? ic / sig2 : 0.0f;
            if (!(thr > 0.0f)) thr = INFINITY;                           // sigma = 0: no hits (S3)
        }

        // ---- A4: passes A, B of one block: Y = X_b . G in packed fp16, straight into the
        //      fragments of pass A; result to exchange buffer wb; one arrival per warp
        auto front = [&]() {
            const int slot = xcnt & 1;
            mbar_wait(sm.bar + 3 + slot, (xcnt >> 1) & 1);
            ++xcnt;
            uint32_t yr[8], yi[8];
            const uint4 *xb = sm.xs + slot * (EXCH_WORDS / 4) + tid;
#pragma unroll
            for (int ci = 0; ci < 4; ++ci) {
                const uint4 xq = xb[ci * NT];
                const uint4 gq = sm.gs[ci * NT + gs_tid];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const __half2 xr = as_h2(h ? xq.z : xq.x), xi = as_h2(h ? xq.w : xq.y);
                    const __half2 gr = as_h2(h ? gq.z : gq.x), gi = as_h2(h ? gq.w : gq.y);
                    yr[2 * ci + h] = as_u32(__hfma2(__hneg2(xi), gi, __hmul2(xr, gr)));
                    yi[2 * ci + h] = as_u32(__hfma2(xi, gr, __hmul2(xr, gi)));
                }
            }
            chain1<TAILS>(k, yr, yi, sm.exch + wb * (EXCH_WORDS / 4), tid);
            __syncwarp();
            if (lane == 0) mbar_arrive(sm.bar + wb);
            wb = wb + 1 == N_EXCH ? 0 : wb + 1;
        };

        const float4 *rn2p_s = MULTI ? rn2p + (int64_t)sg * n_blocks * (NT * 2) : rn2p;
        const float *rn2_s = MULTI ? sa.rn2[sg] : rn2;
        const float4 *rp_run = rn2p_s + tid * 2;       // MULTI: this thread's normalisers, block by block
        // A7 inside the thread: the low three mantissa bits of q (2^-21 relative, far below the fp16
        // operand noise) are replaced by 7 - rank, rank = 4 e + i the order of the lag among the
        // thread's eight lags of a block (lag = .. + i + 64 e): the largest key is the largest q and,
        // on a tie, the smallest lag (reading C8) -- one LOP3 per lag and a tree of three-input
        // maxima instead of a compare, a select and an index update per lag (-9 instructions per
        // block).  bcmp = bkey with its low bits at 7, so that a later block wins only with a larger
        // q.  NaN keys (0 x -inf, or -inf with rank bits: lags past the last one) never win a maximum.
        float bkey = -1.0f, bcmp = -1.0f;
        int32_t bblk = 0;
        if (n_blocks > 0) front();
        for (int32_t b = 0; b < n_blocks; ++b) {
            mbar_wait(sm.bar + rb, (fpar >> rb) & 1);
            fpar ^= 1u << rb;
            // every warp has read the X slot of block b: refill it with the block two ahead
            if (tid == COPY_TID && issued < total_blocks) {
                const int slot = (int)(issued & 1);
                mbar_expect_tx(sm.bar + 3 + slot, XB_BYTES);
                bulk_load(sm.xs + slot * (EXCH_WORDS / 4), xh + (int64_t)next_b * (EXCH_WORDS / 4), XB_BYTES,
                          sm.bar + 3 + slot);
                next_b = next_b + 1 == seq_blocks ? 0 : next_b + 1;
                ++issued;
                // The next template's parameters (cp.async of COPY_TID, issued a whole G stage ago:
                // this wait does not stall) become visible to every warp through COPY_TID's arrivals
                // in the front halves that follow.  With n_blocks >= 2 this branch is taken in every
                // block iteration of a template that has a successor.
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            const uint4 *rbuf = sm.exch + rb * (EXCH_WORDS / 4);
            rb = rb + 1 == N_EXCH ? 0 : rb + 1;
            // ---- the two halves of an iteration: passes A, B of block b + 1 ("front"), then passes
            //      C, D + A5-A7 of block b ("back").  (Running them in the other order in half of the
            //      warps of every scheduler, so that tensor-pipe bursts meet FMA bursts, was measured
            //      slower: DESIGN.md 10.)
            auto back = [&]() {
                // ---- passes C, D and A5-A7 on the 8 lags of this thread
                const float4 *rp = MULTI ? rp_run : rn2p_s + ((int64_t)b * NT + tid) * 2;
                if (MULTI) rp_run += NT * 2;
                const float4 ra = __ldg(rp), rb4 = __ldg(rp + 1);
                const float2 rr[4] = {make_float2(ra.x, ra.y), make_float2(ra.z, ra.w),
                                      make_float2(rb4.x, rb4.y), make_float2(rb4.z, rb4.w)};
                float2 qs4[4];
                float qmax = 0.0f;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    cpair z, zu;
                    chain2<false, TC_HALF>(k, rbuf, 4 * w + i, lane, z, zu, nowu);
                    const float2 q = __fmul2_rn(__ffma2_rn(z.i, z.i, __fmul2_rn(z.r, z.r)), rr[i]);
                    if (TAILS) {
                        qs4[i] = q;
                        qmax = fmaxf(qmax, fmaxf(q.x, q.y));
                    } else {
                        qs4[i].x = rank_key(q.x, m8, 7u - i);
                        qs4[i].y = rank_key(q.y, m8, 3u - i);
                    }
                }
                if (!TAILS) {
                    const float bm = fmaxf(fmaxf(fmaxf(qs4[0].x, qs4[1].x), qs4[2].x),
                                           fmaxf(fmaxf(fmaxf(qs4[3].x, qs4[0].y), qs4[1].y),
                                                 fmaxf(fmaxf(qs4[2].y, qs4[3].y), -1.0f)));
                    if (bm > bcmp) { bkey = bm; bcmp = __uint_as_float(__float_as_uint(bm) | 7u); bblk = b; }
                }
                if (TAILS && qmax > thr) {                 // rare: at least one of this thread's 8 lags is a hit
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const float qe = e ? qs4[i].y : qs4[i].x;
                            if (qe > thr) {
                                const unsigned long long at = atomicAdd(ta.n_hits, 1ull);
                                if (at < (unsigned long long)ta.capacity) {
                                    ta.hit_template[at] = (int32_t)j;
                                    ta.hit_lag[at] = (int32_t)(lag_begin + (int64_t)b * TCV + (4 * w + i) + 64 * (2 * t + e) + 512 * g);
                                    ta.hit_rho[at] = sqrtf(qe * rsig2);
                                }
                            }
                        }
                    }
                }
            };
            if (b + 1 < n_blocks) front();
            back();
        }
        // ---- tail lags from the transform of the last block: lag n_blocks TCV + r is its output
        //      n = 4096 + r, i.e. row delta = 8 of the last pass (the rows chain2<FULL> adds) of unit
        //      U = r (any warp can run it: warp 8 does) -- lane 0 holds (gamma, delta) = (0, 8).  That buffer
        //      is intact: the next writers of it are two transforms away, behind the next barrier.
        if (n_ftail > 0 && w == 8) {
            const uint4 *lbuf = sm.exch + (rb == 0 ? N_EXCH - 1 : rb - 1) * (EXCH_WORDS / 4);
            uint32_t w16u[2][3];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < 3; ++q) w16u[h][q] = sm.w16u[(h * 3 + q) * 32 + lane];
            const float qsl = (float)__ldg(qs + ((MULTI ? sg * n_blocks : 0) + n_blocks - 1));
#pragma unroll 1
            for (int r = 0; r < n_ftail; ++r) {
                cpair z, zu;
                chain2<true, TC_HALF>(k, lbuf, r, lane, z, zu, w16u);
                const float m2 = fmaf(zu.i.x, zu.i.x, zu.r.x * zu.r.x) * qsl;
                if (lane == 0) {
                    if (TAILS) {
                        if (m2 > thr) {
                            const unsigned long long at = atomicAdd(ta.n_hits, 1ull);
                            if (at < (unsigned long long)ta.capacity) {
                                ta.hit_template[at] = (int32_t)j;
                                ta.hit_lag[at] = (int32_t)(lag_begin + (int64_t)n_blocks * TCV + r);
                                ta.hit_rho[at] = sqrtf(m2 * rsig2);
                            }
                        }
                    } else {
                        const float q = m2 * __ldg(rn2_s + (int64_t)n_blocks * TCV + r);
                        const float kq = rank_key(q, m8, 7u - (uint32_t)r);
                        if (kq > bcmp) { bkey = kq; bcmp = __uint_as_float(__float_as_uint(kq) | 7u); bblk = n_blocks; }
                    }
                }
            }
        }
        // ---- tail lags (direct sums) and the CTA-wide maximum, ties to the smallest lag
        if (n_tail > 0 && tid < n_tail) {
            const float *tl = sm.tail + ps * (16 * 2 * MAX_TAIL);
            float c = 0.0f, s = 0.0f;
            for (int ww = 0; ww < 16; ++ww) {
                c += tl[(ww * MAX_TAIL + tid) * 2];
                s += tl[(ww * MAX_TAIL + tid) * 2 + 1];
            }
            if (TAILS) {
                const float q = fmaf(s, s, c * c);                       // raw samples: no block scale
                if (q > thr) {
                    const unsigned long long at = atomicAdd(ta.n_hits, 1ull);
                    if (at < (unsigned long long)ta.capacity) {
                        ta.hit_template[at] = (int32_t)j;
                        ta.hit_lag[at] = (int32_t)(lag_begin + (int64_t)n_blocks * TCV + tid);
                        ta.hit_rho[at] = sqrtf(q * rsig2);
                    }
                }
            } else {
                const float q = fmaf(s, s, c * c) * __ldg(rn2_s + (int64_t)n_blocks * TCV + tid);
                const float kq = rank_key(q, m8, 7u - (uint32_t)tid);
                if (kq > bcmp) { bkey = kq; bcmp = __uint_as_float(__float_as_uint(kq) | 7u); bblk = n_blocks; }
            }
        }
        if (!TAILS) {
            unsigned long long p = 0ull;
            const float best = __uint_as_float(__float_as_uint(bkey) & 0xFFFFFFF8u);
            if (best > 0.0f) {                         // q = 0 everywhere: rho = 0 at the first lag (write_out)
                const int bb = bblk, rank = 7 - (int)(__float_as_uint(bkey) & 7u);   // rank = 4 e + i (tail lags: r)
                const uint32_t li = bb >= n_blocks ? (uint32_t)n_blocks * TCV + (uint32_t)rank
                                                   : (uint32_t)bb * TCV + (uint32_t)((4 * w + (rank & 3)) +
                                                                                     64 * (2 * t + (rank >> 2)) + 512 * g);
                p = ((unsigned long long)__float_as_uint(best) << 32) | (unsigned long long)(0xFFFFFFFFu - li);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long q = __shfl_xor_sync(0xffffffffu, p, o);
                p = q > p ? q : p;
            }
            if (lane == 0) sm.red[16 * ((MULTI ? MAX_SEG : 1) * ps + sg) + w] = p;   // combined by OUT_TID after the next template's first barrier
        }
        } while (MULTI && ++sg < n_seg);               // segments
        if (!TAILS && tid == 0) sm.icv[ps] = *reinterpret_cast<const float *>(sm.par + 32 * ps + 24);
        if (seq_blocks < 2) {                          // too few block iterations to publish the parameters through
            if (tid == COPY_TID) asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();
        }
    }
    if (!TAILS && blockIdx.x < T) {
        __syncthreads();
        if (tid == OUT_TID) write_out(j - gridDim.x, ps ^ 1);
    }
}

// Diagnostic: the bare transform on one natural-order input (bfly_debug_fft_tc).
__global__ void __launch_bounds__(NT, 1)
tc_debug_fft_kernel(const float2 *__restrict__ y, float2 *__restrict__ z, int full)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const TcSmem sm = carve_tc(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, t = lane & 3;
    Consts k;
    make_consts(k, tid);
    uint32_t w16u[2][3];
#pragma unroll
    for (int h = 0; h < 2; ++h) dft_frag(w16u[h], 16, S16, 8 + g, 8 * h + 2 * t);
    uint32_t yr[8], yi[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int c = 4 * (w >> 3) + (u >> 1), dp = (w & 7) + 8 * (u & 1);
        const int n0 = 1024 * (2 * t) + 128 * g + 16 * c + dp;
        const float2 v0 = y[n0], v1 = y[n0 + 1024];
        yr[u] = pack_h2(v0.x, v1.x);
        yi[u] = pack_h2(v0.y, v1.y);
    }
    chain1(k, yr, yi, sm.exch, tid);
    __syncthreads();
    const float r16 = 1.0f / S16;
    for (int i = 0; i < 4; ++i) {
        cpair o, ou;
        if (full) chain2<true, TC_HALF>(k, sm.exch, 4 * w + i, lane, o, ou, w16u);
        else chain2<false, TC_HALF>(k, sm.exch, 4 * w + i, lane, o, ou, w16u);
        for (int e = 0; e < 2; ++e) {
            const int m = (4 * w + i) + 64 * (2 * t + e) + 512 * g;
            z[m] = make_float2((e ? o.r.y : o.r.x) * r16, (e ? o.i.y : o.i.x) * r16);
            if (full) z[m + 4096] = make_float2((e ? ou.r.y : ou.r.x) * r16, (e ? ou.i.y : ou.i.x) * r16);
        }
    }
}

}  // namespace

// Blocks of 4096 lags done by the transform and lags left to the direct tail sums.
void tc_plan(int64_t n_lags, int64_t *n_blocks, int32_t *n_tail)
{
    int64_t nb = n_lags / TCV;
    int64_t rem = n_lags - nb * TCV;
    if (rem > MAX_TAIL) { nb += 1; rem = 0; }
    *n_blocks = nb;
    *n_tail = (int32_t)rem;
}

int64_t tc_blocks_needed(int64_t n_lags)
{
    int64_t nb; int32_t nt;
    tc_plan(n_lags, &nb, &nt);
    return nb;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize of every kernel of this file, once per device
static int tc_attrs(int device)
{
    static PerDeviceOnce once;
    return once.run(device, []() -> int {
        BFLY_CUDA(cudaFuncSetAttribute(tc_spectra_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft32::FFT_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_wspec_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft32::FFT_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<false, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<true, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<false, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<false, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<true, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<false, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<false, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_correlate_kernel<true, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        BFLY_CUDA(cudaFuncSetAttribute(tc_debug_fft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM));
        return BFLY_OK;
    });
}

// Whether the lags past the last whole block come from the last block's transform: output
// n = 4096 + r of that transform is a valid (unwrapped) lag while 4096 + r <= B - L; then the kernel
// takes them from the rows delta >= 8 (n_ftail) and the synthesis carries no direct sums.
static bool tail_from_transform(int32_t L, int64_t n_blocks, int32_t n_tail)
{
    return n_tail > 0 && n_blocks > 0 && (int64_t)(n_tail - 1) <= (int64_t)TCV - (int64_t)L;
}

// Several equal-length segments in one launch need every lag to come from a transform.
bool tc_multi_supported(int32_t L, int64_t n_lags)
{
    int64_t nb; int32_t nt;
    tc_plan(n_lags, &nb, &nt);
    return L >= BFLY_TC_MIN_L && nb > 0 && (nt == 0 || tail_from_transform(L, nb, nt));
}

// n_seg segments x[s] of n_samples samples each, the same lag range in each; rn2 of segment s at
// b->rn2 + s n_lags (written by the caller); spectra, scales and normalisers of segment s occupy
// blocks s n_blocks .. of the bank's workspace.
static int launch_tc_common(const bfly_bank *b, int n_seg, const float *const *x, int64_t n_samples,
                            int64_t lag_begin, int64_t lag_end, float *const *rho_max, int32_t *const *arg_lag,
                            const TailArgs *tails, cudaStream_t stream)
{
    int rc = tc_attrs(b->device);
    if (rc) return rc;
    const int64_t n_lags = lag_end - lag_begin;
    if (n_lags >= (1LL << 31) - 2 * TCV) { set_error("too many lags"); return BFLY_ERANGE; }
    int64_t n_blocks; int32_t n_tail;
    tc_plan(n_lags, &n_blocks, &n_tail);
    if (n_seg < 1 || n_seg > MAX_SEG || (n_seg > 1 && (tails || !tc_multi_supported(b->L, n_lags)))) {
        set_error("unsupported multi-segment launch (internal)");
        return BFLY_EINVAL;
    }
    if (n_seg * n_blocks * 2 * EXCH_WORDS > b->xh_cap || n_seg * n_blocks * TCV > b->rn2p_cap ||
        n_seg * n_blocks > b->qs_cap || (n_seg > 1 && n_seg * n_lags > b->rn2_cap)) {
        set_error("FFT workspace too small (internal)");
        return BFLY_EINVAL;
    }
    if (n_blocks > 0) {
        for (int sg = 0; sg < n_seg; ++sg) {
            tc_spectra_kernel<<<(unsigned)n_blocks, fft32::NT, fft32::FFT_SMEM, stream>>>(
                x[sg], n_samples, lag_begin, b->xh + (int64_t)sg * n_blocks * 2 * EXCH_WORDS, b->qs + sg * n_blocks);
            count_launch();
            BFLY_CUDA(cudaGetLastError());
            const int64_t n_slots = n_blocks * TCV;
            tc_norm_kernel<<<(unsigned)((n_slots + 255) / 256), 256, 0, stream>>>(
                x[sg], b->L, lag_begin, n_lags - n_tail, b->qs + sg * n_blocks, b->rn2p + (int64_t)sg * n_slots, n_slots,
                tails ? 1 : 0);
            count_launch();
            BFLY_CUDA(cudaGetLastError());
        }
    }
    const int64_t ctas = b->T < (int64_t)b->sm_count ? b->T : (int64_t)b->sm_count;
    const bool tail_by_fft = tail_from_transform(b->L, n_blocks, n_tail);
    const int32_t n_ftail = tail_by_fft ? n_tail : 0, n_dtail = tail_by_fft ? 0 : n_tail;
    SegArgs sa{};
    sa.n_seg = n_seg;
    for (int sg = 0; sg < n_seg; ++sg) {
        sa.rn2[sg] = b->rn2 + (int64_t)sg * n_lags;
        sa.lag_begin[sg] = lag_begin;
        sa.rho_max[sg] = rho_max ? rho_max[sg] : nullptr;
        sa.arg_lag[sg] = arg_lag ? arg_lag[sg] : nullptr;
    }
    core_timer_start(b, stream);
#define BFLY_TC_LAUNCH(TAILS_, FAM_, MULTI_, ARGS_)                                                    \
    tc_correlate_kernel<TAILS_, FAM_, MULTI_><<<(unsigned)ctas, NT, TC_SMEM, stream>>>(                \
        b->T, b->L, b->phA, b->phB, b->phC, b->inc2, b->ins2, reinterpret_cast<const uint4 *>(b->xh), \
        reinterpret_cast<const float4 *>(b->rn2p), x[0], b->rn2, lag_begin, (int32_t)n_blocks, n_dtail, \
        n_ftail, b->qs, sa.rho_max[0], sa.arg_lag[0], sa, ARGS_)
    const int fam = b->family == BFLY_FAMILY_SETTLE ? 2 : b->has_f2 ? 1 : 0;
    if (tails) {
        if (fam == 2) BFLY_TC_LAUNCH(true, 2, false, *tails);
        else if (fam == 1) BFLY_TC_LAUNCH(true, 1, false, *tails);
        else BFLY_TC_LAUNCH(true, 0, false, *tails);
    } else if (n_seg > 1) {
        if (fam == 2) BFLY_TC_LAUNCH(false, 2, true, TailArgs{});
        else if (fam == 1) BFLY_TC_LAUNCH(false, 1, true, TailArgs{});
        else BFLY_TC_LAUNCH(false, 0, true, TailArgs{});
    } else {
        if (fam == 2) BFLY_TC_LAUNCH(false, 2, false, TailArgs{});
        else if (fam == 1) BFLY_TC_LAUNCH(false, 1, false, TailArgs{});
        else BFLY_TC_LAUNCH(false, 0, false, TailArgs{});
    }
#undef BFLY_TC_LAUNCH
    core_timer_stop(b, stream);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

int launch_fft_tc(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                  int64_t lag_end, float *rho_max, int32_t *arg_lag, cudaStream_t stream)
{
    return launch_tc_common(b, 1, &x, n_samples, lag_begin, lag_end, &rho_max, &arg_lag, nullptr, stream);
}

int launch_fft_tc_multi(const bfly_bank *b, int n_seg, const float *const *x, int64_t n_samples, int64_t lag_begin,
                        int64_t lag_end, float *const *rho_max, int32_t *const *arg_lag, cudaStream_t stream)
{
    return launch_tc_common(b, n_seg, x, n_samples, lag_begin, lag_end, rho_max, arg_lag, nullptr, stream);
}

// bfly_tails: predictor step (autocorrelation of the segment, its transform W), then the
// correlate kernel in TAILS mode.  racf / wspec are workspace of the bank (sized by the caller).
int launch_tails_tc(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin,
                    int64_t lag_end, float kappa, float *sigma, int64_t capacity,
                    int32_t *hit_template, int32_t *hit_lag, float *hit_rho,
                    unsigned long long *n_hits, cudaStream_t stream)
{
    tc_autocorr_kernel<<<(unsigned)b->L, 256, 0, stream>>>(x, n_samples, b->racf);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    const int rc = tc_attrs(b->device);
    if (rc) return rc;
    tc_wspec_kernel<<<1, fft32::NT, fft32::FFT_SMEM, stream>>>(b->racf, b->L, b->wspec);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    TailArgs ta;
    ta.wspec = reinterpret_cast<const float4 *>(b->wspec);
    ta.sig_norm = 1.0 / (2.0 * (double)n_samples * (double)FFT_B);
    ta.kappa = kappa;
    ta.sigma = sigma;
    ta.capacity = (long long)capacity;
    ta.hit_template = hit_template;
    ta.hit_lag = hit_lag;
    ta.hit_rho = hit_rho;
    ta.n_hits = n_hits;
    return launch_tc_common(b, 1, &x, n_samples, lag_begin, lag_end, nullptr, nullptr, &ta, stream);
}

// ------------------------------------------------------------------------------------------
// bfly_correlate_static: the default form with its per-call scratch (data-block spectra, per-lag
// normalisers, block scales) in a file-scope device array instead of the bank's cudaMalloc'ed
// workspace, for callers that must not allocate (CUDA graph capture, serving loops).  The array is
// sized for one segment of BFLY_STATIC_MAX_SAMPLES samples (16 overlap-save blocks); every GPU
// that loads the library holds it until exit.  All calls share it: calls that overlap on the GPU
// race.  Nothing in it has to start at zero -- every region the kernels read is written first by
// the same call (spectra and scales by tc_spectra_kernel, normalisers by tc_norm_kernel and
// sliding_norm_kernel) -- so the previous call's contents are simply overwritten.
constexpr int64_t STATIC_MAX_BLOCKS = BFLY_STATIC_MAX_SAMPLES / TCV;                       // 16
constexpr size_t ST_OFF_XH = 0;                                                             // 16 x 32 KB, fp16
constexpr size_t ST_OFF_RN2P = ST_OFF_XH + (size_t)STATIC_MAX_BLOCKS * 2 * EXCH_WORDS * 2;  // 16 x 16 KB, fp32
constexpr size_t ST_OFF_RN2 = ST_OFF_RN2P + (size_t)STATIC_MAX_BLOCKS * TCV * 4;            // 64 Ki lags, fp32
constexpr size_t ST_OFF_QS = ST_OFF_RN2 + (size_t)BFLY_STATIC_MAX_SAMPLES * 4;              // 16 doubles
constexpr size_t ST_BYTES = ST_OFF_QS + 256;
static __device__ __align__(256) unsigned char tc_static_scratch[ST_BYTES];                // 1 MB + 256 B

// In host code `tc_static_scratch` is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
static int tc_static_base(int device, unsigned char **base)
{
    static PerDeviceOnce once;
    static unsigned char *ptr[MAX_DEVICES] = {};
    const int rc = once.run(device, [device]() -> int {
        void *p = nullptr;
        BFLY_CUDA(cudaGetSymbolAddress(&p, tc_static_scratch));
        ptr[device] = static_cast<unsigned char *>(p);
        return BFLY_OK;
    });
    if (rc) return rc;
    *base = ptr[device];
    return BFLY_OK;
}

int launch_fft_tc_static(const bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin, int64_t lag_end,
                         float *rho_max, int32_t *arg_lag, cudaStream_t stream)
{
    const int64_t n_lags = lag_end - lag_begin;
    int64_t n_blocks; int32_t n_tail;
    tc_plan(n_lags, &n_blocks, &n_tail);
    if (n_samples > BFLY_STATIC_MAX_SAMPLES || n_lags > BFLY_STATIC_MAX_SAMPLES || n_blocks > STATIC_MAX_BLOCKS) {
        set_error("bfly_correlate_static: n_samples = %lld exceeds BFLY_STATIC_MAX_SAMPLES = %d (the static scratch "
                  "array holds one segment of that size; use bfly_correlate)", (long long)n_samples,
                  (int)BFLY_STATIC_MAX_SAMPLES);
        return BFLY_ERANGE;
    }
    unsigned char *base = nullptr;
    int rc = tc_static_base(b->device, &base);
    if (rc) return rc;
    // a host-side view of the bank whose workspace is the static array (the bank itself is not touched)
    bfly_bank view = *b;
    view.xh = reinterpret_cast<__half *>(base + ST_OFF_XH);
    view.xh_cap = STATIC_MAX_BLOCKS * 2 * EXCH_WORDS;
    view.rn2p = reinterpret_cast<float *>(base + ST_OFF_RN2P);
    view.rn2p_cap = STATIC_MAX_BLOCKS * TCV;
    view.rn2 = reinterpret_cast<float *>(base + ST_OFF_RN2);
    view.rn2_cap = BFLY_STATIC_MAX_SAMPLES;
    view.qs = reinterpret_cast<double *>(base + ST_OFF_QS);
    view.qs_cap = STATIC_MAX_BLOCKS;
    view.timing = 0;
    if ((rc = launch_sliding_norm(x, n_samples, view.L, lag_begin, n_lags, view.rn2, stream))) return rc;
    return launch_tc_common(&view, 1, &x, n_samples, lag_begin, lag_end, &rho_max, &arg_lag, nullptr, stream);
}

int launch_debug_fft_tc(const float2 *y, float2 *z, int full, cudaStream_t stream)
{
    int dev = 0;
    BFLY_CUDA(cudaGetDevice(&dev));
    const int rc = tc_attrs(dev);
    if (rc) return rc;
    tc_debug_fft_kernel<<<1, NT, TC_SMEM, stream>>>(y, z, full);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

}  // namespace bfly
