// BFLY_FORM_DENSE_TC: the correlation core as a dense contraction on the 5th-generation tensor
// cores (north_star (3)(a); rows A3-A7 of DESIGN.md).
//
//     c_j(tau) = sum_k h_c,j[k] x[tau + k]       D_c[j, tau] = A_c[j, k] . B[k, tau]
//     s_j(tau) = sum_k h_s,j[k] x[tau + k]       D_s[j, tau] = A_s[j, k] . B[k, tau]
//
// with A = a tile of 128 templates synthesised on the fly from (f0, f1) into shared memory (fp16,
// un-normalised, K-major, 128-byte swizzle: the bank never streams from HBM) and B = the Hankel
// matrix of the data, B[k, tau] = x[tau + k], delivered by TMA.  A Hankel tile has rows one sample
// apart, which a tensor map cannot express (strides are multiples of 16 bytes), so dense_prep_kernel
// writes eight copies of the fp16 series shifted by 0..7 samples and the 3-D tensor map
// {k: 64 contiguous, r: stride 16 bytes, s: stride one copy} delivers the 256-lag x 64-k tile with
// row s * 32 + r holding lag 8 r + s (rows overlap in memory; the epilogue undoes the permutation).
// tcgen05.mma (cta_group::1, kind::f16, M = 128, N = 256, K = 16) accumulates both quadratures in
// fp32 in tensor memory: D_c in columns 0..255, D_s in columns 256..511 (all of TMEM, one CTA per
// SM).  Roles: warps 0-7 synthesise A (two threads per template row, 32 samples of each K-block
// each) and run the epilogue (one TMEM lane = one template, the two threads of a row take half of
// the columns each: A5-A7 with one two-way merge per template), warp 8 allocates TMEM and issues
// the MMAs; a 3-stage full/empty mbarrier ring joins them.  A CTA owns a tile of
// 128 templates across ALL lag tiles, so the running maximum stays in registers and the only HBM
// traffic is 32 B in and 8 B out per template.
//
// Accuracy: operands fp16 (11-bit significand: SURVEY 7.3 item 1 measured max |d rho| 2.9e-5 for
// this rounding), accumulation fp32.  The series is scaled by a power of two that puts max |x|
// in [64, 128) (rho is scale invariant; the factor is folded into the per-lag normaliser).
#include <cuda.h>

#include <algorithm>
#include <type_traits>

#include "bfly_internal.cuh"

namespace bfly {

namespace {

constexpr int DT_M = 128;          // templates per tile (TMEM lanes)
constexpr int DT_N = 256;          // lags per tile (TMEM columns per quadrature)
constexpr int DT_K = 64;           // samples per K-block (one 128-byte swizzle row of fp16)
constexpr int DT_STAGES = 3;
constexpr int DT_PRODUCER_WARPS = 8;
constexpr int DT_THREADS = (DT_PRODUCER_WARPS + 1) * 32;   // warps 0-7: producers + epilogue, warp 8: TMEM + MMA issue
constexpr uint32_t DT_A_BYTES = DT_M * DT_K * 2;              // 16 KB per quadrature
constexpr uint32_t DT_B_BYTES = DT_N * DT_K * 2;              // 32 KB
constexpr uint32_t DT_STAGE_BYTES = 2 * DT_A_BYTES + DT_B_BYTES;
constexpr size_t DT_SMEM = (size_t)DT_STAGES * DT_STAGE_BYTES + 1024 /* alignment slack */ + 128 /* barriers */ +
                           DT_M * 8 /* merge */;

// ------------------------------------------------------------------------------------------
// PTX wrappers (PTX ISA: mbarrier, cp.async.bulk.tensor, tcgen05)
__device__ __forceinline__ uint32_t saddr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "DT_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DT_DONE;\n"
        "bra DT_WAIT;\n"
        "DT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *map, int c0, int c1, int c2,
                                            uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] . B[smem]; one thread issues for the CTA
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                         uint32_t accumulate)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
// arrive on an mbarrier when all MMAs issued so far by this thread have completed
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// Shared-memory matrix descriptor of a K-major tile with 128-byte rows and 128-byte swizzle:
// start address >> 4 in bits 0-13, stride between 8-row groups (1024 B) >> 4 in bits 32-45,
// descriptor version 1 in bits 46-47, layout type 2 (SWIZZLE_128B) in bits 61-63.  Stepping
// along K by 16 fp16 inside the swizzle row adds 32 bytes to the start address.
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr)
{
    return (uint64_t)((addr & 0x3FFFFu) >> 4) | ((uint64_t)(1024u >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor, kind::f16: D fp32 (bits 4-5 = 1), A and B fp16 (0), both K-major (0),
// N >> 3 in bits 17-22, M >> 4 in bits 24-28.
constexpr uint32_t DT_IDESC = (1u << 4) | ((uint32_t)(DT_N >> 3) << 17) | ((uint32_t)(DT_M >> 4) << 24);

// ------------------------------------------------------------------------------------------
// Preparation (once per call): max |x| over the samples the call touches -> power-of-two scale;
// eight shifted fp16 copies of the scaled series; per-lag normaliser 1 / (n2 scale^2), 0 past the
// last lag.
__global__ void dense_absmax_kernel(const float *__restrict__ x, int64_t first, int64_t count,
                                    unsigned int *__restrict__ maxbits)
{
    float m = 0.0f;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count;
         i += (int64_t)gridDim.x * blockDim.x) {
        const float v = fabsf(__ldg(x + first + i));
        if (isfinite(v)) m = fmaxf(m, v);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0.0f) atomicMax(maxbits, __float_as_uint(m));   // m >= 0
}

__device__ __forceinline__ float dense_scale(unsigned int maxbits)
{
    const float m = __uint_as_float(maxbits);
    if (!(m > 0.0f)) return 1.0f;
    int ex;
    frexpf(m, &ex);                       // m = f 2^ex, f in [0.5, 1)
    return ldexpf(1.0f, 7 - ex);          // max |x| scale in [64, 128)
}

// ys[s][m] = fp16(x[first + m + s] scale), 0 past the series; rn2s[i] = rn2[i] / scale^2
__global__ void dense_prep_kernel(const float *__restrict__ x, int64_t n_samples, int64_t first,
                                  int64_t copy_len, const unsigned int *__restrict__ maxbits,
                                  __half *__restrict__ ys, const float *__restrict__ rn2,
                                  int64_t n_lags, int64_t n_lags_padded, float *__restrict__ rn2s)
{
    const float sc = dense_scale(*maxbits);
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < copy_len) {
#pragma unroll
        for (int s = 0; s < 8; ++s) {
            const int64_t gi = first + idx + s;
            ys[(int64_t)s * copy_len + idx] = __float2half_rn(gi < n_samples ? __ldg(x + gi) * sc : 0.0f);
        }
    }
    if (idx < n_lags_padded) {
        const float inv = 1.0f / sc;      // a power of two: the products below are exact
        // stored in the order the epilogue reads it: lag 8 r + s of a 256-lag tile at s * 32 + r
        const int64_t e = (idx & ~(int64_t)255) + (idx & 7) * 32 + ((idx & 255) >> 3);
        rn2s[e] = idx < n_lags ? __ldg(rn2 + idx) * inv * inv : 0.0f;
    }
}

// ------------------------------------------------------------------------------------------
// The contraction.  Grid: persistent, one CTA per SM, strided over tiles of 128 templates.
__global__ void __launch_bounds__(DT_THREADS, 1)
dense_tc_kernel(const __grid_constant__ CUtensorMap xmap, int64_t T, int32_t L, int family, int linear,
                const uint64_t *__restrict__ phA, const uint64_t *__restrict__ phB,
                const uint64_t *__restrict__ phC, const float *__restrict__ inc2, const float *__restrict__ ins2,
                const float *__restrict__ rn2s, int64_t n_lags, int32_t n_lag_tiles,
                int64_t lag_begin, float *__restrict__ rho_max, int32_t *__restrict__ arg_lag)
{
    extern __shared__ unsigned char dt_raw[];
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t sbase = (saddr(dt_raw) + 1023u) & ~1023u;           // swizzle-128B tiles: 1024-B aligned
    const uint32_t bars = sbase + DT_STAGES * DT_STAGE_BYTES;          // full[3] empty[3] tmem_full tmem_empty
    const uint32_t tmem_slot = bars + 64;
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (DT_STAGES + s); };
    const uint32_t tmem_full = bars + 8u * (2 * DT_STAGES), tmem_empty = tmem_full + 8u;

    if (tid == 0) {
        for (int s = 0; s < DT_STAGES; ++s) {
            bar_init(full(s), DT_PRODUCER_WARPS * 32 + 1);   // producer arrivals + the expect_tx arrival
            bar_init(empty(s), 1);             // one tcgen05.commit
        }
        bar_init(tmem_full, 1);
        bar_init(tmem_empty, DT_PRODUCER_WARPS * 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == DT_PRODUCER_WARPS) {           // all of tensor memory: 512 columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(tmem_slot) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot) : "memory");

    const int32_t n_kb = (L + DT_K - 1) / DT_K;
    const int64_t n_ttiles = (T + DT_M - 1) / DT_M;

    if (warp < DT_PRODUCER_WARPS) {
        // ===== producers (A3) and epilogue (A5-A7).  Two threads per template row: thread
        //       (row, half) synthesises samples [32 half, 32 half + 32) of every K-block and, in
        //       the epilogue, reads TMEM lane `row`, columns [128 half, 128 half + 128) of each
        //       quadrature (warp w may touch lanes 32 (w mod 4) .. + 31 only) =====
        int stage = 0;
        uint32_t phase = 0, tiles_done = 0;
        const int row = tid & (DT_M - 1), half = tid >> 7;
        const uint32_t row_off = (uint32_t)row * 128u, row_x = (uint32_t)row & 7u;
        uint32_t m32 = 0xFFFFFFE0u;                // in a register: (q & m32) | rank is then one LOP3
        asm volatile("" : "+r"(m32));
        unsigned long long *merge = reinterpret_cast<unsigned long long *>(dt_raw + (sbase - saddr(dt_raw)) +
                                                                          DT_STAGES * DT_STAGE_BYTES + 128);
        for (int64_t tt = blockIdx.x; tt < n_ttiles; tt += gridDim.x) {
            const int64_t j = tt * DT_M + row;
            const bool valid = j < T;
            const uint64_t A = valid ? phA[j] : 0ull, Bq = valid ? phB[j] : 0ull, Cq = valid ? phC[j] : 0ull;
            const float ic = valid ? inc2[j] : 0.0f, is = valid ? ins2[j] : 0.0f;
            // linear chirps: w = exp(2 pi i dd), dd = 2 B the (constant) second phase difference, a tiny
            // angle (|f1| / fs^2 cycles): two terms of the series are exact in fp32
            const float wx = (float)(long long)(2ull * Bq) * 3.4061215800865545e-19f;   // 2 pi 2^-64
            const float wr = fmaf(-0.5f * wx, wx, 1.0f), wi = fmaf(wx * wx * (-1.0f / 6.0f), wx, wx);
            float bkey = -1.0f, bcmp = -1.0f;      // running key of this thread's columns, and the same with its rank bits set
            int32_t bchunk = 0;                    // 8 lt + s of the chunk that holds it
            for (int32_t lt = 0; lt < n_lag_tiles; ++lt) {
                for (int32_t kb = 0; kb < n_kb; ++kb) {
                    bar_wait(empty(stage), phase ^ 1u);
                    const uint32_t st = sbase + (uint32_t)stage * DT_STAGE_BYTES;
                    if (tid == 0) {
                        bar_expect_tx(full(stage), DT_B_BYTES);
                        tma_load_3d(st + 2 * DT_A_BYTES, &xmap, 0, (lt * DT_N + kb * DT_K) / 8, 0, full(stage));
                    }
                    // phase of this thread's first sample and its first three differences, exact to
                    // 2^-32 cycle, then a third-order recurrence in 32-bit fixed point (wrap = mod 1
                    // cycle; the third difference is the constant 6 C of a cubic phase, 0 for a
                    // linear chirp; for the settling family (reading N2) it is taken from four exact
                    // phases and held over the 32 samples: fourth-difference error < 1e-8 cycle).  Half a cycle is added so that the bit pattern 0x3F800000 | (ph >> 9),
                    // a float in [1, 2), minus 1.5 is the phase in [-1/2, 1/2) cycles: no
                    // int-to-float conversion (those share the XU pipe with sin / cos).
                    const uint64_t k0 = (uint64_t)kb * DT_K + 32u * (uint32_t)half;
                    const bool whole = valid && (int32_t)k0 + 32 <= L;
                    if (linear) {
                        // Linear chirps (the default family): u_k = exp(2 pi i phi_k) by the rotation
                        // recurrence u_{k+1} = u_k v_k, v_{k+1} = v_k w with v_k = exp(2 pi i (phi_{k+1} -
                        // phi_k)): 8 fp32 FMAs per sample on the FMA pipe instead of two SFU calls (the XU
                        // pipe, 16 lanes per SM, was the co-limiter of this kernel: 16384 sin/cos per
                        // K-block = 1024 cycles, the same as the K-block's MMAs).  u and v are re-seeded
                        // from the exact fixed-point phase at the thread's first sample of every K-block
                        // (4 SFU calls per 32 samples); the phase error inside a run of 32 is below 2e-5 rad.
                        const uint64_t p0 = template_phase(A, Bq, 0ull, k0), p1 = template_phase(A, Bq, 0ull, k0 + 1);
                        const float fu = __uint_as_float(__funnelshift_r((uint32_t)(p0 >> 32) ^ 0x80000000u, 0x7Fu, 9));
                        const float fv = __uint_as_float(__funnelshift_r((uint32_t)((p1 - p0) >> 32) ^ 0x80000000u, 0x7Fu, 9));
                        const float au = fmaf(fu, 6.283185307179586f, -9.42477796076938f);
                        const float av = fmaf(fv, 6.283185307179586f, -9.42477796076938f);
                        float ur = __cosf(au), ui = __sinf(au), vr = __cosf(av), vi = __sinf(av);
                        // the samples past L are masked only in the (rare) warps that own any: a
                        // warp-uniform branch, so the common path carries no selects
                        auto synth32 = [&](auto masked) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            uint32_t cw[4], sw[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                float cs[2], sn[2];
#pragma unroll
                                for (int e = 0; e < 2; ++e) {
                                    cs[e] = ur;
                                    sn[e] = ui;
                                    if (decltype(masked)::value) {
                                        const bool on = valid && (int32_t)k0 + 8 * c + 2 * i + e < L;
                                        cs[e] = on ? cs[e] : 0.0f;
                                        sn[e] = on ? sn[e] : 0.0f;
                                    }
                                    const float nr = fmaf(ur, vr, -(ui * vi)), ni = fmaf(ur, vi, ui * vr);
                                    const float mr = fmaf(vr, wr, -(vi * wi)), mi = fmaf(vr, wi, vi * wr);
                                    ur = nr; ui = ni; vr = mr; vi = mi;
                                }
                                __half2 hc = __floats2half2_rn(cs[0], cs[1]), hs = __floats2half2_rn(sn[0], sn[1]);
                                cw[i] = *reinterpret_cast<uint32_t *>(&hc);
                                sw[i] = *reinterpret_cast<uint32_t *>(&hs);
                            }
                            const uint32_t off = row_off + (((uint32_t)(4 * half + c) ^ row_x) << 4);
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + off), "r"(cw[0]), "r"(cw[1]),
                                         "r"(cw[2]), "r"(cw[3]) : "memory");
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + DT_A_BYTES + off), "r"(sw[0]),
                                         "r"(sw[1]), "r"(sw[2]), "r"(sw[3]) : "memory");
                        }
                        };
                        if (__all_sync(0xffffffffu, whole)) synth32(std::false_type{});
                        else synth32(std::true_type{});
                    } else {
                        const uint64_t p0 = family_phase(family, A, Bq, Cq, k0), p1 = family_phase(family, A, Bq, Cq, k0 + 1),
                                       p2 = family_phase(family, A, Bq, Cq, k0 + 2);
                        const uint32_t d3 = family == BFLY_FAMILY_SETTLE
                            ? (uint32_t)((family_phase(family, A, Bq, Cq, k0 + 3) - 3ull * p2 + 3ull * p1 - p0) >> 32)
                            : (uint32_t)((6ull * Cq) >> 32);
                        uint32_t ph = (uint32_t)(p0 >> 32) ^ 0x80000000u;
                        uint32_t d = (uint32_t)((p1 - p0) >> 32);
                        uint32_t dd = (uint32_t)((p2 - 2ull * p1 + p0) >> 32);
    #pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            uint32_t cw[4], sw[4];
    #pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                float cs[2], sn[2];
    #pragma unroll
                                for (int e = 0; e < 2; ++e) {
                                    const float f = __uint_as_float(__funnelshift_r(ph, 0x7Fu, 9));
                                    const float ang = fmaf(f, 6.283185307179586f, -9.42477796076938f);   // 2 pi (f - 1.5)
                                    cs[e] = __cosf(ang);
                                    sn[e] = __sinf(ang);
                                    if (!whole) {
                                        const bool on = valid && (int32_t)k0 + 8 * c + 2 * i + e < L;
                                        cs[e] = on ? cs[e] : 0.0f;
                                        sn[e] = on ? sn[e] : 0.0f;
                                    }
                                    ph += d;
                                    d += dd;
                                    dd += d3;
                                }
                                __half2 hc = __floats2half2_rn(cs[0], cs[1]), hs = __floats2half2_rn(sn[0], sn[1]);
                                cw[i] = *reinterpret_cast<uint32_t *>(&hc);
                                sw[i] = *reinterpret_cast<uint32_t *>(&hs);
                            }
                            const uint32_t off = row_off + (((uint32_t)(4 * half + c) ^ row_x) << 4);
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + off), "r"(cw[0]), "r"(cw[1]),
                                         "r"(cw[2]), "r"(cw[3]) : "memory");
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + DT_A_BYTES + off), "r"(sw[0]),
                                         "r"(sw[1]), "r"(sw[2]), "r"(sw[3]) : "memory");
                        }
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes -> tensor-core reads
                    bar_arrive(full(stage));
                    if (++stage == DT_STAGES) { stage = 0; phase ^= 1u; }
                }
                // ---- epilogue of this lag tile: column s * 32 + r holds lag 8 r + s of the tile.  A7 per
                //      thread by rank-in-mantissa keys: the low five mantissa bits of q (2^-18 relative)
                //      are replaced by 31 - r, so that the maximum key of a 32-column chunk is its largest
                //      q and, on a tie, its smallest lag; chunks are compared by one test each (the tie of
                //      two chunks is resolved on the lags themselves).  Lags past the last one carry a
                //      normaliser of 0 (q = 0: they never beat a positive q).
                bar_wait(tmem_full, tiles_done & 1u);
                tc_fence_after();
                const uint32_t lane_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
#pragma unroll 1
                for (int s = 4 * half; s < 4 * half + 4; ++s) {
                    uint32_t vc[32], vs[32];
                    tmem_ld32(lane_addr + (uint32_t)(s * 32), vc);
                    tmem_ld32(lane_addr + (uint32_t)(DT_N + s * 32), vs);
                    tmem_ld_wait();
                    if (s == 4 * half + 3) {           // the accumulators are in registers: the next tile's MMAs may start
                        tc_fence_before();
                        bar_arrive(tmem_empty);
                    }
                    const float4 *rp = reinterpret_cast<const float4 *>(rn2s + ((int64_t)lt * DT_N + s * 32));
                    float m[4] = {-1.0f, -1.0f, -1.0f, -1.0f};
#pragma unroll
                    for (int r4 = 0; r4 < 8; ++r4) {
                        const float4 rv = __ldg(rp + r4);
                        const float rr[4] = {rv.x, rv.y, rv.z, rv.w};
#pragma unroll
                        for (int kq = 0; kq < 4; ++kq) {
                            const int r = 4 * r4 + kq;
                            const float c = __uint_as_float(vc[r]), sq = __uint_as_float(vs[r]);
                            const float q = fmaf(sq * sq, is, c * c * ic) * rr[kq];
                            uint32_t key;
                            asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(key) : "r"(__float_as_uint(q)), "r"(m32), "r"(31u - r));
                            m[kq] = fmaxf(m[kq], __uint_as_float(key));
                        }
                    }
                    const float bm = fmaxf(fmaxf(m[0], m[1]), fmaxf(m[2], m[3]));
                    const uint32_t bmu = __float_as_uint(bm);
                    const int32_t chunk = lt * 8 + s;
                    if (bm > bcmp) {
                        bkey = bm; bcmp = __uint_as_float(bmu | 31u); bchunk = chunk;
                    } else if ((bmu | 31u) == __float_as_uint(bcmp)) {      // equal q: the smaller lag (rare)
                        const int32_t l_new = (chunk >> 3) * DT_N + 8 * (31 - (int32_t)(bmu & 31u)) + (chunk & 7);
                        const int32_t l_old = (bchunk >> 3) * DT_N + 8 * (31 - (int32_t)(__float_as_uint(bkey) & 31u)) + (bchunk & 7);
                        if (l_new < l_old) { bkey = bm; bchunk = chunk; }
                    }
                }
                ++tiles_done;
            }
            unsigned long long best = 0ull;
            {
                const uint32_t ku = __float_as_uint(bkey), qbits = ku & 0xFFFFFFE0u;
                if (__uint_as_float(qbits) > 0.0f) {
                    const uint32_t li = (uint32_t)((bchunk >> 3) * DT_N + 8 * (31 - (int32_t)(ku & 31u)) + (bchunk & 7));
                    best = ((unsigned long long)qbits << 32) | (unsigned long long)(0xFFFFFFFFu - li);
                }
            }
            // the two column halves of a row meet in shared memory (the tile handshakes keep the
            // next tile's writes behind this tile's reads)
            if (half == 1) merge[row] = best;
            asm volatile("bar.sync 1, %0;" ::"n"(DT_PRODUCER_WARPS * 32) : "memory");
            if (half == 0 && valid) {
                const unsigned long long other = merge[row];
                best = other > best ? other : best;
                if (best == 0ull) {
                    rho_max[j] = 0.0f;
                    arg_lag[j] = (int32_t)lag_begin;
                } else {
                    rho_max[j] = sqrtf(__uint_as_float((uint32_t)(best >> 32)));
                    arg_lag[j] = (int32_t)(lag_begin + (int64_t)(0xFFFFFFFFu - (uint32_t)(best & 0xFFFFFFFFull)));
                }
            }
        }
    } else if (tid == DT_PRODUCER_WARPS * 32) {
        // ===== MMA issuer (A4): one thread =====
        int stage = 0;
        uint32_t phase = 0, tiles_done = 0;
        for (int64_t tt = blockIdx.x; tt < n_ttiles; tt += gridDim.x) {
            for (int32_t lt = 0; lt < n_lag_tiles; ++lt) {
                bar_wait(tmem_empty, (tiles_done & 1u) ^ 1u);      // the epilogue has drained the accumulators
                tc_fence_after();
                for (int32_t kb = 0; kb < n_kb; ++kb) {
                    bar_wait(full(stage), phase);
                    tc_fence_after();
                    const uint32_t st = sbase + (uint32_t)stage * DT_STAGE_BYTES;
                    const uint64_t da_c = smem_desc(st), da_s = smem_desc(st + DT_A_BYTES), db = smem_desc(st + 2 * DT_A_BYTES);
#pragma unroll
                    for (int k = 0; k < DT_K / 16; ++k) {
                        const uint32_t acc = (kb > 0 || k > 0) ? 1u : 0u;
                        umma_f16(tmem_base, da_c + 2u * k, db + 2u * k, DT_IDESC, acc);
                        umma_f16(tmem_base + DT_N, da_s + 2u * k, db + 2u * k, DT_IDESC, acc);
                    }
                    umma_commit(empty(stage));                     // frees the stage when these MMAs are done
                    if (++stage == DT_STAGES) { stage = 0; phase ^= 1u; }
                }
                umma_commit(tmem_full);
                ++tiles_done;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == DT_PRODUCER_WARPS) {
        __syncwarp();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

template <typename P>
static int grow_ws(P **ptr, int64_t *cap, int64_t need)
{
    if (need <= *cap) return BFLY_OK;
    if (*ptr) {
        BFLY_CUDA(cudaFree(*ptr));
        *ptr = nullptr;
        *cap = 0;
    }
    BFLY_CUDA(cudaMalloc((void **)ptr, sizeof(P) * (size_t)need));
    *cap = need;
    return BFLY_OK;
}

int launch_dense_tc(bfly_bank *b, const float *x, int64_t n_samples, int64_t lag_begin, int64_t lag_end,
                    float *rho_max, int32_t *arg_lag, cudaStream_t stream)
{
    static EncodeTiledFn encode = nullptr;
    static PerDeviceOnce once;           // function attributes are per device
    static std::mutex encode_mutex;
    std::unique_lock<std::mutex> encode_lock(encode_mutex);
    if (!encode) {
        cudaDriverEntryPointQueryResult q;
        void *fn = nullptr;
        BFLY_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled is not available"); return BFLY_EUNSUPPORTED; }
        encode = (EncodeTiledFn)fn;
    }
    encode_lock.unlock();
    const int rc_attr = once.run(b->device, []() -> int {
        BFLY_CUDA(cudaFuncSetAttribute(dense_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DT_SMEM));
        return BFLY_OK;
    });
    if (rc_attr) return rc_attr;
    const int64_t n_lags = lag_end - lag_begin;
    const int64_t n_lag_tiles = (n_lags + DT_N - 1) / DT_N;
    const int64_t n_kb = (b->L + DT_K - 1) / DT_K;
    const int64_t copy_len = n_lag_tiles * DT_N + n_kb * DT_K;       // halves per shifted copy (multiple of 64)
    if (n_lag_tiles * DT_N >= (1LL << 31)) { set_error("too many lags"); return BFLY_ERANGE; }
    int rc;
    if ((rc = grow_ws(&b->ys, &b->ys_cap, 8 * copy_len))) return rc;
    if ((rc = grow_ws(&b->rn2s, &b->rn2s_cap, n_lag_tiles * DT_N))) return rc;
    if ((rc = grow_ws(&b->maxbits, &b->maxbits_cap, 1))) return rc;

    BFLY_CUDA(cudaMemsetAsync(b->maxbits, 0, sizeof(unsigned int), stream));
    const int64_t touched = n_lags + b->L - 1;     // with no lag at all the kernel writes rho = 0 at lag_begin
    dense_absmax_kernel<<<(unsigned)std::min<int64_t>((touched + 255) / 256, 1184), 256, 0, stream>>>(
        x, lag_begin, touched, b->maxbits);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    const int64_t prep_n = std::max(copy_len, n_lag_tiles * DT_N);
    dense_prep_kernel<<<(unsigned)((prep_n + 255) / 256), 256, 0, stream>>>(
        x, n_samples, lag_begin, copy_len, b->maxbits, b->ys, b->rn2, n_lags, n_lag_tiles * DT_N, b->rn2s);
    count_launch();
    BFLY_CUDA(cudaGetLastError());

    // Hankel view of the eight shifted copies: element (k, r, s) = ys[s][8 r + k] = x[first + 8 r + s + k]
    CUtensorMap map;
    const cuuint64_t dims[3] = {(cuuint64_t)DT_K, (cuuint64_t)((copy_len - DT_K) / 8 + 1), 8};
    const cuuint64_t strides[2] = {16, (cuuint64_t)copy_len * sizeof(__half)};
    const cuuint32_t box[3] = {(cuuint32_t)DT_K, 32, 8}, estr[3] = {1, 1, 1};
    const CUresult cr = encode(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, b->ys, dims, strides, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d)", (int)cr); return BFLY_ECUDA; }

    const int64_t n_ttiles = (b->T + DT_M - 1) / DT_M;
    const int64_t ctas = std::min<int64_t>(n_ttiles, b->sm_count);
    core_timer_start(b, stream);
    dense_tc_kernel<<<(unsigned)ctas, DT_THREADS, DT_SMEM, stream>>>(
        map, b->T, b->L, b->family, (b->family == BFLY_FAMILY_POLY && !b->has_f2) ? 1 : 0, b->phA, b->phB, b->phC, b->inc2, b->ins2, b->rn2s, n_lags, (int32_t)n_lag_tiles, lag_begin,
        rho_max, arg_lag);
    core_timer_stop(b, stream);
    count_launch();
    BFLY_CUDA(cudaGetLastError());
    return BFLY_OK;
}

}  // namespace bfly
