// bfly_debug_peak: microbenchmarks of the units the correlation kernels are bound by, run on the
// box itself so that bench.py's roofline denominators are measured, not derived (SURVEY 8(d):
// "FP32 FMA peak measured by a microbenchmark on the box and measured shared-memory bandwidth").
// Each kernel keeps ONE unit busy with independent work on every SM and is timed with CUDA
// events; nothing here is on the product path.
#include <cuda_fp16.h>

#include <vector>

#include "bfly_internal.cuh"
#include "bfly_tcgen05.cuh"

namespace bfly {

namespace {

using namespace t5;

// ---- FP32 FMA issue rate: 8 independent FFMA chains per thread ---------------------------------
__global__ void __launch_bounds__(1024) peak_ffma_kernel(float *out, int iters)
{
    float a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = (float)(threadIdx.x + j) * 1e-3f;
    const float m = 1.0f - 1e-6f * (float)(blockIdx.x & 1), c = 1e-7f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = fmaf(a[j], m, c);
    }
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j];
    if (s == 123.456f) out[0] = s;               // keeps the chains alive
}

// packed FFMA2 (two fp32 FMAs per instruction, sm_100): the instruction class of the FFT twiddles
__global__ void __launch_bounds__(1024) peak_ffma2_kernel(float *out, int iters)
{
    float2 a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = make_float2((float)(threadIdx.x + j) * 1e-3f, (float)j);
    const float2 m = make_float2(1.0f - 1e-6f * (float)(blockIdx.x & 1), 0.999f), c = make_float2(1e-7f, 1e-6f);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = __ffma2_rn(a[j], m, c);
    }
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j].x + a[j].y;
    if (s == 123.456f) out[0] = s;
}

// ---- shared-memory read bandwidth: conflict-free ld.shared.v4 stream ----------------------------
__global__ void __launch_bounds__(1024) peak_lds_kernel(float *out, int iters)
{
    extern __shared__ uint4 lds_buf[];            // 64 KB
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) lds_buf[i] = make_uint4(i, i + 1, i + 2, i + 3);
    __syncthreads();
    uint4 acc = make_uint4(0, 0, 0, 0);
    uint32_t idx = threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const uint4 v = lds_buf[(idx + 512u * r) & 4095u];    // 8 distinct addresses; a warp reads 512 contiguous bytes
            acc.x ^= v.x; acc.y ^= v.y; acc.z ^= v.z; acc.w ^= v.w;
        }
        idx += 32;
    }
    if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345678u) out[0] = 1.0f;
}

// ---- the legacy tensor path: independent mma.sync.m16n8k16 f16 -> f32 -----------------------------
__global__ void __launch_bounds__(512) peak_hmma_kernel(float *out, int iters)
{
    float d[8][4];
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
        for (int q = 0; q < 4; ++q) d[j][q] = 0.0f;
    const uint32_t a0 = 0x3C003C00u + threadIdx.x, a1 = 0x38003800u, b0 = 0x3C003800u, b1 = 0x34003C00u;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j)
            asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%4,%5}, {%6,%7}, {%0,%1,%2,%3};"
                         : "+f"(d[j][0]), "+f"(d[j][1]), "+f"(d[j][2]), "+f"(d[j][3])
                         : "r"(a0), "r"(a1), "r"(b0), "r"(b1));
    }
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += d[j][0] + d[j][1] + d[j][2] + d[j][3];
    if (s == 123.456f) out[0] = s;
}

// ---- warp shuffles ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) peak_shfl_kernel(float *out, int iters)
{
    float a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = (float)(threadIdx.x * 8 + j);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = __shfl_xor_sync(0xffffffffu, a[j], 16);
    }
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j];
    if (s == -1.0f) out[0] = s;
}

// ---- L2 read bandwidth on a small hot set (every CTA streams the same 480 KB, as the FFT kernels
//      stream the data-block spectra) ----------------------------------------------------------------
__global__ void __launch_bounds__(512) peak_l2_kernel(const uint4 *__restrict__ src, float *out, int iters)
{
    uint4 acc = make_uint4(0, 0, 0, 0);
    const int n = 480 * 1024 / 16;
    int at = (blockIdx.x * 2048 + threadIdx.x) % n;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            uint4 v;
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                         : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(src + at));
            acc.x ^= v.x; acc.y ^= v.y; acc.z ^= v.z; acc.w ^= v.w;
            at += 512;
            if (at >= n) at -= n;
        }
    }
    if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345678u) out[0] = 1.0f;
}

// ---- tcgen05: MMA issue rate (A from shared or tensor memory), TMEM load rate, and both beside a
//      shared-memory store/load stream ---------------------------------------------------------------
// variant bits: 0-1: 0 = no MMA, 1 = A and B from shared memory (SS), 2 = A from tensor memory (TS)
//               2  : N = 256 instead of 128
//               3  : warps 0-15 stream st.shared.v4 + ld.shared.v4 over 64 KB
//               4  : warps 0-15 stream tcgen05.ld.32x32b.x32
//               5  : consecutive MMAs accumulate into two different tiles in turn (N <= 128)
//               6  : N = 64
// results[0] = clock cycles of the MMA thread, results[1] = cycles of the slowest streaming warp
constexpr int PK_THREADS = 17 * 32;
constexpr size_t PK_SMEM = 1024 + 32768 + 32768 + 65536 + 256;
__global__ void __launch_bounds__(PK_THREADS, 1) peak_umma_kernel(long long *cycles, float *out, int iters, int variant)
{
    extern __shared__ unsigned char pk_raw[];
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t base = (saddr(pk_raw) + 1023u) & ~1023u;
    const uint32_t a_tile = base, b_tile = base + 32768, stream = base + 65536, bars = stream + 65536, slot = bars + 64;
    const int mma_mode = variant & 3;
    const bool wide = variant & 4, do_smem = variant & 8, do_ldtm = variant & 16;
    // operands: small fp16 numbers (|v| < 1) so that nothing overflows; 64 KB covers A and B tiles
    for (int i = tid; i < 65536 / 4; i += PK_THREADS)
        reinterpret_cast<uint32_t *>(pk_raw + (base - saddr(pk_raw)))[i] = 0x2C002E00u + (uint32_t)(i & 0xff);
    if (tid == 0) {
        bar_init(bars, 1);
        bar_init_fence();
    }
    if (warp == 16) tmem_alloc(slot, 512);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(slot) : "memory");
    if (warp < 4) {                               // A operand in tensor memory: columns 384..447
        uint32_t r[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) r[j] = 0x2C002E00u + (uint32_t)j;
        for (int c = 0; c < 4; ++c) tmem_st16(tmem + ((uint32_t)(warp * 32) << 16) + 384u + 16u * c, r);
        tmem_st_wait();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    long long t0 = clock64();
    if (tid == 16 * 32) {
        if (mma_mode) {
            const int n_cols = (variant & 64) ? 64 : wide ? 256 : 128;
            const bool interleave = variant & 32;     // consecutive MMAs accumulate into different tiles
            const uint32_t idesc = idesc_f16(128, n_cols);
            const uint64_t da = smem_desc_k128(a_tile), db = smem_desc_k128(b_tile);
            for (int i = 0; i < iters; ++i) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    // four K-steps inside each of two 64-wide swizzle atoms of both tiles
                    const uint32_t ko = (uint32_t)(k & 3) * 2u + (uint32_t)(k >> 2) * (16384u >> 4);
                    // interleaved: two accumulator tiles take the K-steps in turn (kk = the K-step of the tile)
                    const uint32_t d = tmem + (interleave ? (uint32_t)(k & 1) : (uint32_t)(i & 1)) * 128u;
                    const uint32_t acc = interleave ? (uint32_t)(k > 1 || (i & 3) != 0) : (uint32_t)(k > 0);
                    if (mma_mode == 1) umma_ss(d, da + ko, db + ko, idesc, acc);
                    else umma_ts(d, tmem + 384u + 8u * k, db + ko, idesc, acc);
                }
            }
            umma_commit(bars);
            bar_wait(bars, 0);
            tc_fence_after();
        }
        cycles[blockIdx.x * 2] = clock64() - t0;
    } else if (warp < 16) {
        uint4 acc = make_uint4(tid, 1, 2, 3);
        if (do_smem) {
            uint32_t at = (uint32_t)tid * 16u;
            for (int i = 0; i < iters; ++i) {
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const uint32_t off = (at + 8192u * r) & 65535u;
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(stream + off), "r"(acc.x), "r"(acc.y), "r"(acc.z), "r"(acc.w) : "memory");
                    uint4 v;
                    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(stream + (off ^ 32768u)) : "memory");
                    acc.x += v.x; acc.y ^= v.y; acc.z += v.z; acc.w ^= v.w;
                }
                at += 512u;
            }
        }
        if (do_ldtm) {
            const uint32_t lane_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + 256u + 32u * (uint32_t)((warp >> 2) & 3);
            for (int i = 0; i < iters; ++i) {
                uint32_t r[32];
                tmem_ld32(lane_addr, r);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 32; ++j) acc.x ^= r[j];
            }
        }
        const long long dt = clock64() - t0;
        if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345678u) out[0] = 1.0f;
        if ((tid & 31) == 0) atomicMax(reinterpret_cast<unsigned long long *>(cycles + blockIdx.x * 2 + 1), (unsigned long long)dt);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 16) tmem_dealloc(tmem, 512);
}

}  // namespace

}  // namespace bfly

using namespace bfly;

extern "C" int bfly_debug_peak(int which, int variant, int iters, double *value_out, double *ms_out)
{
    if (!value_out || iters < 1) { set_error("bad arguments"); return BFLY_EINVAL; }
    int dev = 0;
    BFLY_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    BFLY_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) { set_error("device %d is sm_%d%d; sm_100a only", dev, prop.major, prop.minor); return BFLY_EUNSUPPORTED; }
    const int sms = prop.multiProcessorCount;
    float *out = nullptr;
    long long *cyc = nullptr;
    uint4 *src = nullptr;
    BFLY_CUDA(cudaMalloc((void **)&out, 256));
    BFLY_CUDA(cudaMalloc((void **)&cyc, sizeof(long long) * 2 * sms));
    BFLY_CUDA(cudaMemset(cyc, 0, sizeof(long long) * 2 * sms));
    cudaEvent_t e0, e1;
    BFLY_CUDA(cudaEventCreate(&e0));
    BFLY_CUDA(cudaEventCreate(&e1));
    double work = 0.0;                  // flop, bytes or shuffles per launch
    int rc = BFLY_OK;
    for (int rep = 0; rep < 3 && rc == BFLY_OK; ++rep) {      // two warm-ups, the third is timed
        cudaEventRecord(e0, 0);
        switch (which) {
            case BFLY_PEAK_FFMA:
                peak_ffma_kernel<<<2 * sms, 1024>>>(out, iters);
                work = 2.0 * sms * 1024.0 * iters * 64.0 * 2.0;
                break;
            case BFLY_PEAK_FFMA2:
                peak_ffma2_kernel<<<2 * sms, 1024>>>(out, iters);
                work = 2.0 * sms * 1024.0 * iters * 64.0 * 4.0;
                break;
            case BFLY_PEAK_LDS:
                cudaFuncSetAttribute(peak_lds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
                peak_lds_kernel<<<sms, 1024, 65536>>>(out, iters);
                work = (double)sms * 1024.0 * iters * 8.0 * 16.0;
                break;
            case BFLY_PEAK_HMMA:
                peak_hmma_kernel<<<sms, 512>>>(out, iters);
                work = (double)sms * 16.0 * iters * 8.0 * 4096.0;
                break;
            case BFLY_PEAK_SHFL:
                peak_shfl_kernel<<<sms, 512>>>(out, iters);
                work = (double)sms * 16.0 * iters * 8.0;
                break;
            case BFLY_PEAK_L2:
                if (!src) {
                    if (cudaMalloc((void **)&src, 480 * 1024) != cudaSuccess) { rc = BFLY_ENOMEM; break; }
                    cudaMemset(src, 1, 480 * 1024);
                }
                peak_l2_kernel<<<2 * sms, 512>>>(src, out, iters);
                work = 2.0 * sms * 512.0 * iters * 4.0 * 16.0;
                break;
            case BFLY_PEAK_UMMA:
                cudaFuncSetAttribute(peak_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PK_SMEM);
                peak_umma_kernel<<<sms, PK_THREADS, PK_SMEM>>>(cyc, out, iters, variant);
                work = (double)sms * iters * 8.0 * 2.0 * 128.0 * ((variant & 64) ? 64.0 : (variant & 4) ? 256.0 : 128.0) * 16.0;
                break;
            default:
                set_error("unknown microbenchmark %d", which);
                rc = BFLY_EINVAL;
        }
        cudaEventRecord(e1, 0);
        count_launch();
    }
    float ms = 0.0f;
    if (rc == BFLY_OK) {
        cudaError_t e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) rc = cuda_fail(e, "microbenchmark");
    }
    if (rc == BFLY_OK) {
        if (which == BFLY_PEAK_UMMA) {
            // value_out[0]: MMA flop per clock and SM; value_out[1]: cycles of the streaming warps per iteration
            std::vector<long long> h(2 * (size_t)sms);
            cudaMemcpy(h.data(), cyc, sizeof(long long) * h.size(), cudaMemcpyDeviceToHost);
            long long cm = 0, cs = 0;
            for (int i = 0; i < sms; ++i) { cm = h[2 * i] > cm ? h[2 * i] : cm; cs = h[2 * i + 1] > cs ? h[2 * i + 1] : cs; }
            value_out[0] = (variant & 3) ? work / sms / (double)cm : 0.0;
            value_out[1] = (double)cs / iters;
        } else {
            value_out[0] = work / (ms * 1e-3);
        }
        if (ms_out) *ms_out = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    cudaFree(cyc);
    if (src) cudaFree(src);
    return rc;
}
