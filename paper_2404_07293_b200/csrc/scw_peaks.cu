// Roofline denominators measured on the device the library runs on (scw_measure_peak, include/scwatter.h):
// small hand-written microbenchmarks of the units the hot path is bound by -- FP64 tensor cores (DMMA, the complex128
// contractions), FP32 FMA and MUFU pipes (point path), HBM read / write streams (assembly reads V, synthesis writes E).
// bench.py runs them before the timed step and divides by these numbers; nothing here is on the hot path.
#include <cstdio>

#include "scw_internal.h"
#include "scw_tc_common.cuh"

namespace scw {

// ---- FP64 DMMA: mma.sync.m8n8k4.f64, 8 independent accumulator pairs per warp --------------------------------------
__global__ void __launch_bounds__(256) k_peak_dmma(int iters, double* __restrict__ sink)
{
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;                      // never true: keeps the loop alive
}

// ---- FP32 FMA: 16 independent chains per thread -------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_peak_ffma(int iters, float* __restrict__ sink)
{
    float v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = 1e-3f * (threadIdx.x + i);
    const float a = 0.999f, b = 1e-4f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = fmaf(v[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i];
    if (s == 123.456f) sink[0] = s;
}

// ---- MUFU: ex2.approx chains (the XU pipe of the point path's sin / cos / ex2) ------------------------------------------
__global__ void __launch_bounds__(256) k_peak_mufu(int iters, float* __restrict__ sink)
{
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = -1e-3f * (threadIdx.x + i + 1);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(v[i]));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 123.456f) sink[0] = s;
}

// ---- MUFU mix of the point path: one sin, one cos and one ex2 per term on independent chains (sin / cos also cost their
// range pre-scale FMUL on the FMA pipe, as in the kernel).  Tells whether SIN / COS issue at the EX2 rate.
__global__ void __launch_bounds__(256) k_peak_mufu_mix(int iters, float* __restrict__ sink)
{
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = 1e-3f * (threadIdx.x + i + 1);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            float a, b, c;
            asm volatile("sin.approx.ftz.f32 %0, %1;" : "=f"(a) : "f"(v[i]));
            asm volatile("cos.approx.ftz.f32 %0, %1;" : "=f"(b) : "f"(v[i]));
            asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(c) : "f"(-v[i]));
            v[i] = a * b + c;
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 123.456f) sink[0] = s;
}

// ---- HBM read: every thread streams 16-byte loads, grid-stride, four loads in flight -----------------------------------
__global__ void __launch_bounds__(512) k_peak_read(const uint4* __restrict__ src, size_t n16, unsigned* __restrict__ sink)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned acc = 0;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const uint4 a = __ldcs(src + i), b = __ldcs(src + i + stride), c = __ldcs(src + i + 2 * stride),
                    d = __ldcs(src + i + 3 * stride);
        acc ^= a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
    }
    for (; i < n16; i += stride) {
        const uint4 a = __ldcs(src + i);
        acc ^= a.x ^ a.y ^ a.z ^ a.w;
    }
    if (acc == 0x12345678u) sink[0] = acc;
}

// ---- HBM write, SM-driven: 16-byte st.global, a warp writes 512 contiguous bytes -----------------------------------------
__global__ void __launch_bounds__(512) k_peak_write(uint4* __restrict__ dst, size_t n16)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const uint4 v = make_uint4(threadIdx.x, blockIdx.x, 3u, 4u);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) dst[i] = v;
}

// ---- HBM write through the TMA engine: bulk shared -> global copies of 16 KB (what a staged synthesis epilogue would do)
constexpr int PEAK_TMA_CHUNK = 16384;
__global__ void __launch_bounds__(128) k_peak_write_tma(uint8_t* __restrict__ dst, size_t n_chunks)
{
    extern __shared__ __align__(128) uint8_t smem[];                 // two 16 KB buffers
    for (int i = threadIdx.x; i < 2 * PEAK_TMA_CHUNK / 16; i += blockDim.x)
        reinterpret_cast<uint4*>(smem)[i] = make_uint4(i, blockIdx.x, 3u, 4u);
    tc::fence_proxy_async();
    __syncthreads();
    if (threadIdx.x == 0) {
        int b = 0;
        for (size_t c = blockIdx.x; c < n_chunks; c += gridDim.x, b ^= 1) {
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst + c * PEAK_TMA_CHUNK),
                         "r"(tc::smem_u32(smem + b * PEAK_TMA_CHUNK)), "r"(PEAK_TMA_CHUNK)
                         : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
}

}  // namespace scw

using namespace scw;

extern "C" int32_t scw_measure_peak(scw_ctx* ctx, int32_t which, void* buf, size_t bytes, int32_t reps, double* value)
{
    if (!ctx || !value) return SCW_ERR_NULL;
    ctx->msg[0] = 0;
    *value = 0.0;
    if (which < SCW_PEAK_FP64_DMMA || which > SCW_PEAK_MUFU_MIX || reps < 1) {
        snprintf(ctx->msg, sizeof(ctx->msg), "scw_measure_peak: unknown unit %d or reps < 1", which);
        return SCW_ERR_VALUE;
    }
    const bool mem = which >= SCW_PEAK_HBM_READ && which <= SCW_PEAK_HBM_WRITE_TMA;
    if (!buf || bytes < 256) {
        snprintf(ctx->msg, sizeof(ctx->msg), "scw_measure_peak: a device buffer is required (%s)",
                 mem ? ">= 1 GiB recommended: larger than L2" : "256 bytes");
        return SCW_ERR_NULL;
    }
    const int sms = ctx->sm_count;
    const int iters = 4096;
    const size_t n16 = bytes / 16, n_chunks = bytes / PEAK_TMA_CHUNK;
    if (which == SCW_PEAK_HBM_WRITE_TMA)
        cudaFuncSetAttribute(k_peak_write_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * PEAK_TMA_CHUNK);
    auto launch = [&]() {
        switch (which) {
            case SCW_PEAK_FP64_DMMA: k_peak_dmma<<<sms * 8, 256, 0, ctx->stream>>>(iters, (double*)buf); break;
            case SCW_PEAK_FP32_FMA: k_peak_ffma<<<sms * 8, 256, 0, ctx->stream>>>(iters, (float*)buf); break;
            case SCW_PEAK_MUFU: k_peak_mufu<<<sms * 8, 256, 0, ctx->stream>>>(iters, (float*)buf); break;
            case SCW_PEAK_MUFU_MIX: k_peak_mufu_mix<<<sms * 8, 256, 0, ctx->stream>>>(iters, (float*)buf); break;
            case SCW_PEAK_HBM_READ: k_peak_read<<<sms * 4, 512, 0, ctx->stream>>>((const uint4*)buf, n16, (unsigned*)buf); break;
            case SCW_PEAK_HBM_WRITE: k_peak_write<<<sms * 4, 512, 0, ctx->stream>>>((uint4*)buf, n16); break;
            default: k_peak_write_tma<<<sms * 4, 128, 2 * PEAK_TMA_CHUNK, ctx->stream>>>((uint8_t*)buf, n_chunks); break;
        }
    };
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    launch();                                           // warm-up
    double best_ms = 1e30;
    for (int r = 0; r < reps; ++r) {                    // best of `reps` single launches (burst figure)
        cudaEventRecord(e0, ctx->stream);
        launch();
        cudaEventRecord(e1, ctx->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms > 0.f && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    const cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) {
        ctx->cuda_err = (int32_t)err;
        snprintf(ctx->msg, sizeof(ctx->msg), "scw_measure_peak: %s", cudaGetErrorString(err));
        return SCW_ERR_CUDA;
    }
    const double s = best_ms * 1e-3;
    const double threads = (double)sms * 8 * 256;
    switch (which) {
        case SCW_PEAK_FP64_DMMA: *value = threads / 32 * iters * 8.0 * (2.0 * 8 * 8 * 4) / s / 1e12; break;   // TFLOP/s
        case SCW_PEAK_FP32_FMA: *value = threads * iters * 16.0 * 2.0 / s / 1e12; break;                      // TFLOP/s
        case SCW_PEAK_MUFU: *value = threads * iters * 8.0 / s / 1e9; break;                                  // Gop/s
        case SCW_PEAK_MUFU_MIX: *value = threads * iters * 8.0 * 3.0 / s / 1e9; break;                        // Gop/s (3 per term)
        case SCW_PEAK_HBM_WRITE_TMA: *value = (double)n_chunks * PEAK_TMA_CHUNK / s / 1e9; break;             // GB/s
        default: *value = (double)n16 * 16.0 / s / 1e9; break;                                                // GB/s
    }
    return SCW_OK;
}
