// probe.cu -- lya_measure_mufu_peak: the tau kernel's roofline denominator, measured on the device in use.
// A pure ex2.approx.ftz.f32 kernel (8 independent dependent-chains per thread, one 1024-thread CTA per SM)
// timed with CUDA events; on B200 it returns 16.0 results / clk / SM (profiles/r1_mufu_probe.md).
#include "lya_internal.h"

namespace {

__global__ void __launch_bounds__(1024) mufu_peak_kernel(float *out, int iters, float seed)
{
    float a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = seed + 0.01f * i + 1e-6f * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            float y;
            asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a[i] - 1.0f));
            a[i] = y;
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" lya_status lya_measure_mufu_peak(lya_ctx *ctx, double *ex2_per_s)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!ex2_per_s) return lya_fail(ctx, LYA_EINVAL, "lya_measure_mufu_peak: null pointer");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    const int iters = 8192, grid = ctx->sm_count, threads = 1024;
    float *buf = nullptr;
    LYA_CUDA(ctx, cudaMalloc((void **)&buf, (size_t)grid * threads * sizeof(float)));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {        // first repetition is the warm-up
        cudaEventRecord(e0, ctx->stream);
        mufu_peak_kernel<<<grid, threads, 0, ctx->stream>>>(buf, iters, 0.3f);
        cudaEventRecord(e1, ctx->stream);
        ctx->launches++;
        e = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)grid * threads * 8.0 * iters / ((double)ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_measure_mufu_peak");
    *ex2_per_s = best;
    return LYA_OK;
}

// lya_measure_hbm_peak: the HBM roofline denominator measured with the access pattern of this library's own
// elementwise kernels -- 128-bit streaming loads and stores, 1 read : 1 write, a grid of many short grid-stride
// loops -- over a buffer far larger than L2.  Reported next to MEASURED_PEAKS.json's torch-copy figure.
namespace {

__global__ void __launch_bounds__(256) copy_peak_kernel(const float4 *__restrict__ src, float4 *__restrict__ dst, size_t n4)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < n4; i += 2 * stride) {
        const float4 a = __ldcs(src + i), b = __ldcs(src + i + stride);
        __stcs(dst + i, a);
        __stcs(dst + i + stride, b);
    }
    if (i < n4) __stcs(dst + i, __ldcs(src + i));
}

}  // namespace

extern "C" lya_status lya_measure_hbm_peak(lya_ctx *ctx, size_t n_bytes, double *gb_per_s)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!gb_per_s || n_bytes < ((size_t)1 << 20)) return lya_fail(ctx, LYA_EINVAL, "lya_measure_hbm_peak: null pointer or fewer than 2^20 bytes");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t n4 = n_bytes / 32;                               // half of n_bytes is read, half written
    float4 *buf = nullptr;
    if (cudaMalloc((void **)&buf, 2 * n4 * sizeof(float4)) != cudaSuccess) {
        cudaGetLastError();
        return lya_fail(ctx, LYA_ENOMEM, "lya_measure_hbm_peak: allocation failed");
    }
    cudaMemsetAsync(buf, 0, 2 * n4 * sizeof(float4), ctx->stream);
    size_t want = (n4 + 255) / 256, cap = want / 12;
    if (cap < (size_t)ctx->sm_count * 8) cap = (size_t)ctx->sm_count * 8;
    const int grid = (int)(want < cap ? want : cap);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {        // first repetition is the warm-up
        cudaEventRecord(e0, ctx->stream);
        copy_peak_kernel<<<grid, 256, 0, ctx->stream>>>(buf, buf + n4, n4);
        cudaEventRecord(e1, ctx->stream);
        ctx->launches++;
        e = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double rate = 2.0 * (double)n4 * sizeof(float4) / ((double)ms * 1e-3) / 1e9;
        if (rep > 0 && rate > best) best = rate;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_measure_hbm_peak");
    *gb_per_s = best;
    return LYA_OK;
}
