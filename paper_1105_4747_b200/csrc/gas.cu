// gas.cu -- S1: gas state per cell (Eq.4, Eq.5 with pivot, Doppler parameter).
//
//   D   = 1 + delta                      Dt = min(D, pivot)
//   T   = T0 Dt^(gamma-1)                                              (Eq.5)
//   b   = sqrt(2 kB T / m_p) = b0 Dt^((gamma-1)/2)
//   nHI = nbarHI (T/T0)^-0.7 D^2 = nbarHI Dt^(-1.4 (gamma-1)/2) D^2    (Eq.4 with the local T: reading C4)
//
// HBM-bound: 4 B read + 8 B written per cell.  One lg2 and two ex2 per cell; 128-bit loads/stores,
// grid-stride over a grid that is a multiple of the SM count (256 CTAs per SM: see lya_launch_gas).
#include "gas_cell.h"
#include "lya_internal.h"

namespace {

__device__ __forceinline__ void gas_cell4(const GasK &k, const float4 &d, float4 &n, float4 &w)
{
    gas_cell(k, d.x, n.x, w.x);
    gas_cell(k, d.y, n.y, w.y);
    gas_cell(k, d.z, n.z, w.z);
    gas_cell(k, d.w, n.w, w.w);
}

// two independent 128-bit loads in flight per thread and iteration; streaming (evict-first) loads and stores
__global__ void __launch_bounds__(256) gas_vec4_kernel(const float4 *__restrict__ delta, size_t n4,
                                                       float4 *__restrict__ n_hi, float4 *__restrict__ b,
                                                       GasK k)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < n4; i += 2 * stride) {
        const float4 d0 = __ldcs(delta + i), d1 = __ldcs(delta + i + stride);
        float4 n0, w0, n1, w1;
        gas_cell4(k, d0, n0, w0);
        gas_cell4(k, d1, n1, w1);
        __stcs(n_hi + i, n0);
        __stcs(b + i, w0);
        __stcs(n_hi + i + stride, n1);
        __stcs(b + i + stride, w1);
    }
    if (i < n4) {
        const float4 d0 = __ldcs(delta + i);
        float4 n0, w0;
        gas_cell4(k, d0, n0, w0);
        __stcs(n_hi + i, n0);
        __stcs(b + i, w0);
    }
}

__global__ void __launch_bounds__(256) gas_scalar_kernel(const float *__restrict__ delta, size_t i0, size_t n,
                                                         float *__restrict__ n_hi, float *__restrict__ b, GasK k)
{
    size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = i0 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        gas_cell(k, delta[i], n_hi[i], b[i]);
}

}  // namespace

lya_status lya_launch_gas(lya_ctx *ctx, const float *delta, size_t n, float *n_hi, float *b,
                          float nbar_hi, float b0, float half_gm1, float pivot)
{
    GasK k{nbar_hi, b0, half_gm1, (float)(2.0 * LYA_ALPHA_T) * half_gm1, pivot};
    bool aligned = (((uintptr_t)delta | (uintptr_t)n_hi | (uintptr_t)b) & 15) == 0;
    size_t n4 = aligned ? n / 4 : 0;
    if (n4) {
        size_t want = (n4 + 255) / 256;
        // about 8 float4 per thread, between 8 and 256 CTAs per SM (several waves of short grid-stride loops):
        // measured 92-95 % of the HBM copy bandwidth on 512^3 / 1024^3 against 80-85 % for 8 resident CTAs per SM
        size_t cap = want / 8;
        if (cap < (size_t)ctx->sm_count * 8) cap = (size_t)ctx->sm_count * 8;
        if (cap > (size_t)ctx->sm_count * 256) cap = (size_t)ctx->sm_count * 256;
        int grid = (int)(want < cap ? want : cap);
        gas_vec4_kernel<<<grid, 256, 0, ctx->stream>>>((const float4 *)delta, n4, (float4 *)n_hi, (float4 *)b, k);
        ctx->launches++;
    }
    if (n4 * 4 < n) {
        size_t rem = n - n4 * 4;
        size_t want = (rem + 255) / 256;
        int grid = (int)(want < (size_t)ctx->sm_count * 8 ? want : (size_t)ctx->sm_count * 8);
        gas_scalar_kernel<<<grid, 256, 0, ctx->stream>>>(delta, n4 * 4, n, n_hi, b, k);
        ctx->launches++;
    }
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}
