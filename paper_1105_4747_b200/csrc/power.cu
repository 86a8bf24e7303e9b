// power.cu -- 1D flux power spectrum along the line of sight, averaged over rows:
//   P(k_m) = (V/N^2) < |sum_i dF_i exp(-2 pi i m i / N)|^2 >,  dF = F / <F> - 1,  m = 0 .. N/2   (reading O5)
//
// One CTA transforms two rows at a time as ONE complex FFT (row A in the real part, row B in the imaginary
// part; X_A(m) = (Z(m) + conj Z(N-m))/2, X_B(m) = (Z(m) - conj Z(N-m))/(2i)): an iterative radix-2
// decimation-in-time FFT in shared memory (bit-reversed load, log2 N butterfly stages, twiddles from a
// shared table built once per CTA with sincospif), |X|^2 accumulated in double per CTA and added to the
// global accumulator once at the end.  4 B read per pixel; the butterflies make it shared-memory bound, not
// HBM bound.
#include "lya_internal.h"

namespace {

struct PowArgs {
    const float *flux;
    size_t       n_rows;
    int          n, log2n;
    float        inv_mean;
    double      *acc;          // device, n/2 + 1 doubles, zeroed by the host
};

__global__ void __launch_bounds__(256) flux_power_kernel(const PowArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = a.n, nh = n >> 1;
    double *pw  = reinterpret_cast<double *>(smem_raw);                    // [nh + 1] (+1 pad)
    float2 *z   = reinterpret_cast<float2 *>(pw + nh + 2);                 // [n]
    float2 *tw  = z + n;                                                   // [nh]
    const int tid = threadIdx.x, T = blockDim.x;

    for (int k = tid; k < nh; k += T) {
        float s, c;
        sincospif(2.0f * (float)k / (float)n, &s, &c);
        tw[k] = make_float2(c, -s);
    }
    for (int m = tid; m <= nh; m += T) pw[m] = 0.0;

    const size_t n_pairs = (a.n_rows + 1) >> 1;
    for (size_t pair = blockIdx.x; pair < n_pairs; pair += gridDim.x) {
        const float *ra = a.flux + (2 * pair) * (size_t)n;
        const bool has_b = 2 * pair + 1 < a.n_rows;
        const float *rb = ra + n;
        __syncthreads();                                   // previous pair's read-out done (and tables built)
        for (int i = tid; i < n; i += T) {
            const int r = (int)(__brev((unsigned int)i) >> (32 - a.log2n));
            const float fa = fmaf(__ldcs(ra + i), a.inv_mean, -1.0f);
            const float fb = has_b ? fmaf(__ldcs(rb + i), a.inv_mean, -1.0f) : 0.0f;
            z[r] = make_float2(fa, fb);
        }
        __syncthreads();
        for (int s = 0; s < a.log2n; ++s) {
            const int half = 1 << s, tstep = nh >> s;
            for (int bfly = tid; bfly < nh; bfly += T) {
                const int pos = bfly & (half - 1);
                const int i0 = ((bfly >> s) << (s + 1)) + pos, i1 = i0 + half;
                const float2 w = tw[pos * tstep], u = z[i0], v = z[i1];
                const float tr = w.x * v.x - w.y * v.y, ti = w.x * v.y + w.y * v.x;
                z[i0] = make_float2(u.x + tr, u.y + ti);
                z[i1] = make_float2(u.x - tr, u.y - ti);
            }
            __syncthreads();
        }
        for (int m = tid; m <= nh; m += T) {
            const float2 p = z[m], q = z[(n - m) & (n - 1)];
            // X_A = (p + conj q)/2, X_B = (p - conj q)/(2i)
            const float ar = 0.5f * (p.x + q.x), ai = 0.5f * (p.y - q.y);
            const float br = 0.5f * (p.y + q.y), bi = 0.5f * (q.x - p.x);
            pw[m] += (double)(ar * ar + ai * ai) + (double)(br * br + bi * bi);
        }
    }
    __syncthreads();
    for (int m = tid; m <= nh; m += T)
        if (pw[m] != 0.0) atomicAdd(a.acc + m, pw[m]);
}

}  // namespace

extern "C" lya_status lya_flux_power_rows(lya_ctx *ctx, size_t n_rows, int32_t n_pix, double dv_kms,
                                          const float *flux, double mean_flux, double *power)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!flux || ((uintptr_t)flux & 3) || !power) return lya_fail(ctx, LYA_EINVAL, "lya_flux_power_rows: null or misaligned pointer");
    if (n_rows < 1 || !(dv_kms > 0.0) || !(mean_flux > 0.0))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_power_rows: n_rows >= 1, dv > 0 and mean_flux > 0 required");
    int log2n = 0;
    while ((1 << log2n) < n_pix) ++log2n;
    if (n_pix < 8 || n_pix > 8192 || (1 << log2n) != n_pix)
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_power_rows: n_pix must be a power of two in [8, 8192]");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    const int nk = n_pix / 2 + 1;
    LYA_CUDA(ctx, cudaMemsetAsync(ctx->d_stats, 0, (size_t)nk * sizeof(double), ctx->stream));
    PowArgs a{flux, n_rows, n_pix, log2n, (float)(1.0 / mean_flux), ctx->d_stats};
    const size_t smem = (size_t)(nk + 1) * sizeof(double) + (size_t)n_pix * sizeof(float2) + (size_t)(n_pix / 2) * sizeof(float2);
    int threads = n_pix / 2;
    threads = threads < 32 ? 32 : (threads > 256 ? 256 : threads);
    LYA_CUDA(ctx, cudaFuncSetAttribute(flux_power_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    LYA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, flux_power_kernel, threads, smem));
    if (per_sm < 1) return lya_fail(ctx, LYA_ECUDA, "flux_power_kernel: zero occupancy");
    const size_t n_pairs = (n_rows + 1) / 2, cap = (size_t)ctx->sm_count * per_sm;
    flux_power_kernel<<<(int)(n_pairs < cap ? n_pairs : cap), threads, smem, ctx->stream>>>(a);
    ctx->launches++;
    LYA_CUDA(ctx, cudaGetLastError());
    LYA_CUDA(ctx, cudaMemcpyAsync(power, ctx->d_stats, (size_t)nk * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const double scale = dv_kms / ((double)n_pix * (double)n_rows);        // V / N^2 / n_rows
    for (int m = 0; m < nk; ++m) power[m] *= scale;
    return LYA_OK;
}
