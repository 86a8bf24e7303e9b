// forest_host.cu -- lya_forest_host: S1..S5 end to end from HOST buffers, z-slab streamed
// (the build's analogue of the paper's "only read into memory a small section of the volume at any one
// time", App. B).  Slab s+1 is copied host->device on ctx->copy_stream while slab s runs
// S1 + S3 (one kernel: LYA_TAU_FROM_DENSITY) on ctx->stream; tau stays resident for S4; S5 streams F back chunk by chunk.
#include "lya_internal.h"

namespace {

lya_status ensure_ws(lya_ctx *ctx, size_t bytes)
{
    if (ctx->ws_bytes >= bytes) return LYA_OK;
    if (ctx->ws) { cudaFree(ctx->ws); ctx->ws = nullptr; ctx->ws_bytes = 0; }
    cudaError_t e = cudaMalloc(&ctx->ws, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return lya_fail(ctx, LYA_ENOMEM, "lya_forest_host: device workspace allocation failed"); }
    ctx->ws_bytes = bytes;
    return LYA_OK;
}

}  // namespace

extern "C" lya_status lya_forest_host(lya_ctx *ctx, const lya_params *p, int axis, int32_t slab_nz,
                                      const float *delta_h, const float *v_pec_h, double f_target,
                                      double rel_tol, int max_iter, float *tau_h, float *flux_h,
                                      double *a_out, double *f_achieved, int *iters)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!p || !delta_h || !v_pec_h) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: null pointer");
    if (axis < 0 || axis > 2) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: axis must be 0, 1 or 2");
    lya_scalars sc;
    if (lya_scalars_from_params(p, axis, &sc) != LYA_OK) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: bad parameters");
    if (!(f_target > 0.0 && f_target < 1.0) || !(rel_tol > 0.0) || max_iter < 2)
        return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: bad f_target / rel_tol / max_iter");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));

    const size_t plane = (size_t)p->nx * p->ny, total = plane * p->nz;
    int snz = slab_nz;
    if (axis == 2) snz = p->nz;
    if (snz <= 0) {                                   // ~16 slabs, each between 2^20 and 2^28 cells: only the
        size_t cells = total / 16;                    // first slab's copy and the last slab's sums are exposed
        if (cells < ((size_t)1 << 20)) cells = (size_t)1 << 20;
        if (cells > ((size_t)1 << 28)) cells = (size_t)1 << 28;
        snz = (int)((cells + plane - 1) / plane);
    }
    if (snz > p->nz) snz = p->nz;
    const size_t slab_cells = plane * snz;
    const int n_slabs = (p->nz + snz - 1) / snz;

    lya_status st = ensure_ws(ctx, (total + 4 * slab_cells) * sizeof(float) + 256);
    if (st != LYA_OK) return st;
    float *tau = (float *)ctx->ws;
    float *d_delta[2] = {tau + total, tau + total + slab_cells};
    float *d_v[2]     = {tau + total + 2 * slab_cells, tau + total + 3 * slab_cells};

    auto copy_in = [&](int s) -> cudaError_t {
        const int buf = s & 1;
        const size_t off = (size_t)s * slab_cells;
        const size_t cells = (s == n_slabs - 1) ? total - off : slab_cells;
        cudaError_t e = cudaSuccess;
        if (s >= 2) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_comp[buf], 0);   // buffer free again
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_delta[buf], delta_h + off, cells * 4, cudaMemcpyHostToDevice, ctx->copy_stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_v[buf], v_pec_h + off, cells * 4, cudaMemcpyHostToDevice, ctx->copy_stream);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_copy[buf], ctx->copy_stream);
        return e;
    };

    LYA_CUDA(ctx, copy_in(0));
    for (int s = 0; s < n_slabs; ++s) {
        const int buf = s & 1;
        if (s + 1 < n_slabs) LYA_CUDA(ctx, copy_in(s + 1));
        const size_t off = (size_t)s * slab_cells;
        const size_t cells = (s == n_slabs - 1) ? total - off : slab_cells;
        const int nzl = (int)(cells / plane);
        LYA_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_copy[buf], 0));
        // S1 fused into the staging of S3 (bit-identical to the two-call path; n_HI and b never touch memory)
        st = lya_tau_sightlines_opt(ctx, p, axis, nzl, LYA_TAU_FROM_DENSITY, d_delta[buf], nullptr, d_v[buf],
                                    tau + off, nullptr);
        if (st != LYA_OK) return st;
        LYA_CUDA(ctx, cudaEventRecord(ctx->ev_comp[buf], ctx->stream));
    }
    if (tau_h) LYA_CUDA(ctx, cudaMemcpyAsync(tau_h, tau, total * 4, cudaMemcpyDeviceToHost, ctx->stream));

    double A = 0.0;
    st = lya_normalize_mean_flux(ctx, tau, total, f_target, rel_tol, max_iter, &A, f_achieved, iters);
    if (a_out) *a_out = A;
    if (st != LYA_OK && st != LYA_ENOCONV) return st;
    const lya_status st_norm = st;

    if (flux_h) {                                      // S5 in place, chunk c+1 computed while chunk c returns
        for (int s = 0; s < n_slabs; ++s) {
            const int buf = s & 1;
            const size_t off = (size_t)s * slab_cells;
            const size_t cells = (s == n_slabs - 1) ? total - off : slab_cells;
            st = lya_flux(ctx, tau + off, cells, A, tau + off);
            if (st != LYA_OK) return st;
            LYA_CUDA(ctx, cudaEventRecord(ctx->ev_comp[buf], ctx->stream));
            LYA_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_comp[buf], 0));
            LYA_CUDA(ctx, cudaMemcpyAsync(flux_h + off, tau + off, cells * 4, cudaMemcpyDeviceToHost, ctx->copy_stream));
        }
    }
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return st_norm;
}
