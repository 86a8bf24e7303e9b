// forest_host.cu -- S1..S5 end to end from HOST buffers, z-slab streamed (the build's analogue of the paper's
// "only read into memory a small section of the volume at any one time", App. B).
//
//   lya_forest_host_begin   slab s+1 is copied host->device on ctx->copy_stream while slab s runs S1 + S3 (one
//                           kernel: LYA_TAU_FROM_DENSITY) on ctx->stream; tau stays resident in the ctx workspace
//   lya_forest_moment_sums  the five tilted moments of the resident tau at a trial A (sharded S4: the caller
//                           all-reduces them over ranks and applies lya_root_update_moments)
//   lya_forest_host_finish  S5 in place, chunk by chunk, F streamed back while the next chunk is computed
//   lya_forest_host         begin + lya_normalize_mean_flux on the resident tau + finish (one rank = whole grid)
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

// leave no copy or kernel in flight on the caller's host buffers, whatever went wrong
lya_status drain(lya_ctx *ctx, lya_status st)
{
    cudaStreamSynchronize(ctx->copy_stream);
    cudaStreamSynchronize(ctx->stream);
    return st;
}

#define LYA_CUDA_DRAIN(ctx, call)                                                    \
    do {                                                                             \
        cudaError_t e__ = (call);                                                    \
        if (e__ != cudaSuccess) return drain((ctx), lya_cuda_fail((ctx), e__, #call)); \
    } while (0)

}  // namespace

extern "C" lya_status lya_forest_host_begin(lya_ctx *ctx, const lya_params *p, int axis, int32_t slab_nz,
                                            const float *delta_h, const float *v_pec_h, float *tau_h)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    ctx->forest_total = 0;
    if (!p || !delta_h || !v_pec_h) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: null pointer");
    if (axis < 0 || axis > 2) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: axis must be 0, 1 or 2");
    lya_scalars sc;
    if (lya_scalars_from_params(p, axis, &sc) != LYA_OK) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: bad parameters");
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

    const int n_ax = axis == 0 ? p->nx : (axis == 1 ? p->ny : p->nz);
    const size_t n_rows = total / n_ax, rows_per_plane = axis == 2 ? 0 : plane / n_ax;
    const size_t fl = (total + 4 * slab_cells + 1) & ~(size_t)1;          // floats before the (8-byte aligned) moments
    lya_status st = ensure_ws(ctx, fl * sizeof(float) + n_rows * 5 * sizeof(double) + 256);
    if (st != LYA_OK) return st;
    float *tau = (float *)ctx->ws;
    double *rowm = reinterpret_cast<double *>(tau + fl);                   // per-sightline plain moments: S4's A = 0 pass
    float *d_delta[2] = {tau + total, tau + total + slab_cells};
    float *d_v[2]     = {tau + total + 2 * slab_cells, tau + total + 3 * slab_cells};

    // the workspace is shared with lya_fields_from_dm and with earlier calls whose kernels may still be queued on
    // ctx->stream: the copy stream must not overwrite it before they have finished
    LYA_CUDA(ctx, cudaEventRecord(ctx->ev_comp[0], ctx->stream));
    LYA_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_comp[0], 0));

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

    LYA_CUDA_DRAIN(ctx, copy_in(0));
    for (int s = 0; s < n_slabs; ++s) {
        const int buf = s & 1;
        if (s + 1 < n_slabs) LYA_CUDA_DRAIN(ctx, copy_in(s + 1));
        const size_t off = (size_t)s * slab_cells;
        const size_t cells = (s == n_slabs - 1) ? total - off : slab_cells;
        const int nzl = (int)(cells / plane);
        LYA_CUDA_DRAIN(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_copy[buf], 0));
        // S1 fused into the staging of S3 (bit-identical to the two-call path; n_HI and b never touch memory)
        st = lya_tau_sightlines_opt(ctx, p, axis, nzl, LYA_TAU_FROM_DENSITY, d_delta[buf], nullptr, d_v[buf],
                                    tau + off, nullptr, rowm + 5 * rows_per_plane * (size_t)s * snz);
        if (st != LYA_OK) return drain(ctx, st);
        LYA_CUDA_DRAIN(ctx, cudaEventRecord(ctx->ev_comp[buf], ctx->stream));
    }
    if (tau_h) LYA_CUDA_DRAIN(ctx, cudaMemcpyAsync(tau_h, tau, total * 4, cudaMemcpyDeviceToHost, ctx->stream));
    ctx->forest_total = total;
    ctx->forest_slab = slab_cells;
    ctx->forest_rowm = rowm;
    ctx->forest_rows = n_rows;
    return LYA_OK;
}

extern "C" lya_status lya_forest_moment_sums_sub(lya_ctx *ctx, double a_trial, int32_t every, double *sums5, uint64_t *n_sub)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!ctx->forest_total) return lya_fail(ctx, LYA_EINVAL, "lya_forest_moment_sums: no resident tau (call lya_forest_host_begin)");
    if (a_trial == 0.0 && every <= 1) {                    // the A = 0 sums over all pixels: tau is not re-read
        if (n_sub) *n_sub = ctx->forest_total;
        return lya_row_moment_sums(ctx, ctx->forest_rowm, ctx->forest_rows, sums5);
    }
    return lya_flux_moment_sums_sub(ctx, (const float *)ctx->ws, ctx->forest_total, a_trial, every, sums5, n_sub);
}

extern "C" lya_status lya_forest_moment_sums(lya_ctx *ctx, double a_trial, double *sums5)
{
    return lya_forest_moment_sums_sub(ctx, a_trial, 1, sums5, nullptr);
}

extern "C" lya_status lya_forest_host_finish(lya_ctx *ctx, double a, float *flux_h)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!ctx->forest_total) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host_finish: no resident tau (call lya_forest_host_begin)");
    if (!(a >= 0.0) || !(a < 1.0e30)) return lya_fail(ctx, LYA_EINVAL, "lya_forest_host_finish: A must be finite and >= 0");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    float *tau = (float *)ctx->ws;
    const size_t total = ctx->forest_total, slab_cells = ctx->forest_slab;
    ctx->forest_total = 0;                              // F overwrites tau: the resident tau is consumed
    if (flux_h) {                                       // S5 in place, chunk c+1 computed while chunk c returns
        int s = 0;
        for (size_t off = 0; off < total; off += slab_cells, ++s) {
            const int buf = s & 1;
            const size_t cells = (total - off < slab_cells) ? total - off : slab_cells;
            lya_status st = lya_flux(ctx, tau + off, cells, a, tau + off);
            if (st != LYA_OK) return drain(ctx, st);
            LYA_CUDA_DRAIN(ctx, cudaEventRecord(ctx->ev_comp[buf], ctx->stream));
            LYA_CUDA_DRAIN(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_comp[buf], 0));
            LYA_CUDA_DRAIN(ctx, cudaMemcpyAsync(flux_h + off, tau + off, cells * 4, cudaMemcpyDeviceToHost, ctx->copy_stream));
        }
    }
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return LYA_OK;
}

extern "C" lya_status lya_forest_host(lya_ctx *ctx, const lya_params *p, int axis, int32_t slab_nz,
                                      const float *delta_h, const float *v_pec_h, double f_target,
                                      double rel_tol, int max_iter, float *tau_h, float *flux_h,
                                      double *a_out, double *f_achieved, int *iters)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!(f_target > 0.0 && f_target < 1.0) || !(rel_tol > 0.0) || max_iter < 2)
        return lya_fail(ctx, LYA_EINVAL, "lya_forest_host: bad f_target / rel_tol / max_iter");
    lya_status st = lya_forest_host_begin(ctx, p, axis, slab_nz, delta_h, v_pec_h, tau_h);
    if (st != LYA_OK) return st;
    double A = 0.0;
    st = lya_normalize_mean_flux_rows(ctx, (const float *)ctx->ws, ctx->forest_total, ctx->forest_rowm, ctx->forest_rows,
                                      f_target, rel_tol, max_iter, &A, f_achieved, iters);
    if (a_out) *a_out = A;
    if (st != LYA_OK && st != LYA_ENOCONV) { ctx->forest_total = 0; return drain(ctx, st); }
    const lya_status st_norm = st;
    st = lya_forest_host_finish(ctx, A, flux_h);
    return st != LYA_OK ? st : st_norm;
}
