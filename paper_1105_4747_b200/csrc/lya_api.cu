// lya_api.cu -- host side of the C ABI declared in include/lya.h: context, argument validation, the
// double-precision scalars of DESIGN.md "Notation", and the kernel launch wrappers.  No CPU fallback.
#include <math.h>
#include <mutex>
#include <new>

#include "lya_internal.h"
#include "root_iter.h"

namespace {

int axis_len(const lya_params *p, int axis) { return axis == 0 ? p->nx : (axis == 1 ? p->ny : p->nz); }

bool params_ok(const lya_params *p)
{
    return p && p->nx >= 1 && p->ny >= 1 && p->nz >= 1 && p->box_mpch > 0 && p->h > 0 && p->T0 > 0 &&
           p->gamma_m12 > 0 && p->omega_b_h2 > 0 && p->z > -1.0 && isfinite(p->gamma) && p->y_he < 1.0 &&
           p->omega_m >= 0;
}

}  // namespace

// Dynamic shared-memory opt-in and occupancy of a kernel, asked from the driver once per (device, kernel, block,
// bytes) and remembered process-wide: the two runtime calls cost several microseconds each, which is most of a
// launch on the small grids.  The opt-in is only ever RAISED, so launches whose answer is cached stay valid whatever
// another context on the same device asked for in between.
lya_status lya_kernel_occupancy(lya_ctx *ctx, const void *fn, int threads, size_t smem, int *per_sm)
{
    struct Entry { int dev; const void *fn; int threads; size_t smem; int per_sm; };
    static Entry table[256];
    static int n_entries = 0;
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    size_t raised = 0;
    for (int i = 0; i < n_entries; ++i) {
        const Entry &e = table[i];
        if (e.dev != ctx->device || e.fn != fn) continue;
        if (e.threads == threads && e.smem == smem) { *per_sm = e.per_sm; return LYA_OK; }
        if (e.smem > raised) raised = e.smem;
    }
    if (smem > raised && smem > 48 * 1024)
        LYA_CUDA(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int n = 0;
    LYA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fn, threads, smem));
    if (n_entries < 256) table[n_entries++] = Entry{ctx->device, fn, threads, smem, n};
    *per_sm = n;
    return LYA_OK;
}

lya_status lya_stats_begin(lya_ctx *ctx, size_t n_doubles)
{
    if (ctx->stats_dirty) {                                // an earlier statistics call failed midway: start clean
        LYA_CUDA(ctx, cudaMemsetAsync(ctx->d_stats, 0, LYA_STATS_DOUBLES * sizeof(double), ctx->stream));
        LYA_CUDA(ctx, cudaMemsetAsync(ctx->d_sched + 4, 0, sizeof(unsigned int), ctx->stream));
    }
    (void)n_doubles;
    ctx->stats_dirty = 1;
    return LYA_OK;
}

lya_status lya_stats_end(lya_ctx *ctx)
{
    LYA_CUDA(ctx, cudaGetLastError());
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->stats_dirty = 0;
    return LYA_OK;
}

extern "C" {

int lya_version(void) { return LYA_VERSION; }

const char *lya_status_string(lya_status s)
{
    switch (s) {
        case LYA_OK:      return "ok";
        case LYA_EINVAL:  return "invalid argument";
        case LYA_ECUDA:   return "CUDA error";
        case LYA_ENOROOT: return "no root";
        case LYA_ENOCONV: return "not converged";
        case LYA_ENOMEM:  return "out of memory";
    }
    return "unknown";
}

// Scalars of Eq.4 / Eq.6, all in double on the host.
lya_status lya_scalars_from_params(const lya_params *p, int axis, lya_scalars *s)
{
    if (!s || !params_ok(p) || axis < 0 || axis > 2) return LYA_EINVAL;
    const int n = axis_len(p, axis);
    const double zp1 = 1.0 + p->z;
    s->n_pix  = n;
    s->Ez     = sqrt(p->omega_m * zp1 * zp1 * zp1 + (1.0 - p->omega_m));
    s->Hz     = 100.0 * p->h * s->Ez;
    const double dR_mpc = p->box_mpch / ((double)n * p->h * zp1);           // proper pixel width [Mpc]
    s->dR_cm  = dR_mpc * LYA_CM_PER_MPC;
    s->dv_kms = s->Hz * dR_mpc;
    s->V_kms  = s->dv_kms * (double)n;
    s->b0_kms = sqrt(2.0 * LYA_K_BOLTZ * p->T0 / LYA_M_PROTON) * 1.0e-5;
    s->nbarH  = (1.0 - p->y_he) * p->omega_b_h2 * LYA_RHOCRIT100 * (zp1 * zp1 * zp1) / LYA_M_HATOM;
    s->nbarHI = LYA_NHI_COEFF * s->nbarH * pow(p->T0 * 1.0e-4, LYA_ALPHA_T) * (p->omega_b_h2 / 0.024) /
                p->gamma_m12 * pow(zp1 * 0.25, 3.0);                        // Eq.4 at delta = 0
    s->K      = LYA_C_CGS * LYA_SIGMA_LYA * s->dR_cm / sqrt(M_PI);          // Eq.6 prefactor
    s->tau0   = s->K * s->nbarHI / (s->b0_kms * 1.0e5);
    s->tauGP  = LYA_C_CGS * LYA_SIGMA_LYA * s->nbarHI / (s->Hz * 1.0e5 / LYA_CM_PER_MPC);
    return LYA_OK;
}

lya_status lya_create(lya_ctx **out, int device, void *cuda_stream)
{
    if (!out) return LYA_EINVAL;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) {
        cudaGetLastError();
        return LYA_ECUDA;                                   // no device: there is no fallback path
    }
    lya_ctx *ctx = new (std::nothrow) lya_ctx();
    if (!ctx) return LYA_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = device;
    ctx->taps_key[0] = ctx->bins_key[0] = -1.0;
    ctx->norm_sub_every = 32;                              // S4's nested iteration (lya_set_normalize_subsample)
    ctx->norm_sub_min = (size_t)1 << 24;
    ctx->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->coop_ok, cudaDevAttrCooperativeLaunch, device);
    const size_t part_bytes = (size_t)2 * LYA_MAX_RED_BLOCKS * 2 * LYA_MAX_TRIALS * sizeof(double);
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_partials, part_bytes);
    if (e == cudaSuccess) e = cudaMallocHost((void **)&ctx->h_pinned, (LYA_PINNED_STATS + LYA_STATS_DOUBLES) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_stats, LYA_STATS_DOUBLES * sizeof(double));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_stats, 0, LYA_STATS_DOUBLES * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_sched, 8 * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_sched, 0, 8 * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&ctx->ev_copy[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_comp[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
        lya_destroy(ctx);
        return e == cudaErrorMemoryAllocation ? LYA_ENOMEM : LYA_ECUDA;
    }
    *out = ctx;
    return LYA_OK;
}

void lya_destroy(lya_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    lya_fields_release(ctx);
    if (ctx->ws) cudaFree(ctx->ws);
    if (ctx->d_partials) cudaFree(ctx->d_partials);
    if (ctx->d_sched) cudaFree(ctx->d_sched);
    if (ctx->d_stats) cudaFree(ctx->d_stats);
    if (ctx->d_taps) cudaFree(ctx->d_taps);
    free(ctx->h_taps);
    if (ctx->d_bins) cudaFree(ctx->d_bins);
    free(ctx->h_bins);
    if (ctx->h_pinned) cudaFreeHost(ctx->h_pinned);
    for (int i = 0; i < 2; ++i) {
        if (ctx->ev_copy[i]) cudaEventDestroy(ctx->ev_copy[i]);
        if (ctx->ev_comp[i]) cudaEventDestroy(ctx->ev_comp[i]);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
}

const char *lya_last_error(const lya_ctx *ctx) { return ctx ? ctx->err : "null context"; }
int lya_sm_count(const lya_ctx *ctx) { return ctx ? ctx->sm_count : 0; }
uint64_t lya_launch_count(const lya_ctx *ctx) { return ctx ? ctx->launches : 0; }

lya_status lya_gas_from_density(lya_ctx *ctx, const lya_params *p, const float *delta, size_t n_cells,
                                float *n_hi, float *b_kms)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!params_ok(p)) return lya_fail(ctx, LYA_EINVAL, "lya_gas_from_density: bad parameters");
    if (n_cells == 0) return LYA_OK;                 // nothing to do; pointers of empty arrays may be NULL
    if (!delta || !n_hi || !b_kms) return lya_fail(ctx, LYA_EINVAL, "lya_gas_from_density: null pointer");
    if ((((uintptr_t)delta | (uintptr_t)n_hi | (uintptr_t)b_kms) & 3) != 0)
        return lya_fail(ctx, LYA_EINVAL, "lya_gas_from_density: pointers must be 4-byte aligned");
    if (n_hi == delta || b_kms == delta || n_hi == b_kms)
        return lya_fail(ctx, LYA_EINVAL, "lya_gas_from_density: outputs may not alias");
    lya_scalars s;
    lya_scalars_from_params(p, 0, &s);          // nbarHI and b0 do not depend on the axis
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    const float pivot = p->delta_pivot > 0.0 ? (float)p->delta_pivot : INFINITY;
    return lya_launch_gas(ctx, delta, n_cells, n_hi, b_kms, (float)s.nbarHI, (float)s.b0_kms,
                          (float)(0.5 * (p->gamma - 1.0)), pivot);
}

lya_status lya_tau_sightlines_opt(lya_ctx *ctx, const lya_params *p, int axis, int32_t nz_local, unsigned flags,
                                  const float *n_hi, const float *b_kms, const float *v_pec_kms, float *tau,
                                  uint64_t *pairs_evaluated, double *row_moments)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    const bool fused = (flags & LYA_TAU_FROM_DENSITY) != 0;
    if (flags & ~(LYA_TAU_WINDOWED | LYA_TAU_FROM_DENSITY)) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: unknown flag");
    if (!params_ok(p)) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: bad parameters");
    if (axis < 0 || axis > 2) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: axis must be 0, 1 or 2");
    if (nz_local < 1 || nz_local > p->nz) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: bad nz_local");
    if (axis == 2 && nz_local != p->nz)
        return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: axis 2 needs the whole grid (nz_local == nz)");
    if (fused) b_kms = nullptr;
    if (!n_hi || (!fused && !b_kms) || !v_pec_kms || !tau) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: null pointer");
    if ((((uintptr_t)n_hi | (uintptr_t)b_kms | (uintptr_t)v_pec_kms | (uintptr_t)tau) & 3) != 0)
        return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: pointers must be 4-byte aligned");
    if (tau == n_hi || tau == b_kms || tau == v_pec_kms)
        return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: tau may not alias an input");
    if ((uintptr_t)row_moments & 7) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: row_moments must be 8-byte aligned");
    if (axis_len(p, axis) > (1 << 22))
        return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: more than 2^22 pixels per sightline");
    lya_scalars s;
    lya_scalars_from_params(p, axis, &s);
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    const float pivot = p->delta_pivot > 0.0 ? (float)p->delta_pivot : INFINITY;
    const float half_gm1 = (float)(0.5 * (p->gamma - 1.0));
    const float gas5[5] = {(float)s.nbarHI, (float)s.b0_kms, half_gm1, (float)(2.0 * LYA_ALPHA_T) * half_gm1, pivot};
    unsigned long long *d_pairs = nullptr;
    if (pairs_evaluated) {
        d_pairs = reinterpret_cast<unsigned long long *>(ctx->d_sched + 2);      // 8-byte aligned slot
        LYA_CUDA(ctx, cudaMemsetAsync(d_pairs, 0, sizeof(unsigned long long), ctx->stream));
    }
    // amplitude a_j = K nHI / (b[km/s] 1e5 cm/km): K 1e-5 is passed so that fp32 operands stay O(1e11 x 1e-11)
    lya_status st = lya_launch_tau(ctx, axis, p->nx, p->ny, nz_local, n_hi, b_kms, v_pec_kms, tau, s.K * 1.0e-5,
                                   s.dv_kms, flags, gas5, d_pairs, row_moments);
    if (st != LYA_OK || !pairs_evaluated) return st;
    unsigned long long host = 0;
    LYA_CUDA(ctx, cudaMemcpyAsync(&host, d_pairs, sizeof(host), cudaMemcpyDeviceToHost, ctx->stream));
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    *pairs_evaluated = host;
    return LYA_OK;
}

lya_status lya_tau_sightlines(lya_ctx *ctx, const lya_params *p, int axis, int32_t nz_local,
                              const float *n_hi, const float *b_kms, const float *v_pec_kms, float *tau)
{
    return lya_tau_sightlines_opt(ctx, p, axis, nz_local, 0u, n_hi, b_kms, v_pec_kms, tau, nullptr, nullptr);
}

lya_status lya_normalize_mean_flux_rows(lya_ctx *ctx, const float *tau, size_t n_pix, const double *row_moments,
                                        size_t n_rows, double f_target, double rel_tol, int max_iter, double *a_out,
                                        double *f_achieved, int *iters)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (n_pix == 0) return lya_fail(ctx, LYA_EINVAL, "lya_normalize_mean_flux: n_pix == 0");
    if (!tau || ((uintptr_t)tau & 3)) return lya_fail(ctx, LYA_EINVAL, "lya_normalize_mean_flux: bad tau pointer");
    if ((row_moments != nullptr) != (n_rows > 0) || ((uintptr_t)row_moments & 7))
        return lya_fail(ctx, LYA_EINVAL, "lya_normalize_mean_flux_rows: row_moments and n_rows go together (8-byte aligned)");
    if (!(f_target > 0.0 && f_target < 1.0))
        return lya_fail(ctx, LYA_EINVAL, "lya_normalize_mean_flux: f_target must lie in (0,1)");
    if (!(rel_tol > 0.0) || max_iter < 2)
        return lya_fail(ctx, LYA_EINVAL, "lya_normalize_mean_flux: rel_tol > 0 and max_iter >= 2 required");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    return lya_run_normalize(ctx, tau, n_pix, row_moments, n_rows, f_target, rel_tol, max_iter, a_out, f_achieved, iters);
}

lya_status lya_normalize_mean_flux(lya_ctx *ctx, const float *tau, size_t n_pix, double f_target,
                                   double rel_tol, int max_iter, double *a_out, double *f_achieved, int *iters)
{
    return lya_normalize_mean_flux_rows(ctx, tau, n_pix, nullptr, 0, f_target, rel_tol, max_iter, a_out, f_achieved, iters);
}

lya_status lya_set_normalize_subsample(lya_ctx *ctx, int32_t every, size_t min_pix)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (every < 0 || every > 65536) return lya_fail(ctx, LYA_EINVAL, "lya_set_normalize_subsample: 0 <= every <= 65536 required");
    ctx->norm_sub_every = every < 2 ? 1 : (size_t)every;
    ctx->norm_sub_min = min_pix;
    return LYA_OK;
}

lya_status lya_last_normalize_stats(const lya_ctx *ctx, lya_normalize_stats *out)
{
    if (!ctx || !out) return LYA_EINVAL;
    out->tau_passes = (int32_t)ctx->norm_stats[0];
    out->sub_passes = (int32_t)ctx->norm_stats[1];
    out->row_pass   = (int32_t)ctx->norm_stats[2];
    out->n_sub      = (uint64_t)ctx->norm_stats[3];
    return LYA_OK;
}

lya_status lya_row_moment_sums(lya_ctx *ctx, const double *row_moments, size_t n_rows, double *sums5)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if ((n_rows > 0 && (!row_moments || ((uintptr_t)row_moments & 7))) || !sums5)
        return lya_fail(ctx, LYA_EINVAL, "lya_row_moment_sums: null or misaligned pointer");
    if (n_rows == 0) { for (int i = 0; i < 5; ++i) sums5[i] = 0.0; return LYA_OK; }
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    return lya_run_row_moment_sums(ctx, row_moments, n_rows, sums5);
}

lya_status lya_flux_partial_sums(lya_ctx *ctx, const float *tau, size_t n_pix, const double *a_trial, int k,
                                 double *sums, double *dsums)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if ((n_pix > 0 && (!tau || ((uintptr_t)tau & 3))) || !a_trial || !sums)
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_partial_sums: null or misaligned pointer");
    if (k < 1 || k > LYA_MAX_TRIALS) return lya_fail(ctx, LYA_EINVAL, "lya_flux_partial_sums: k must be 1..8");
    for (int i = 0; i < k; ++i)
        if (!(a_trial[i] >= 0.0) || !(a_trial[i] < 1.0e30))
            return lya_fail(ctx, LYA_EINVAL, "lya_flux_partial_sums: trial A must be finite and >= 0");
    if (n_pix == 0) {
        for (int i = 0; i < k; ++i) { sums[i] = 0.0; if (dsums) dsums[i] = 0.0; }
        return LYA_OK;
    }
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    return lya_run_partial_sums(ctx, tau, n_pix, a_trial, k, sums, dsums);
}

lya_status lya_flux_with_pdf(lya_ctx *ctx, const float *tau, size_t n_pix, double a, float *flux, int32_t n_bins,
                             double f_lo, double width, uint64_t *counts, double *pdf)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (n_pix > 0 && (!tau || !flux || (((uintptr_t)tau | (uintptr_t)flux) & 3)))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_with_pdf: null or misaligned pointer");
    if (!(a >= 0.0) || !(a < 1.0e30)) return lya_fail(ctx, LYA_EINVAL, "lya_flux_with_pdf: A must be finite and >= 0");
    if (n_bins < 1 || n_bins > 256 || !(width > 0.0))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_with_pdf: 1 <= n_bins <= 256 and width > 0 required");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    return lya_run_flux_with_pdf(ctx, tau, n_pix, a, flux, n_bins, f_lo, width, counts, pdf);
}

lya_status lya_root_init(lya_root_state *s, double f_target, double rel_tol, double n_pix_global)
{
    if (!s || !(f_target > 0.0 && f_target < 1.0) || !(rel_tol > 0.0) || !(n_pix_global >= 1.0)) return LYA_EINVAL;
    lya_root_reset(s, f_target, rel_tol, n_pix_global);
    return LYA_OK;
}

lya_status lya_flux_moment_sums_sub(lya_ctx *ctx, const float *tau, size_t n_pix, double a_trial, int32_t every,
                                    double *sums5, uint64_t *n_sub)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if ((n_pix > 0 && (!tau || ((uintptr_t)tau & 3))) || !sums5) return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums: null or misaligned pointer");
    if (!(a_trial >= 0.0) || !(a_trial < 1.0e30)) return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums: trial A must be finite and >= 0");
    if (every < 1 || every > 65536) return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums_sub: 1 <= every <= 65536 required");
    if (n_pix == 0) {
        for (int i = 0; i < 5; ++i) sums5[i] = 0.0;
        if (n_sub) *n_sub = 0;
        return LYA_OK;
    }
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    return lya_run_moment_sums(ctx, tau, n_pix, a_trial, (size_t)every, sums5, n_sub);
}

lya_status lya_flux_moment_sums(lya_ctx *ctx, const float *tau, size_t n_pix, double a_trial, double *sums5)
{
    return lya_flux_moment_sums_sub(ctx, tau, n_pix, a_trial, 1, sums5, nullptr);
}

lya_status lya_root_update_moments(lya_root_state *s, const double *sums5)
{
    if (!s || !sums5 || s->done) return LYA_EINVAL;
    lya_root_step_moments(s, sums5);
    return (lya_status)s->status;
}

lya_status lya_root_update(lya_root_state *s, double sum_exp, double sum_tau_exp)
{
    if (!s || s->done) return LYA_EINVAL;
    lya_root_step(s, sum_exp, sum_tau_exp);
    return (lya_status)s->status;
}

lya_status lya_flux(lya_ctx *ctx, const float *tau, size_t n_pix, double a, float *flux)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (n_pix > 0 && (!tau || !flux || (((uintptr_t)tau | (uintptr_t)flux) & 3)))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux: null or misaligned pointer");
    if (!(a >= 0.0) || !(a < 1.0e30)) return lya_fail(ctx, LYA_EINVAL, "lya_flux: A must be finite and >= 0");
    if (n_pix == 0) return LYA_OK;
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    return lya_launch_flux(ctx, tau, n_pix, a, flux);
}

}  // extern "C"
