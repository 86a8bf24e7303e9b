// lya_internal.h -- private to the CUDA library (never included by oracle/ or tests).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/lya.h"

struct lya_ctx {
    int           device;
    cudaStream_t  stream;         // caller's stream: every kernel goes here
    cudaStream_t  copy_stream;    // lya_forest_host: H2D/D2H overlap
    cudaEvent_t   ev_copy[2], ev_comp[2];
    int           sm_count;
    int           max_smem_optin; // bytes per block
    int           coop_ok;        // cooperative launch supported
    uint64_t      launches;
    // reduction scratch (device): per-block partial sums, root state
    double       *d_partials;     // [2 parities][LYA_MAX_RED_BLOCKS][2*LYA_MAX_TRIALS]
    double       *h_pinned;       // pinned host memory: [0, 64) written by the kernels directly (UVA: S4 results,
                                  // partial sums), [LYA_PINNED_STATS, +LYA_STATS_DOUBLES) DMA target of the statistics
    unsigned int *d_sched;        // tau kernels' work counter [0..1] (zeroed on the stream before every launch), pair counter [2..3],
                                  // [4] ticket of the statistics kernels (the last CTA to finish writes the result to h_pinned)
    int           stats_dirty;    // a statistics call did not complete: d_stats / the ticket are re-zeroed before the next one
    double       *d_stats;        // 8192 doubles: flux-PDF counts (as uint64) / power-spectrum accumulators
    float        *d_taps, *h_taps; // lya_observe_rows: Gaussian taps (device / host staging), grown on demand
    size_t        taps_cap;
    double        taps_key[4];    // (sigma_px, Kl, Kr, KO) of the taps now on the device
    void         *d_bins, *h_bins; // lya_observe_rows: per-bin geometry table (int4 per output bin)
    size_t        bins_cap;
    double        bins_key[3];    // (bin_px, n_pix, n_bins) of the table now on the device
    int           fft_dims[3];    // lya_fields_from_dm: cached cuFFT plans (handles are ints) for [nz][ny][nx]
    int           fft_r2c, fft_c2r;
    // lya_forest_host / lya_fields_from_dm workspace (device), grown on demand
    void         *ws;
    size_t        ws_bytes;
    double       *forest_rowm;                 // per-sightline plain moments of that tau (inside ws)
    size_t        forest_rows;
    size_t        forest_total, forest_slab;   // cells of the tau lya_forest_host_begin left resident in ws (0: none), chunk size
    size_t        norm_sub_every, norm_sub_min;  // S4's nested iteration: subsample stride [4 KiB chunks], smallest n_pix that uses it
    int           norm_occ;                      // CTAs of normalize_kernel per SM (0: not asked yet, -1: none)
    double        norm_stats[4];                 // last lya_normalize_mean_flux: passes over tau, subsample passes, row pass, n_sub
    char          err[512];
};

#define LYA_MAX_RED_BLOCKS 2048
#define LYA_MAX_TRIALS     8
#define LYA_STATS_DOUBLES   8192
#define LYA_PINNED_STATS    64

// Statistics kernels (flux PDF, S5 + PDF, flux power) accumulate into ctx->d_stats with atomics; the LAST CTA to finish
// (ticket d_sched[4]) copies the totals to the mapped pinned mirror and leaves d_stats and the ticket zeroed for the next
// call, so a call is one launch and one synchronisation: no memset, no copy to enqueue.
lya_status lya_stats_begin(lya_ctx *ctx, size_t n_doubles);
// replicas of an n-entry accumulator inside d_stats (a CTA adds into replica blockIdx.x % reps; the last CTA sums them).
// They matter when the launch is short: all CTAs finish together and their atomics to the same n addresses serialise
// (256^3: 25 of the flux-PDF kernel's 47 us).  On long launches the CTAs drift apart and the replicas only add work to
// the last CTA, so inputs beyond 2^28 pixels take one copy; max_reps bounds the last CTA's n * reps loads.
static inline int lya_stats_replicas(size_t n, size_t n_pixels, int max_reps)
{
    size_t r = n ? LYA_STATS_DOUBLES / n : 1;
    if (n_pixels > ((size_t)1 << 28)) return 1;
    return (int)(r < 1 ? 1 : (r > (size_t)max_reps ? (size_t)max_reps : r));
}
lya_status lya_stats_end(lya_ctx *ctx);                  // synchronises; the results are in h_pinned + LYA_PINNED_STATS

static inline lya_status lya_fail(lya_ctx *ctx, lya_status s, const char *msg)
{
    if (ctx) {
        strncpy(ctx->err, msg, sizeof(ctx->err) - 1);
        ctx->err[sizeof(ctx->err) - 1] = 0;
    }
    return s;
}

static inline lya_status lya_cuda_fail(lya_ctx *ctx, cudaError_t e, const char *where)
{
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s: %s", where, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? LYA_ENOMEM : LYA_ECUDA;
}

#define LYA_CUDA(ctx, call)                                              \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return lya_cuda_fail((ctx), e__, #call); \
    } while (0)

// Physical constants (cgs, CODATA 2018 / IAU 2015), typed in here independently of oracle/.
#define LYA_K_BOLTZ    1.380649e-16           // erg/K
#define LYA_M_PROTON   1.67262192369e-24      // g   (b uses m_p: DESIGN.md reading C6)
#define LYA_M_HATOM    1.6735575e-24          // g   (nbar_H)
#define LYA_CM_PER_MPC 3.0856775814913673e24
#define LYA_C_CGS      2.99792458e10          // cm/s
#define LYA_SIGMA_LYA  4.48e-18               // cm^2
#define LYA_RHOCRIT100 1.87834e-29            // g/cm^3 for h = 1
#define LYA_NHI_COEFF  7.24e-6                // Eq.4
#define LYA_ALPHA_T    (-0.7)                 // recombination-rate temperature slope

void lya_fields_release(lya_ctx *ctx);   // fields.cu: destroys the cached cuFFT plans

// lya_api.cu: raises the kernel's dynamic shared-memory limit to `smem` if needed and returns the resident CTAs per SM
// (both remembered process-wide per device, kernel, block size and byte count)
lya_status lya_kernel_occupancy(lya_ctx *ctx, const void *fn, int threads, size_t smem, int *per_sm);

// kernels' host launchers (each enqueues on ctx->stream and bumps ctx->launches)
lya_status lya_launch_gas(lya_ctx *ctx, const float *delta, size_t n, float *n_hi, float *b,
                          float nbar_hi, float b0, float half_gm1, float pivot);
// flags: LYA_TAU_*; gas5 = {nbar_hi, b0, (gamma-1)/2, -0.7 (gamma-1), pivot} when LYA_TAU_FROM_DENSITY (n_hi
// then points at delta, b is ignored); d_pairs: device counter of evaluated pairs or NULL
lya_status lya_launch_tau(lya_ctx *ctx, int axis, int nx, int ny, int nz_local,
                          const float *n_hi, const float *b, const float *v, float *tau,
                          double amp_scale, double dv_kms, unsigned flags, const float *gas5,
                          unsigned long long *d_pairs, double *d_rowm);
lya_status lya_launch_flux(lya_ctx *ctx, const float *tau, size_t n, double a, float *flux);
// rowm / n_rows: per-sightline plain moments of lya_tau_sightlines_opt (pass 0 reads them instead of tau) or NULL / 0
lya_status lya_run_normalize(lya_ctx *ctx, const float *tau, size_t n, const double *rowm, size_t n_rows,
                             double f_target, double rel_tol, int max_iter, double *a_out, double *f_out, int *iters);
lya_status lya_run_row_moment_sums(lya_ctx *ctx, const double *rowm, size_t n_rows, double *sums5);
lya_status lya_run_flux_with_pdf(lya_ctx *ctx, const float *tau, size_t n, double a, float *flux, int n_bins,
                                 double f_lo, double width, uint64_t *counts, double *pdf);
// every > 1: over the subsample (every `every`-th 4 KiB chunk of tau); n_sub receives the pixels summed over (or NULL)
lya_status lya_run_moment_sums(lya_ctx *ctx, const float *tau, size_t n, double a_trial, size_t every, double *sums5,
                               uint64_t *n_sub);
lya_status lya_run_partial_sums(lya_ctx *ctx, const float *tau, size_t n, const double *a_trial, int k,
                                double *sums, double *dsums);
