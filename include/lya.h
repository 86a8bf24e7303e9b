/* lya.h -- C ABI of the B200 (sm_100a) Lyman-alpha forest hot path of arXiv:1105.4747
 * (Greig, Bolton & Wyithe), section 2.3, PAPER.md:70-92:
 *
 *   S1  gas state        T = T0 (1+delta)^(gamma-1) with the pivot at 1+delta = 10   Eq.5
 *                        n_HI from photo-ionisation equilibrium                     Eq.4
 *                        b = sqrt(2 k_B T / m_p)
 *   S2  u(j) = v_H(j) + v_pec(j)
 *   S3  tau(i) = c sigma_a dR / sqrt(pi) * sum_j n_HI(j)/b(j) exp(-((v_H(i)-u(j))/b(j))^2)   Eq.6
 *       (periodic in velocity: nearest image, reading C7)
 *   S4  A with <exp(-A tau)> = observed mean flux, over all pixels of all spectra
 *   S5  F = exp(-A tau)
 *
 * Every entry point is extern "C", takes plain pointers and sizes, returns a status code and never
 * throws, exits or prints.  Pointers are marked DEVICE (CUDA global memory of ctx's device, owned by
 * the caller, fp32, 4-byte aligned at least; 16-byte alignment enables the vector paths; the pointers of
 * an EMPTY array -- n_cells, n_pix or n_rows == 0 -- may be NULL: such calls return LYA_OK without a launch,
 * except lya_normalize_mean_flux, for which the mean of nothing is LYA_EINVAL) or HOST.  The library never retains or frees a caller pointer; its only allocations are private
 * scratch inside lya_ctx.  There is no CPU fallback: without a CUDA device lya_create fails with
 * LYA_ECUDA and nothing else can be called.
 *
 * Grid layout everywhere: C order [iz][iy][ix], ix contiguous.  axis 0 = sightlines along x
 * (contiguous rows), 1 = along y (stride nx), 2 = along z (stride nx*ny).
 */
#ifndef LYA_H
#define LYA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LYA_VERSION 100   /* 0.1.0 */

typedef struct lya_ctx lya_ctx;   /* opaque: device, stream, SM count, reduction scratch, workspace */

typedef enum {
    LYA_OK      = 0,
    LYA_EINVAL  = 1,   /* null / misaligned pointer, n < 1, bad axis, T0 <= 0, f_target outside (0,1), aliasing ... */
    LYA_ECUDA   = 2,   /* a CUDA runtime call failed; text via lya_last_error()                                      */
    LYA_ENOROOT = 3,   /* no A > 0 solves <exp(-A tau)> = f_target (e.g. all tau == 0)                               */
    LYA_ENOCONV = 4,   /* max_iter reached; *a_out holds the best estimate                                           */
    LYA_ENOMEM  = 5    /* device or pinned-host allocation failed                                                    */
} lya_status;

/* The paper's free parameters. All host-side doubles. */
typedef struct {
    int32_t nx, ny, nz;     /* full grid                                                                   */
    double  box_mpch;       /* comoving box length ALONG THE SIGHTLINE AXIS [h^-1 Mpc]                      */
    double  z;              /* redshift                                                                    */
    double  omega_m, h;     /* flat LCDM: omega_lambda = 1 - omega_m, radiation neglected                  */
    double  omega_b_h2;     /* Eq.4; its pivot value is 0.024                                              */
    double  gamma_m12;      /* HI photo-ionisation rate / 1e-12 s^-1, Eq.4 (degenerate with A) */
    double  y_he;           /* helium mass fraction in nbar_H = (1-Y) rho_b / m_H (reading C9)             */
    double  T0, gamma;      /* Eq.5                                                                        */
    double  delta_pivot;    /* Eq.5 pivot in 1+delta (paper: 10); <= 0 disables it                         */
} lya_params;

/* Derived scalars of one sightline direction (host double precision). */
typedef struct {
    int32_t n_pix;          /* pixels along the axis                                  */
    double  Ez, Hz;         /* E(z); H(z) [km/s/Mpc]                                  */
    double  dR_cm;          /* proper pixel width                        */
    double  dv_kms;         /* Hubble velocity width of one pixel = H(z) dR           */
    double  V_kms;          /* n_pix * dv: period of the velocity axis                */
    double  b0_kms;         /* sqrt(2 k_B T0 / m_p)                                   */
    double  nbarH, nbarHI;  /* mean proper H density; Eq.4 at delta = 0  [cm^-3]      */
    double  K;              /* c sigma_alpha dR / sqrt(pi), Eq.6 prefactor [cm^4/s]   */
    double  tau0;           /* K nbarHI / b0: line-centre amplitude at mean density   */
    double  tauGP;          /* c sigma_alpha nbarHI / H(z): Gunn-Peterson depth       */
} lya_scalars;

/* Host only, no GPU needed. LYA_EINVAL on null pointers, axis not in {0,1,2}, n < 1, box/h/T0/gamma_m12 <= 0. */
lya_status lya_scalars_from_params(const lya_params *p, int axis, lya_scalars *out);

int         lya_version(void);
const char *lya_status_string(lya_status s);

/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or
 * NULL for the legacy default stream; every kernel below is enqueued on it.  One ctx per host thread. */
lya_status  lya_create(lya_ctx **out, int device, void *cuda_stream);
void        lya_destroy(lya_ctx *ctx);
const char *lya_last_error(const lya_ctx *ctx);          /* "" if none; valid until the next call on ctx */
int         lya_sm_count(const lya_ctx *ctx);

/* S1 (Eq.4, Eq.5 + pivot, b).  delta, n_hi, b_kms: DEVICE, n_cells floats each; outputs may not alias
 * the input.  n_hi in cm^-3, b in km/s.  Precondition (not scanned): 1 + delta > 0 and finite.
 * Asynchronous on ctx's stream. */
lya_status lya_gas_from_density(lya_ctx *ctx, const lya_params *p, const float *delta, size_t n_cells,
                                float *n_hi, float *b_kms);

/* S2 + S3 (Eq.6, full periodic sum: every (i,j) pair of a sightline is evaluated).
 * All four arrays: DEVICE, [nz_local][ny][nx] floats (nz_local == nz for a whole grid; a z-slab of
 * complete rows otherwise; axis == 2 requires nz_local == nz).  v_pec_kms is the proper peculiar velocity
 * component ALONG `axis` in km/s; positive values move absorption to higher pixel index.  tau may not alias
 * an input.  Asynchronous on ctx's stream. */
lya_status lya_tau_sightlines(lya_ctx *ctx, const lya_params *p, int axis, int32_t nz_local,
                              const float *n_hi, const float *b_kms, const float *v_pec_kms, float *tau);

/* Work-efficient variants of S2 + S3, same arrays and conventions as
 * lya_tau_sightlines.  flags:
 *   LYA_TAU_WINDOWED      walk only the source cells that can contribute: a cell further from a pixel than
 *                         11.3 b_j sqrt(ln 2)/dv + |v_pec,j|/dv + 1 pixels adds ex2(-x^2) == 0 exactly in fp32 (the
 *                         result, below 2^-127, is flushed; it is < 2^-127 of the cell's line-centre depth in exact
 *                         arithmetic), so the result is BIT-IDENTICAL to the full sum while ~N / (4 + 2 reach) times
 *                         fewer pairs are evaluated.  Sightlines whose reach does not fit take the full loops.
 *   LYA_TAU_FROM_DENSITY  S1 fused into the staging: n_hi_or_delta is delta (Eq.4/5 are applied per staged
 *                         cell with the arithmetic of lya_gas_from_density, so tau is bit-identical to the
 *                         two-call path); b_kms is ignored and may be NULL.
 * pairs_evaluated: HOST, receives the number of (i,j) pairs actually evaluated, or NULL; non-NULL
 * synchronises the stream.
 * row_moments: DEVICE, [sightlines of this call][5] doubles (8-byte aligned), or NULL: receives per sightline the
 * plain moments sum_i tau_i^k, k = 0..4 (k = 0: the pixel count), summed in the kernels' epilogue while tau is
 * still in registers / shared memory (fp32 within a tile of 128 pixels, double above; fixed order: reproducible).
 * They are S4's first pass (A = 0: PAPER.md:92's mean over "all generated spectra" needs sum tau^k only) --
 * lya_normalize_mean_flux_rows / lya_row_moment_sums -- so tau is read one time fewer.  Sightline index: axis 0
 * iz ny + iy; axis 1 iz nx + ix; axis 2 iy nx + ix (iz local to the slab of this call). */
#define LYA_TAU_WINDOWED     1u
#define LYA_TAU_FROM_DENSITY 2u
lya_status lya_tau_sightlines_opt(lya_ctx *ctx, const lya_params *p, int axis, int32_t nz_local, unsigned flags,
                                  const float *n_hi_or_delta, const float *b_kms, const float *v_pec_kms,
                                  float *tau, uint64_t *pairs_evaluated, double *row_moments);

/* S4.  tau: DEVICE, n_pix floats in any layout (the mean runs over all of them).  Finds the unique A > 0
 * with mean(exp(-A tau)) = f_target by an iteration that runs entirely on the device (one cooperative
 * kernel): every pass over tau yields five tilted moments and a fifth-order step on ln <exp(-A tau)>,
 * safeguarded by Newton's step and a bisection bracket (3-5 passes).  Synchronises the
 * stream because A returns to the HOST.  rel_tol: stop when the step, or the truncation error of the step's
 * model, is below rel_tol * A (suggest 1e-7); max_iter passes over tau (suggest 60).  a_out, f_achieved, iters
 * (passes used): HOST, any may be NULL.  f_achieved is the MODEL's value of the mean flux at the returned A (the
 * iteration stops without a confirming pass when the quartic and cubic cumulant models agree to rel_tol / 10, so
 * it equals f_target to that order by construction); a caller who wants the measured mean flux at A takes
 * lya_flux_partial_sums(tau, {A}) / n_pix -- one more pass -- which the parity tests do. */
lya_status lya_normalize_mean_flux(lya_ctx *ctx, const float *tau, size_t n_pix, double f_target,
                                   double rel_tol, int max_iter,
                                   double *a_out, double *f_achieved, int *iters);

/* S4's nested iteration.  For n_pix >= min_pix the device loop first finds the root of the mean over a SUBSAMPLE of
 * tau -- of its 16-byte aligned body cut into 4 KiB chunks, every `every`-th chunk; 1 / every of the bytes per pass --
 * to 1e-3, and only then streams all of tau, starting from that root: the first full pass's fifth-order step lands on
 * the root of the FULL mean and its truncation estimate proves it, so tau is normally streamed ONCE instead of 3-5
 * times.  The returned A is the root of the mean over all pixels either way (same stopping rule; the subsample only
 * supplies the starting point).  every <= 1 disables; defaults 32 and 2^24.  lya_last_normalize_stats says how the
 * last call spent its passes; `iters` of lya_normalize_mean_flux counts tau_passes (incl. the row-moment pass). */
typedef struct {
    int32_t  tau_passes;   /* passes over ALL pixels: the full passes plus, if row moments were given, the A = 0 pass */
    int32_t  sub_passes;   /* passes over the subsample                                                          */
    int32_t  row_pass;     /* 1: the A = 0 pass read the per-sightline moments, not tau                           */
    uint64_t n_sub;        /* pixels in the subsample (0: none)                                                   */
} lya_normalize_stats;
lya_status lya_set_normalize_subsample(lya_ctx *ctx, int32_t every, size_t min_pix);
lya_status lya_last_normalize_stats(const lya_ctx *ctx, lya_normalize_stats *out);

/* S4 started from the per-sightline plain moments lya_tau_sightlines_opt wrote (row_moments DEVICE [n_rows][5], over
 * exactly the n_pix pixels of tau): the A = 0 pass reads 40 B per sightline instead of 4 B per pixel; everything
 * else as lya_normalize_mean_flux, whose result it reproduces to the iteration's tolerance (the later passes and
 * the final step use the tilted moments of tau itself).  row_moments == NULL and n_rows == 0: the plain call. */
lya_status lya_normalize_mean_flux_rows(lya_ctx *ctx, const float *tau, size_t n_pix, const double *row_moments,
                                        size_t n_rows, double f_target, double rel_tol, int max_iter,
                                        double *a_out, double *f_achieved, int *iters);
/* sums5[k] = sum over the n_rows sightlines of row_moments[.][k] (HOST out; synchronises): the A = 0 sums of a
 * sharded S4 (= lya_flux_moment_sums(tau, 0) without reading tau). */
lya_status lya_row_moment_sums(lya_ctx *ctx, const double *row_moments, size_t n_rows, double *sums5);

/* Building block of S4 for slab-wise or multi-GPU normalisation: for k trial values (1 <= k <= 8) returns
 * sums[t] = sum_p exp(-a_trial[t] tau_p) and, if dsums != NULL, dsums[t] = sum_p tau_p exp(-a_trial[t] tau_p).
 * tau DEVICE; a_trial, sums, dsums HOST.  Synchronises the stream. */
lya_status lya_flux_partial_sums(lya_ctx *ctx, const float *tau, size_t n_pix,
                                 const double *a_trial, int k, double *sums, double *dsums);

/* Host-side root iteration shared by lya_normalize_mean_flux's device loop (restated there) and by
 * callers that own the reduction (slabs, ranks): feed the GLOBAL sums of the current trial, get the next.
 * No GPU needed. */
typedef struct {
    double f_target, rel_tol;
    double n_pix;           /* global pixel count                                        */
    double lo, hi;          /* bracket: f(lo) > f_target >= f(hi); hi < 0 means unknown   */
    double a;               /* current trial                                             */
    double f_at_a;          /* mean flux at the last evaluated trial                     */
    int32_t iters;          /* passes consumed                                           */
    int32_t done;           /* 1 converged (a is final and f_at_a was evaluated AT a)    */
    int32_t status;         /* lya_status                                                */
    int32_t finishing;      /* internal: the next update only records f at the final a   */
} lya_root_state;
lya_status lya_root_init(lya_root_state *s, double f_target, double rel_tol, double n_pix_global);
lya_status lya_root_update(lya_root_state *s, double sum_exp, double sum_tau_exp);

/* The same building blocks with the five tilted moments sums5[k] = sum_p tau_p^k exp(-a_trial tau_p), k = 0..4,
 * which lya_normalize_mean_flux's device loop uses: lya_root_update_moments solves a quartic cumulant model of
 * ln <exp(-A tau)> (fifth-order convergence, 3-4 passes instead of 7-8, no confirming pass: when it sets done,
 * f_at_a is the model's value at the final a).  Feed the GLOBAL sums.  tau DEVICE; sums5 HOST. */
lya_status lya_flux_moment_sums(lya_ctx *ctx, const float *tau, size_t n_pix, double a_trial, double *sums5);
lya_status lya_root_update_moments(lya_root_state *s, const double *sums5);
/* The same sums over the subsample of lya_set_normalize_subsample (every `every`-th 4 KiB chunk of the aligned body of
 * tau; every == 1: all of tau), for callers that run the nested iteration themselves (slabs, ranks); n_sub (HOST, may be
 * NULL) receives the number of pixels summed over -- the n_pix of the subsample's own lya_root_init. */
lya_status lya_flux_moment_sums_sub(lya_ctx *ctx, const float *tau, size_t n_pix, double a_trial, int32_t every,
                                    double *sums5, uint64_t *n_sub);

/* The same five sums (the pass over tau behind every trial A) for callers that may NOT allocate -- code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The call allocates nothing and
 * frees nothing (no cudaMalloc / cudaFree, no allocating library routine) and does not synchronise: it enqueues two
 * kernels on ctx's stream.  Its per-block scratch is a file-scope static __device__ array of
 * 16384 blocks x 5 doubles = 655,360 B, which every GPU that loads the library holds until the process exits.
 *   tau    DEVICE, n_pix floats (4-byte aligned; 128-bit loads if 16-byte aligned), may be NULL if n_pix == 0;
 *   sums5  DEVICE, 5 doubles (8-byte aligned), owned by the caller: valid once the stream has reached this call.
 * Block b sums the fixed pixel range [b, b + 1) * 65536, so the result does not depend on the SM count; it agrees
 * with lya_flux_moment_sums to fp32-grouping rounding (~1e-8 relative).  LYA_EINVAL (message: lya_last_error) for
 * n_pix > LYA_STATIC_MAX_PIX, for a null / misaligned pointer and for a trial outside [0, 1e30).  All calls on a
 * device SHARE the array: calls that overlap on the GPU (different streams with no ordering between them, different
 * ctx or threads) race; calls on one stream are safe back to back.  Nothing in the array has to start at zero: each
 * call writes every partial it reads.  The first call on a device resolves the array's device address
 * (cudaGetSymbolAddress): make that one outside stream capture. */
#define LYA_STATIC_MAX_PIX ((size_t)1 << 30)
lya_status lya_flux_moment_sums_static(lya_ctx *ctx, const float *tau, size_t n_pix, double a_trial, double *sums5);

/* S5.  tau, flux: DEVICE, n_pix floats; flux == tau (in place) allowed.  Asynchronous. */
lya_status lya_flux(lya_ctx *ctx, const float *tau, size_t n_pix, double a, float *flux);

/* End-to-end S1..S5 from HOST buffers (the call bench.py's e2e number times).  delta_h, v_pec_h: HOST
 * [nz][ny][nx] floats (pinned memory makes the copies asynchronous).  The grid is processed in z-slabs of
 * slab_nz planes (0 = choose; axis 2 forces one slab): H2D copy of slab s+1 overlaps S1+S3 of slab s on a
 * second stream; tau stays resident on the device for S4; S5 then streams F back.  tau_h, flux_h: HOST
 * outputs, either may be NULL.  Device workspace is cached in ctx and freed by lya_destroy. */
lya_status lya_forest_host(lya_ctx *ctx, const lya_params *p, int axis, int32_t slab_nz,
                           const float *delta_h, const float *v_pec_h, double f_target,
                           double rel_tol, int max_iter,
                           float *tau_h, float *flux_h,
                           double *a_out, double *f_achieved, int *iters);

/* The same path in three steps, for callers that own the reduction of S4 (one rank per GPU, each holding a z-slab
 * of complete sightlines -- DESIGN.md "Multi-GPU" -- or any other outer loop over A):
 *   lya_forest_host_begin   S1 + S3 of the local grid from HOST delta_h / v_pec_h, slab-streamed exactly as in
 *                           lya_forest_host; tau stays resident in the ctx's device workspace (and is copied to
 *                           tau_h, HOST, if not NULL).  Asynchronous apart from the workspace allocation.
 *   lya_forest_moment_sums  sums5[k] = sum_p tau_p^k exp(-a_trial tau_p), k = 0..4, over the resident tau (HOST
 *                           out; synchronises): all-reduce over ranks, then lya_root_update_moments.
 *   lya_forest_host_finish  S5 with the given A in place on the resident tau, F streamed back to flux_h (HOST, may
 *                           be NULL); synchronises both streams and releases the resident tau (not the workspace).
 * LYA_EINVAL if moment_sums / finish are called with no resident tau (also after lya_fields_from_dm, which shares
 * the workspace).  On any error no copy is left in flight on the caller's buffers. */
lya_status lya_forest_host_begin(lya_ctx *ctx, const lya_params *p, int axis, int32_t slab_nz,
                                 const float *delta_h, const float *v_pec_h, float *tau_h);
lya_status lya_forest_moment_sums(lya_ctx *ctx, double a_trial, double *sums5);
/* ... over the subsample of the resident tau (as lya_flux_moment_sums_sub; every == 1: all of it) */
lya_status lya_forest_moment_sums_sub(lya_ctx *ctx, double a_trial, int32_t every, double *sums5, uint64_t *n_sub);
lya_status lya_forest_host_finish(lya_ctx *ctx, double a, float *flux_h);

/* ---------------------------------------------------------------------------------------------------------
 * After F: the paper's instrument model and its two validation statistics.
 * Spectra are ROWS: n_rows sightlines of n_pix contiguous fp32 pixels of velocity width dv_kms (sightlines
 * along x of a [nz][ny][nx] grid are already in this form), periodic in velocity.
 * --------------------------------------------------------------------------------------------------------- */

/* "convolve the spectra with a Gaussian with a FWHM = 7 km/s, and resample our spectra onto 0.05 A bins ...
 * add Gaussian distributed noise assuming S/N ~ 50 per pixel" (224 km/s, 1.0375 A, S/N 5:
 * PAPER.md:130; 170 km/s, ~1 A, S/N 3.8: PAPER.md:166).  DESIGN.md readings O1-O3. */
typedef struct {
    double fwhm_kms;    /* Gaussian FWHM [km/s]; <= 0: no convolution                                          */
    double bin_kms;     /* output bin width [km/s] (see lya_bin_kms_from_angstrom); <= 0: keep the pixels      */
    double snr;         /* continuum signal-to-noise per output bin; <= 0: no noise                            */
} lya_instrument;

/* c dlambda / (1215.67 A (1+z)): velocity width of a wavelength bin at observed Lyman-alpha.  Host only. */
double     lya_bin_kms_from_angstrom(double z, double dlambda_angstrom);
/* floor(n_pix dv / bin) output bins per row (n_pix if bin_kms <= 0); a ragged last bin is dropped.  Host only. */
int32_t    lya_instrument_bins(int32_t n_pix, double dv_kms, const lya_instrument *inst);

/* flux: DEVICE [n_rows][n_pix].  unit_noise: DEVICE [n_rows][n_bins] N(0,1) draws supplied by the caller, or
 * NULL (then snr must be <= 0).  out: DEVICE [n_rows][n_bins], n_bins = lya_instrument_bins(); may not alias
 * flux.  out = rebin(G * flux) + unit_noise / snr.  LYA_EINVAL if the Gaussian needs more than 4096 taps a
 * side or a row does not fit in shared memory.  Asynchronous on ctx's stream. */
lya_status lya_observe_rows(lya_ctx *ctx, size_t n_rows, int32_t n_pix, double dv_kms, const lya_instrument *inst,
                            const float *flux, const float *unit_noise, float *out);

/* Flux PDF (21 bins of width 0.05, the first -0.025 <= F < 0.025): counts of n fp32 fluxes in
 * n_bins (<= 256) bins [f_lo + b width, f_lo + (b+1) width); fluxes outside fall into the first / last bin
 * (reading O4).  flux DEVICE; counts (uint64) and pdf (counts / (n width)) HOST, either may be NULL.
 * Synchronises the stream. */
lya_status lya_flux_pdf(lya_ctx *ctx, const float *flux, size_t n, int32_t n_bins, double f_lo, double width,
                        uint64_t *counts, double *pdf);

/* S5 and the flux PDF in ONE pass over tau (the paper's statistic "fused on F"): flux as lya_flux (in place
 * allowed), counts / pdf as lya_flux_pdf of that flux -- bit-identical to the two calls, 8 B instead of 12 B of
 * traffic per pixel.  Synchronises the stream. */
lya_status lya_flux_with_pdf(lya_ctx *ctx, const float *tau, size_t n_pix, double a, float *flux, int32_t n_bins,
                             double f_lo, double width, uint64_t *counts, double *pdf);

/* 1D flux power spectrum: P(k_m) = (V/N^2) <|sum_i dF_i exp(-2 pi i m i/N)|^2> over the
 * rows, dF = F/mean_flux - 1, V = n_pix dv, k_m = 2 pi m / V [s/km], m = 0 .. n_pix/2.  n_pix must be a power
 * of two between 8 and 8192 (two rows per complex FFT: one warp per transform for rows of 256 to 2048 pixels, a Stockham
 * radix-16/8/4 FFT per CTA in shared memory otherwise).  flux DEVICE [n_rows][n_pix];
 * power HOST, n_pix/2 + 1 doubles [km/s].  Synchronises the stream. */
lya_status lya_flux_power_rows(lya_ctx *ctx, size_t n_rows, int32_t n_pix, double dv_kms, const float *flux,
                               double mean_flux, double *power);

/* ---------------------------------------------------------------------------------------------------------
 * Before the hot path: the baryon density and the peculiar velocity from a
 * dark-matter density field, sections 2.1-2.2 of the paper.
 *   Eq.1  delta_b(k) = delta_DM(k) / (1 + k^2 / k_F^2)
 *   Eq.3  v(k) = E_+ i k / k^2 delta_DM(k),  E_+ = H(z) f(z) / (1+z)  (delta_DM already at z: U1)
 * k is the comoving wavevector in Mpc^-1, k_i = 2 pi m_i h / L_i (readings U1-U5 in DESIGN.md section 12).  The
 * 3D transforms are cuFFT's (a library primitive, loaded with dlopen on first use: LYA_ECUDA if it is not
 * installed); the k-space operators are the library's own kernels.
 * --------------------------------------------------------------------------------------------------------- */
typedef struct {
    int32_t nx, ny, nz;
    double  box_mpch;        /* comoving box length along x [h^-1 Mpc]; cells are cubic (L_y = L ny/nx, ...)  */
    double  h, z, omega_m;   /* flat LCDM                                                                     */
    double  k_filter_mpc;    /* k_F [comoving Mpc^-1], paper: 6.5; <= 0: delta_b = delta_DM                   */
} lya_field_params;

/* f = dln D_+ / dln a of flat LCDM (Heath 1977 integral by Simpson quadrature).  Host only. */
lya_status lya_growth_rate(double z, double omega_m, double *f_out);

/* delta_dm: DEVICE [nz][ny][nx] fp32.  delta_b, v_x, v_y, v_z: DEVICE outputs of the same shape, any may be NULL
 * (v in km/s, proper, along +axis: what lya_tau_sightlines takes); no output may alias delta_dm or another output.  Asynchronous on ctx's stream apart from the first call's
 * plan creation.  Workspace (one complex half-spectrum, 8 (nx/2+1) ny nz bytes, for delta(k) and one per requested
 * output -- a single k-space kernel then serves all outputs from one read of delta(k); two in all if the device cannot
 * hold that -- plus cuFFT's) is cached in ctx. */
lya_status lya_fields_from_dm(lya_ctx *ctx, const lya_field_params *p, const float *delta_dm,
                              float *delta_b, float *v_x, float *v_y, float *v_z);

/* Roofline denominator of the tau kernel (BASELINE.json: "MUFU.EX2 ... issue rate from SM count x clock"):
 * runs a pure ex2.approx micro-kernel on every SM of ctx's device and returns MUFU.EX2 results per second
 * (HOST double; best of 3 after a warm-up).  Synchronises the stream.  16 / clk / SM on B200. */
lya_status lya_measure_mufu_peak(lya_ctx *ctx, double *ex2_per_s);

/* The HBM roofline denominator measured with this library's own access pattern: a 128-bit streaming copy kernel
 * (1 read : 1 write) over n_bytes of traffic (>= 2^20; use >> L2, e.g. 2^32).  gb_per_s: HOST, read + written bytes
 * per second / 1e9, best of 5.  Allocates and frees n_bytes of device memory; synchronises. */
lya_status lya_measure_hbm_peak(lya_ctx *ctx, size_t n_bytes, double *gb_per_s);

/* Number of kernels the library has launched on this ctx since creation (bench.py's gpu_launches). */
uint64_t lya_launch_count(const lya_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* LYA_H */
