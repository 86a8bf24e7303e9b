/* lya_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of the hot path of arXiv:1105.4747
 * (Greig, Bolton & Wyithe), section 2.3: gas state (Eq.4, Eq.5 with its
 * pivot, Doppler parameter), the optical-depth sum Eq.6 with periodic wrap, the mean-flux
 * normalisation constant A, and F = exp(-A tau).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, load or call this file.  It shares no code, header, table or constant
 * generator with the CUDA library (paper_1105_4747_b200/csrc, include/lya.h); constants
 * below are typed in from the paper / CODATA independently of that library.
 *
 * Every function follows the paper's definition term by term, in the paper's order; no
 * blocking, fusion, windowing or reordering.  The one exception is mode 1 ("skip-zero") of
 * orc_tau_sightlines, which skips calling exp() when the argument is below -750, where
 * IEEE-754 double exp() returns exactly +0 (exp(-745.2) is the last non-zero denormal), so it
 * is bit-identical to mode 0; tests/test_oracle_pins.py asserts that (pin P11).
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1 gas closed values, P2 uniform
 * field = Gunn-Peterson x theta(b/dv), P3 Poisson-summation column identity, P4 cyclic
 * shift, P5 velocity-offset equivariance, P6 single-source analytic profile, P7 brute-force
 * image sum on 8-cell sightlines, P8 Gamma scaling, P9 closed forms for A, P10 tau_eff
 * convention of PAPER.md:92, P11 skip-zero == plain.  The absolute tau/F/A values on the five
 * seeded BASELINE configs are "parity unpinned by the paper" (it prints none); they are
 * pinned only through P1-P11.
 *
 * Readings of the paper: C1 the sum in Eq.6 runs over j; C2 n_HI is
 * n_HI(j); C3 nbar_H is the mean proper density of ALL hydrogen; C4 the T in Eq.4 is the
 * local T of Eq.5 including the pivot; C6 b uses m_p; C7 nearest periodic image in velocity;
 * C9 helium fraction Y enters nbar_H = (1-Y) rho_b / m_H.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* physical constants (cgs) */
#define ORC_KB        1.380649e-16          /* erg/K                                   */
#define ORC_MP        1.67262192369e-24     /* g, proton (reading C6)                  */
#define ORC_MH        1.6735575e-24         /* g, hydrogen atom (nbar_H)               */
#define ORC_MPC_CM    3.0856775814913673e24 /* cm per Mpc                              */
#define ORC_C_CMS     2.99792458e10         /* cm/s                                    */
#define ORC_SIGMA_A   4.48e-18              /* cm^2                       */
#define ORC_RHOC_100  1.87834e-29           /* g/cm^3, critical density for h = 1      */
#define ORC_PI        3.14159265358979323846

typedef struct {
    int32_t n_pix;        /* pixels along the sightline                               */
    double  box_mpch;     /* comoving box side along the sightline [h^-1 Mpc]         */
    double  z, omega_m, h;
    double  omega_b_h2, gamma_m12, y_he;
    double  T0, gamma;
    double  delta_pivot;  /* Eq.5 pivot in 1+delta (paper: 10); <= 0 disables it      */
} orc_params;

typedef struct {
    double Ez;        /* sqrt(Om (1+z)^3 + 1 - Om)                                    */
    double Hz;        /* km/s/Mpc                                                     */
    double dR_cm;     /* proper pixel width                              */
    double dv_kms;    /* Hubble velocity width of one pixel                           */
    double V_kms;     /* n_pix * dv: box length in velocity                           */
    double b0_kms;    /* sqrt(2 kB T0 / m_p)                                          */
    double nbarH;     /* mean proper hydrogen density [cm^-3]                         */
    double nbarHI;    /* Eq.4 at delta = 0, T = T0                                    */
    double K;         /* c sigma_alpha dR / sqrt(pi)   [cm^4/s]                       */
    double tau0;      /* K nbarHI / b0: line-centre amplitude of a mean-density cell  */
    double tauGP;     /* c sigma_alpha nbarHI / H(z): Gunn-Peterson optical depth     */
} orc_scalars;

int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Scalars of section 8.0 of SURVEY.md / Eq.4, Eq.6 text. */
int orc_scalars_from_params(const orc_params *p, orc_scalars *s)
{
    if (!p || !s || p->n_pix < 1 || p->box_mpch <= 0 || p->h <= 0 || p->T0 <= 0 || p->gamma_m12 <= 0)
        return 1;
    double zp1 = 1.0 + p->z;
    s->Ez = sqrt(p->omega_m * zp1 * zp1 * zp1 + 1.0 - p->omega_m);
    s->Hz = 100.0 * p->h * s->Ez;
    double dR_mpc = p->box_mpch / ((double)p->n_pix * p->h * zp1);     /* proper Mpc */
    s->dR_cm = dR_mpc * ORC_MPC_CM;
    s->dv_kms = s->Hz * dR_mpc;
    s->V_kms = s->dv_kms * (double)p->n_pix;
    s->b0_kms = sqrt(2.0 * ORC_KB * p->T0 / ORC_MP) / 1.0e5;
    s->nbarH = (1.0 - p->y_he) * p->omega_b_h2 * ORC_RHOC_100 * zp1 * zp1 * zp1 / ORC_MH;
    s->nbarHI = 7.24e-6 * s->nbarH * pow(p->T0 / 1.0e4, -0.7) * (p->omega_b_h2 / 0.024)
                * (1.0 / p->gamma_m12) * pow(zp1 / 4.0, 3.0);                       /* Eq.4 */
    s->K = ORC_C_CMS * ORC_SIGMA_A * s->dR_cm / sqrt(ORC_PI);                      /* Eq.6 */
    s->tau0 = s->K * s->nbarHI / (s->b0_kms * 1.0e5);
    s->tauGP = ORC_C_CMS * ORC_SIGMA_A * s->nbarHI / (s->Hz * 1.0e5 / ORC_MPC_CM);
    return 0;
}

/* S1. Eq.5 with pivot, Eq.4, b. delta: fp32 input. */
int orc_gas_from_density(const orc_params *p, const float *delta, size_t n_cells,
                         double *T_out /* may be NULL */, double *nHI_out, double *b_out)
{
    orc_scalars s;
    if (orc_scalars_from_params(p, &s)) return 1;
    for (size_t c = 0; c < n_cells; ++c) {
        double D = 1.0 + (double)delta[c];
        double Dt = (p->delta_pivot > 0.0 && D > p->delta_pivot) ? p->delta_pivot : D;
        double T = p->T0 * pow(Dt, p->gamma - 1.0);                                /* Eq.5 */
        double b = sqrt(2.0 * ORC_KB * T / ORC_MP) / 1.0e5;                        /* km/s */
        double nHI = 7.24e-6 * s.nbarH * pow(T / 1.0e4, -0.7) * (p->omega_b_h2 / 0.024)
                     * (1.0 / p->gamma_m12) * D * D * pow((1.0 + p->z) / 4.0, 3.0); /* Eq.4 */
        if (T_out) T_out[c] = T;
        nHI_out[c] = nHI;
        b_out[c] = b;
    }
    return 0;
}

/* S2+S3. Eq.6 for n_sl sightlines stored contiguously [n_sl][n_pix].
 * tau(i) = K sum_j nHI(j)/b(j) exp(-((v_H(i) - u(j))/b(j))^2), u(j) = v_H(j) + v_pec(j),
 * v_H(i) - v_H(j) = (i-j) dv, difference taken to the nearest periodic image (period V).
 * mode 0: plain (exp for every pair).  mode 1: skip-zero (see header).                     */
int orc_tau_sightlines(double K, double dv_kms, int32_t n_pix, size_t n_sl,
                       const double *nHI, const double *b_kms, const float *vpec_kms,
                       double *tau, int mode)
{
    if (n_pix < 1 || dv_kms <= 0 || !nHI || !b_kms || !vpec_kms || !tau) return 1;
    const double V = dv_kms * (double)n_pix;
    long long s;
#pragma omp parallel for schedule(dynamic, 4)
    for (s = 0; s < (long long)n_sl; ++s) {
        const double *n_ = nHI + (size_t)s * n_pix;
        const double *b_ = b_kms + (size_t)s * n_pix;
        const float  *v_ = vpec_kms + (size_t)s * n_pix;
        double *t_ = tau + (size_t)s * n_pix;
        for (int32_t i = 0; i < n_pix; ++i) {
            double acc = 0.0;
            for (int32_t j = 0; j < n_pix; ++j) {
                double d = (double)(i - j) * dv_kms - (double)v_[j];   /* v_H(i) - u(j) */
                d -= V * nearbyint(d / V);                              /* nearest image  */
                double x = d / b_[j];
                double amp = K * n_[j] / (b_[j] * 1.0e5);
                if (mode == 1 && x * x > 750.0) continue;               /* exp() == +0    */
                acc += amp * exp(-x * x);
            }
            t_[i] = acc;
        }
    }
    return 0;
}

/* pairwise sum of exp(-A tau_p) over p in [lo, hi) */
static double sum_exp_pairwise(const double *tau, size_t lo, size_t hi, double A)
{
    if (hi - lo <= 64) {
        double acc = 0.0;
        for (size_t p = lo; p < hi; ++p) acc += exp(-A * tau[p]);
        return acc;
    }
    size_t mid = lo + (hi - lo) / 2;
    return sum_exp_pairwise(tau, lo, mid, A) + sum_exp_pairwise(tau, mid, hi, A);
}

static double sum_pairwise(const double *x, size_t lo, size_t hi)
{
    if (hi - lo <= 8) {
        double acc = 0.0;
        for (size_t p = lo; p < hi; ++p) acc += x[p];
        return acc;
    }
    size_t mid = lo + (hi - lo) / 2;
    return sum_pairwise(x, lo, mid) + sum_pairwise(x, mid, hi);
}

/* <exp(-A tau)> over n_pix pixels.  Fixed 65536-pixel chunks (thread-count
 * independent), each summed pairwise, then a pairwise sum of the chunk partials.          */
double orc_mean_flux(const double *tau, size_t n_pix, double A)
{
    const size_t chunk = 65536;
    size_t n_chunks = (n_pix + chunk - 1) / chunk;
    if (n_pix == 0) return NAN;
    double *part = (double *)malloc(n_chunks * sizeof(double));
    if (!part) return NAN;
    long long c;
#pragma omp parallel for schedule(static)
    for (c = 0; c < (long long)n_chunks; ++c) {
        size_t lo = (size_t)c * chunk, hi = lo + chunk < n_pix ? lo + chunk : n_pix;
        part[c] = sum_exp_pairwise(tau, lo, hi, A);
    }
    double total = sum_pairwise(part, 0, n_chunks);
    free(part);
    return total / (double)n_pix;
}

/* S4. The unique A > 0 with <exp(-A tau)> = f_target ("iterate A until ...").
 * f(A) is strictly decreasing from 1 to the fraction of tau == 0 pixels: bracket by doubling,
 * then bisect to 1e-13 relative (reading C14).  Returns 0 ok, 1 bad args, 3 no root.      */
int orc_normalize_mean_flux(const double *tau, size_t n_pix, double f_target,
                            double *A_out, double *f_achieved, int *iters)
{
    if (!tau || n_pix == 0 || !(f_target > 0.0 && f_target < 1.0)) return 1;
    double lo = 0.0, hi = 1.0;
    int it = 0;
    while (orc_mean_flux(tau, n_pix, hi) > f_target) {
        lo = hi;
        hi *= 2.0;
        if (++it > 2000 || !isfinite(hi)) return 3;
    }
    while (hi - lo > 1e-13 * hi) {
        double mid = 0.5 * (lo + hi);
        if (orc_mean_flux(tau, n_pix, mid) > f_target) lo = mid; else hi = mid;
        if (++it > 4000) break;
    }
    double A = 0.5 * (lo + hi);
    if (A_out) *A_out = A;
    if (f_achieved) *f_achieved = orc_mean_flux(tau, n_pix, A);
    if (iters) *iters = it;
    return 0;
}

/* S5. F = exp(-A tau). */
int orc_flux(const double *tau, size_t n_pix, double A, double *F)
{
    if (!tau || !F) return 1;
    for (size_t p = 0; p < n_pix; ++p) F[p] = exp(-A * tau[p]);
    return 0;
}
