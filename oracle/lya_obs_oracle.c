/* lya_obs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain double-precision CPU statement of the steps that FOLLOW the transmitted flux in arXiv:1105.4747
 * (SURVEY.md section 8(f) ranks 1 and 2):
 *   instrument model   "convolve the spectra with a Gaussian with a FWHM = 7 km/s, and resample our spectra
 *                       onto 0.05 A bins ... add Gaussian distributed noise assuming S/N ~ 50 per pixel"
 *                       (PAPER.md:124); FWHM 224 km/s, 1.0375 A, S/N 5; 170 km/s, ~1 A,
 *                       S/N 3.8
 *   flux PDF           "21 equally spaced flux bins of width dF = 0.05, from F = 0 to F = 1 (i.e. at F = 0,
 *                       the first data point contains flux from -0.025 <= F < 0.025)"
 *   1D flux power      "1D flux PS along the line-of-sight"
 *
 * Only tests/ may build, load or call this file.  It shares nothing with the CUDA library.  Every function is
 * the plain definition: direct O(N^2) circular convolution, overlap-weighted rebinning, a counting loop, a
 * direct O(N^2) DFT.  Readings: O1 the Gaussian is circular (nearest periodic image) and
 * normalised by the discrete sum of its weights; O2 a pixel is the velocity interval [i dv, (i+1) dv) and
 * "resample" is the flux-conserving overlap-weighted mean onto bins [m B, (m+1) B), m < floor(V/B); O3 the
 * noise is N(0,1)/(S/N) relative to the continuum F = 1, its N(0,1) draws passed in; O4 the PDF bins
 * are the paper's real-number intervals [f_lo + b dF, f_lo + (b+1) dF), decided in double against the edges;
 * fluxes outside the range fall into the first / last bin; O5 the
 * power is P(k_m) = (V/N^2) <|sum_i dF_i exp(-2 pi i m i / N)|^2> with dF = F/<F> - 1, k_m = 2 pi m / V.
 *
 * Pins (tests/test_obs_oracle_pins.py): constant in -> constant out; a single spike -> the normalised Gaussian;
 * sum conservation; rebin with B = dv is the identity and with B = 2 dv the pair mean; integral conservation
 * when V/B is an integer; PDF of hand-placed values; a single cosine mode's closed-form power; Parseval;
 * numpy.fft.rfft on random rows.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>

#define OBS_PI 3.14159265358979323846

/* O1.  Fc(i) = sum_k G(d_ik) F(k) / sum_k G(d_ik),  d_ik = nearest periodic image of (i-k) dv,
 * G(d) = exp(-d^2 / (2 sigma^2)),  sigma = FWHM / (2 sqrt(2 ln 2)).  fwhm <= 0: copy. */
int obs_convolve_rows(int32_t n_pix, size_t n_rows, double dv_kms, double fwhm_kms, const double *F, double *Fc)
{
    if (n_pix < 1 || !(dv_kms > 0.0) || !F || !Fc) return 1;
    const double sigma = fwhm_kms / (2.0 * sqrt(2.0 * log(2.0)));
    const double V = dv_kms * (double)n_pix;
    for (size_t r = 0; r < n_rows; ++r) {
        const double *f = F + r * (size_t)n_pix;
        double *o = Fc + r * (size_t)n_pix;
        for (int32_t i = 0; i < n_pix; ++i) {
            if (!(fwhm_kms > 0.0)) { o[i] = f[i]; continue; }
            double num = 0.0, den = 0.0;
            for (int32_t k = 0; k < n_pix; ++k) {
                double d = (double)(i - k) * dv_kms;
                d -= V * nearbyint(d / V);
                const double g = exp(-d * d / (2.0 * sigma * sigma));
                num += g * f[k];
                den += g;
            }
            o[i] = num / den;
        }
    }
    return 0;
}

/* O2.  number of output bins for bin width B: floor(V / B) (a ragged last bin is dropped) */
int32_t obs_n_bins(int32_t n_pix, double dv_kms, double bin_kms)
{
    if (!(bin_kms > 0.0)) return n_pix;
    return (int32_t)floor((double)n_pix * dv_kms / bin_kms + 1e-9);
}

/* O2.  Fb(m) = (1/B) * integral over [m B, (m+1) B) of the piecewise-constant Fc.  bin <= 0: copy. */
int obs_rebin_rows(int32_t n_pix, size_t n_rows, double dv_kms, double bin_kms, const double *Fc, double *Fb)
{
    if (n_pix < 1 || !(dv_kms > 0.0) || !Fc || !Fb) return 1;
    const int32_t nb = obs_n_bins(n_pix, dv_kms, bin_kms);
    for (size_t r = 0; r < n_rows; ++r) {
        const double *f = Fc + r * (size_t)n_pix;
        double *o = Fb + r * (size_t)nb;
        for (int32_t m = 0; m < nb; ++m) {
            if (!(bin_kms > 0.0)) { o[m] = f[m]; continue; }
            const double lo = (double)m * bin_kms, hi = (double)(m + 1) * bin_kms;
            double acc = 0.0;
            for (int32_t i = 0; i < n_pix; ++i) {
                const double a = (double)i * dv_kms, b = (double)(i + 1) * dv_kms;
                const double l = a > lo ? a : lo, h = b < hi ? b : hi;
                if (h > l) acc += (h - l) * f[i];
            }
            o[m] = acc / bin_kms;
        }
    }
    return 0;
}

/* O3.  Fobs = Fb + n / snr, n ~ N(0,1) handed in.  snr <= 0: copy. */
int obs_add_noise(size_t n, double snr, const double *Fb, const float *unit_noise, double *Fobs)
{
    if (!Fb || !Fobs) return 1;
    for (size_t i = 0; i < n; ++i)
        Fobs[i] = (snr > 0.0 && unit_noise) ? Fb[i] + (double)unit_noise[i] / snr : Fb[i];
    return 0;
}

/* O4.  The paper's bins are real-number intervals: "21 equally spaced flux bins of width dF = 0.05 ... the first
 * data point contains flux from -0.025 <= F < 0.025", i.e. bin b = [e_b, e_{b+1}) with the lower
 * edge inclusive, e_b = f_lo + b width.  Each fp32 flux is promoted to double (exact) and compared with the
 * edges e_b = fma(b, width, f_lo): the correctly rounded double of f_lo + b width.  Rounding an edge is monotone,
 * so "F >= e_b" here equals the real-number comparison for every fp32 F except an F that IS the rounded edge;
 * for the paper's bins the rounded edges are the correctly rounded (2b-1)/40 -- exactly 0.125, 0.375, 0.625,
 * 0.875 where those are dyadic -- which tests/test_obs_oracle_pins.py pins.  The bin is found by counting edges,
 * no arithmetic on F.  Fluxes below the first / above the last edge fall into the first / last bin; NaN compares
 * false with every edge and goes to bin 0.  pdf[b] = counts[b] / (n width). */
int obs_flux_pdf(const float *F, size_t n, int32_t n_bins, double f_lo, double width, uint64_t *counts, double *pdf)
{
    if (!F || n_bins < 1 || !(width > 0.0) || !counts || !pdf) return 1;
    for (int32_t b = 0; b < n_bins; ++b) counts[b] = 0;
    for (size_t i = 0; i < n; ++i) {
        const double f = (double)F[i];
        int32_t b = 0;
        while (b + 1 < n_bins && f >= fma((double)(b + 1), width, f_lo)) ++b;
        counts[b] += 1;
    }
    for (int32_t b = 0; b < n_bins; ++b) pdf[b] = n ? (double)counts[b] / ((double)n * width) : 0.0;
    return 0;
}

/* the edge e_b itself, for the pins */
double obs_flux_pdf_edge(int32_t b, double f_lo, double width) { return fma((double)b, width, f_lo); }

/* O5.  P[m], m = 0 .. n_pix/2, by direct summation of the DFT of dF = F/mean_flux - 1, averaged over rows. */
int obs_flux_power(int32_t n_pix, size_t n_rows, double dv_kms, const double *F, double mean_flux, double *P)
{
    if (n_pix < 1 || n_rows < 1 || !(dv_kms > 0.0) || !(mean_flux > 0.0) || !F || !P) return 1;
    const int32_t nk = n_pix / 2 + 1;
    const double V = dv_kms * (double)n_pix;
    for (int32_t m = 0; m < nk; ++m) P[m] = 0.0;
    for (size_t r = 0; r < n_rows; ++r) {
        const double *f = F + r * (size_t)n_pix;
        for (int32_t m = 0; m < nk; ++m) {
            double re = 0.0, im = 0.0;
            for (int32_t i = 0; i < n_pix; ++i) {
                const double d = f[i] / mean_flux - 1.0;
                const double ph = -2.0 * OBS_PI * (double)(((int64_t)m * i) % n_pix) / (double)n_pix;
                re += d * cos(ph);
                im += d * sin(ph);
            }
            P[m] += re * re + im * im;
        }
    }
    for (int32_t m = 0; m < nk; ++m) P[m] *= V / ((double)n_pix * (double)n_pix) / (double)n_rows;
    return 0;
}
