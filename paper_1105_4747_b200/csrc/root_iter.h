// root_iter.h -- the scalar iteration on A ("iterate A until the mean transmitted flux ...
// matches"), shared by the device-side loop of normalize.cu and the host-side lya_root_update().
//
// f(A) = mean_p exp(-A tau_p) is strictly decreasing for tau >= 0 and g(A) = ln f(A) (a cumulant generating
// function) is decreasing and CONVEX, so Newton's iteration on g(A) = ln f_target started at A = 0 climbs
// monotonically to the unique root -- and, g being exactly linear when all tau are equal, in far fewer steps
// than Newton on f itself (7-8 passes on the lognormal test fields; lya_root_step_moments below needs 3-4).
// A bracket [lo, hi] is kept from the sign of f - f_target and any step that leaves it is replaced by the
// midpoint (bisection), which makes the loop safe against rounding in f.  One pass over tau gives both sums f
// and -f' for the trial.
#pragma once
#include <math.h>

#include "../../include/lya.h"

#if defined(__CUDACC__)
#define LYA_HD __host__ __device__ __forceinline__
#else
#define LYA_HD static inline
#endif

LYA_HD void lya_root_reset(lya_root_state *s, double f_target, double rel_tol, double n_pix)
{
    s->f_target = f_target;
    s->rel_tol = rel_tol;
    s->n_pix = n_pix;
    s->lo = 0.0;
    s->hi = -1.0;
    s->a = 0.0;
    s->f_at_a = 1.0;
    s->iters = 0;
    s->done = 0;
    s->status = LYA_OK;
    s->finishing = 0;
}

// sum_exp = sum_p exp(-a tau_p), sum_tau_exp = sum_p tau_p exp(-a tau_p), both over ALL pixels, at a = s->a.
LYA_HD void lya_root_step(lya_root_state *s, double sum_exp, double sum_tau_exp)
{
    const double f  = sum_exp / s->n_pix;
    const double fp = sum_tau_exp / s->n_pix;          // -f'(a) >= 0
    s->iters += 1;
    s->f_at_a = f;
    if (s->finishing) { s->done = 1; return; }
    double a_new;
    if (s->a == 0.0) {                                 // first pass: f = 1, fp = mean tau
        if (!(fp > 0.0) || !(fp < 1.0e300)) { s->status = LYA_ENOROOT; s->done = 1; return; }
        a_new = -log(s->f_target) / fp;                // Newton on ln f from 0; convexity => a_new <= root
    } else {
        if (f > s->f_target) s->lo = s->a; else s->hi = s->a;
        a_new = (fp > 0.0 && f > 0.0) ? s->a + (log(f) - log(s->f_target)) * f / fp : -1.0;
        if (s->hi >= 0.0) {
            if (!(a_new > s->lo && a_new < s->hi)) a_new = 0.5 * (s->lo + s->hi);
        } else if (!(a_new > s->lo) || !(a_new < 1.0e30)) {
            a_new = 2.0 * s->a;                        // flat f: expand
        }
    }
    if (!(a_new < 1.0e30)) { s->status = LYA_ENOROOT; s->done = 1; return; }        // f never reaches f_target
    double step = a_new - s->a;
    if (step < 0.0) step = -step;
    const bool conv = (step <= s->rel_tol * a_new) ||
                      (s->hi >= 0.0 && (s->hi - s->lo) <= s->rel_tol * s->hi);
    s->a = a_new;
    if (conv) s->finishing = 1;                        // one more pass records f at the final a
}

// The same iteration fed with the first FIVE tilted moments of one pass, S[k] = sum_p tau_p^k exp(-a tau_p):
// around the current a, ln f(a + h) = ln f(a) + K(-h) with K the cumulant generating function of tau under the
// weights exp(-a tau), so the step solves the quartic  ln f(a) - ln f_target - k1 h + k2 h^2/2 - k3 h^3/6 +
// k4 h^4/24 = 0  (fifth-order convergence instead of Newton's second).  The cubic model's root is computed as
// well: when the two agree to rel_tol/10 the truncation error is below the tolerance and the iteration stops
// WITHOUT a confirming pass (f at the final a is the model's value, exact to the same order).  Typically 3-4
// passes instead of 7.  Every model step is checked against the bracket and against the Newton-on-ln-f step
// (a lower bound of the true step by convexity); anything suspicious falls back to lya_root_step's rule.
LYA_HD double lya_poly_root(double t, double k1, double k2, double k3, double k4, double h0)
{
    double h = h0;                                     // Newton on the polynomial model from the Newton step
    for (int it = 0; it < 30; ++it) {
        const double q  = t + h * (-k1 + h * (0.5 * k2 + h * (-k3 / 6.0 + h * (k4 / 24.0))));
        const double dq = -k1 + h * (k2 + h * (-0.5 * k3 + h * (k4 / 6.0)));
        if (!(dq < 0.0)) return -h0 * 1.0e300;         // model not monotone here: the caller rejects the sign
        const double dh = -q / dq;
        h += dh;
        if ((dh < 0.0 ? -dh : dh) <= 1e-15 * (h < 0.0 ? -h : h)) break;
    }
    return h;
}

LYA_HD void lya_root_step_moments(lya_root_state *s, const double *S)
{
    const double S0 = S[0];
    const double f = S0 / s->n_pix;
    s->iters += 1;
    s->f_at_a = f;
    if (s->finishing) { s->done = 1; return; }
    if (!(S0 > 0.0) || !(S[1] > 0.0) || !(S[1] < 1.0e300)) {                       // all tau == 0 (or garbage)
        if (s->a == 0.0) { s->status = LYA_ENOROOT; s->done = 1; return; }
        lya_root_step(s, S[0], S[1]);
        s->iters -= 1;
        return;
    }
    const double m1 = S[1] / S0, m2 = S[2] / S0, m3 = S[3] / S0, m4 = S[4] / S0;
    const double k1 = m1, k2 = m2 - m1 * m1, k3 = m3 - 3.0 * m2 * m1 + 2.0 * m1 * m1 * m1;
    const double k4 = m4 - 4.0 * m3 * m1 - 3.0 * m2 * m2 + 12.0 * m2 * m1 * m1 - 6.0 * m1 * m1 * m1 * m1;
    const double t = log(f) - log(s->f_target);
    if (s->a > 0.0) { if (f > s->f_target) s->lo = s->a; else s->hi = s->a; }
    const double h_newton = t / k1;
    const double h4 = lya_poly_root(t, k1, k2, k3, k4, h_newton);
    double a_new = s->a + h4;
    const double ratio = h4 / h_newton;
    // by convexity of ln f the Newton step undershoots from the left (t > 0) and overshoots from the right
    bool ok = (h_newton != 0.0) && (t > 0.0 ? (ratio > 0.999999 && ratio < 16.0) : (ratio > 0.0 && ratio < 1.000001)) &&
              (a_new > s->lo) &&
              (s->hi < 0.0 || a_new < s->hi) && (a_new < 1.0e30);
    if (h_newton == 0.0) { s->done = 1; return; }                                  // f == f_target exactly
    if (!ok) {                                         // fall back to the safeguarded Newton / bisection rule
        s->iters -= 1;
        if (s->a > 0.0) { if (f > s->f_target) s->lo = s->a; }                     // (re-applied inside, harmless)
        lya_root_step(s, S[0], S[1]);
        return;
    }
    s->a = a_new;
    // truncation estimate = |quartic root - cubic root|; a step above 5 % of A cannot pass it, so the cubic
    // solve (a dozen double divisions on one thread) is skipped there
    double trunc = 1.0e300;
    if ((h4 < 0.0 ? -h4 : h4) <= 0.05 * a_new) {
        trunc = h4 - lya_poly_root(t, k1, k2, k3, 0.0, h4);
        if (trunc < 0.0) trunc = -trunc;
    }
    if (trunc <= 0.1 * s->rel_tol * a_new) {           // model converged: stop here, report the model's f(a_new)
        const double h = h4;
        s->f_at_a = f * exp(h * (-k1 + h * (0.5 * k2 + h * (-k3 / 6.0 + h * (k4 / 24.0)))));
        s->done = 1;
    }
}
