// root_iter.h -- the scalar iteration on A ("iterate A until the mean transmitted flux ...
// matches"), shared by the device-side loop of normalize.cu and the host-side lya_root_update().
//
// f(A) = mean_p exp(-A tau_p) is strictly decreasing for tau >= 0 and g(A) = ln f(A) (a cumulant generating
// function) is decreasing and CONVEX, so Newton's iteration on g(A) = ln f_target started at A = 0 climbs
// monotonically to the unique root -- and, g being exactly linear when all tau are equal, in far fewer steps
// than Newton on f itself (4-5 passes instead of 7-8 on the lognormal test fields).  A bracket [lo, hi] is
// kept from the sign of f - f_target and any step that leaves it is replaced by the midpoint (bisection),
// which makes the loop safe against rounding in f.  One pass over tau gives both sums f and -f' for the trial.
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
