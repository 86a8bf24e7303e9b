// pdf_bin.h -- the flux-PDF bin decision, shared by flux_pdf_kernel (observe.cu) and
// flux_pdf_fused_kernel (normalize.cu) so that both give identical counts.
//
// The paper's bins are real-number intervals [e_b, e_{b+1}), e_b = f_lo + b width, lower edge inclusive
// ("-0.025 <= F < 0.025").  For an fp32 flux F the comparison F >= e_b is equivalent to F >= thr_b with
// thr_b = the smallest fp32 >= e_b, so the host builds those thresholds once per call in double (e_b as the
// correctly rounded fma(b, width, f_lo)) and no rounding can move a flux across an edge:
//   t = (F - f_lo) * (1 / width) in fp32 differs from the real (F - f_lo) / width by less than
//       eps = 2^-22 (n_bins + 1 + |f_lo| / width)   [three roundings of 2^-24 relative on |t| <= n_bins + 1, plus
//       the rounding of f_lo to fp32; 2^-22 = 4 x 2^-24 leaves a third of margin],
//   so when the fractional part of t lies in (eps, 1 - eps) -- all but ~2 eps of the fluxes -- floor(t) IS the
//   real-number bin and nothing is looked up; otherwise F is compared with thr[guess] and thr[guess + 1] (loops,
//   so any guess error is absorbed; NaN and infinities end up here too).  DESIGN.md reading O4.
#pragma once
#include <math.h>

#define LYA_PDF_MAX_BINS 256

struct PdfEdges {
    float thr[LYA_PDF_MAX_BINS + 1];   // thr[b], b = 1 .. n_bins-1; thr[0] and thr[n_bins] are NaN sentinels:
                                       // every comparison with them is false, which ends the correction loops
                                       // (and sends NaN fluxes to bin 0, +-inf to the last / first bin)
    float f_lo, inv_width;
    float eps, one_minus_eps;          // fast-path band of the fractional part of t (eps >= 0.5: always look up)
    int   n_bins;
};

static inline void lya_pdf_edges(int n_bins, double f_lo, double width, PdfEdges *e)
{
    e->n_bins = n_bins;
    e->f_lo = (float)f_lo;
    e->inv_width = (float)(1.0 / width);
    const double eps = ldexp((double)n_bins + 1.0 + fabs(f_lo) / width, -22);
    e->eps = eps < 0.5 ? (float)eps : 2.0f;
    e->one_minus_eps = eps < 0.5 ? (float)(1.0 - eps) : -1.0f;
    e->thr[0] = e->thr[n_bins] = NAN;
    for (int b = 1; b < n_bins; ++b) {
        const double edge = fma((double)b, width, f_lo);
        float t = (float)edge;                           // nearest fp32
        if ((double)t < edge) t = nextafterf(t, INFINITY);
        e->thr[b] = t;                                   // smallest fp32 >= edge (+-inf if the edge overflows fp32)
    }
}

#if defined(__CUDACC__)
// s_thr: the thresholds in shared memory, n_bins + 1 floats
__device__ __forceinline__ int lya_pdf_bin(float f, const float *s_thr, int n_bins, float f_lo, float inv_width,
                                           float eps, float one_minus_eps)
{
    const float t  = (f - f_lo) * inv_width;
    const float fl = floorf(t);
    const float fr = t - fl;                             // NaN for NaN and +-inf: they take the table
    int b = min(max(__float2int_rz(fl), 0), n_bins - 1); // saturating conversion; NaN -> 0
    if (!(fr > eps && fr < one_minus_eps)) {
        while (f < s_thr[b]) --b;
        while (f >= s_thr[b + 1]) ++b;
    }
    return b;
}

// Epilogue of the statistics kernels, called by every thread of every CTA after the CTA's own atomics into ITS replica
// acc[(blockIdx.x % reps) * n + (0 .. n)): the last CTA to arrive (ticket) moves the totals over the replicas to `host`
// (mapped pinned memory) and leaves acc and the ticket zeroed for the next launch.  T is unsigned long long (counts) or
// double (power sums).  Replicas exist because all CTAs of a launch finish together: 2368 CTAs adding into the same 21
// addresses took ~25 us of same-address atomic serialisation on a 256^3 grid (the kernel: 47 us for 64 MiB).
template <typename T>
__device__ __noinline__ void lya_publish_last_cta(T *acc, int n, T *host, unsigned int *ticket, int reps)
{
    __shared__ int s_last;
    __threadfence();                                     // this thread's atomics are visible device-wide
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // loads first (independent: eight in flight per thread; more would cost every kernel that inlines this registers),
    // zeroing after
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        T sum = (T)0;
#pragma unroll 8
        for (int r = 0; r < reps; ++r) sum += __ldcg(acc + (size_t)r * n + i);
        host[i] = sum;
    }
    __syncthreads();                                     // (s_last is uniform over the CTA) every replica has been read
    for (int i = threadIdx.x; i < n * reps; i += blockDim.x) acc[i] = (T)0;
    if (threadIdx.x == 0) *ticket = 0u;
}
#endif
