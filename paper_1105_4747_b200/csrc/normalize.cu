// normalize.cu -- S4 and S5: mean-flux normalisation constant A and F = exp(-A tau).
//
// S4: one cooperative, persistent kernel runs the whole iteration on the device.  Each pass streams tau once
// (4 B / pixel, 128-bit loads), evaluates e = ex2(-A log2(e) tau) on the MUFU pipe and reduces the five tilted
// moments sum(tau^k e), k = 0..4 -- fp32 only inside one float4, double from the thread level up, warp
// shuffles, then five partials per block; the moments give a fifth-order step (root_iter.h), so the whole
// iteration takes 3-4 passes.  After a grid-wide barrier EVERY block reduces the same partials in the same
// order and applies the same scalar update (root_iter.h), so no second barrier or broadcast is needed and the
// result is bit-reproducible.  The host sees only the final (A, <F>, passes, status).
//
// A log2(e) is split into an fp32 hi/lo pair so that f(A) is not quantised at 6e-8 in A.
#include <cooperative_groups.h>

#include "lya_internal.h"
#include "pdf_bin.h"
#include "root_iter.h"

namespace cg = cooperative_groups;

namespace {

constexpr int RED_THREADS = 256;
constexpr int NORM_THREADS = 1024;   // normalize_kernel: ONE CTA per SM -- every CTA re-reads all per-CTA partials after
                                     // the grid barrier, and with 592 CTAs of 256 that gather (all CTAs hitting the same
                                     // L2 lines) cost 6-9 us per pass and the barrier 7-13 us; with 148 CTAs both are ~1 us
constexpr double LOG2E_D  = 1.4426950408889634074;

__device__ __forceinline__ float ex2_ftz(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

struct Trial { float c_hi, c_lo; };        // -A log2(e) = c_hi + c_lo

__host__ __device__ inline Trial make_trial(double a)
{
    double c = -a * LOG2E_D;
    Trial t;
    t.c_hi = (float)c;
    t.c_lo = (float)(c - (double)t.c_hi);
    return t;
}

__device__ __forceinline__ float flux_of(float tau, const Trial &t)
{
    return ex2_ftz(fmaf(tau, t.c_hi, tau * t.c_lo));
}

// sum over this thread's share of tau of (e, tau e) for K trials; grid-stride float4 body + scalar edges.
template <int K>
__device__ __forceinline__ void accumulate(const float *__restrict__ tau, size_t n, const Trial (&tr)[K],
                                           double (&s0)[K], double (&s1)[K])
{
#pragma unroll
    for (int k = 0; k < K; ++k) { s0[k] = 0.0; s1[k] = 0.0; }
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t gsz  = (size_t)gridDim.x * blockDim.x;
    size_t head = ((16 - ((uintptr_t)tau & 15)) & 15) >> 2;      // scalars before 16-byte alignment
    if (head > n) head = n;
    const size_t n4 = (n - head) >> 2;
    const float4 *t4 = reinterpret_cast<const float4 *>(tau + head);
#pragma unroll 2
    for (size_t i = gtid; i < n4; i += gsz) {
        const float4 t = __ldg(t4 + i);              // re-read every pass: let L2 keep what fits
#pragma unroll
        for (int k = 0; k < K; ++k) {
            float e0 = flux_of(t.x, tr[k]), e1 = flux_of(t.y, tr[k]);
            float e2 = flux_of(t.z, tr[k]), e3 = flux_of(t.w, tr[k]);
            s0[k] += (double)((e0 + e1) + (e2 + e3));
            s1[k] += (double)(fmaf(t.x, e0, t.y * e1) + fmaf(t.z, e2, t.w * e3));
        }
    }
    // edges: head scalars and the < 4 tail scalars
    const size_t tail0 = head + (n4 << 2);
    const size_t n_edge = head + (n - tail0);
    for (size_t e = gtid; e < n_edge; e += gsz) {
        const size_t i = e < head ? e : tail0 + (e - head);
        const float t = tau[i];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            float ex = flux_of(t, tr[k]);
            s0[k] += (double)ex;
            s1[k] += (double)(t * ex);
        }
    }
}

// the same stream, five tilted moments sum tau^k e, k = 0..4, for one trial (lya_root_step_moments).
// SUB: only the SUBSAMPLE of tau -- of the 16-byte aligned body, cut into chunks of 256 float4 (4 KiB), every
// `every`-th chunk; `items` = float4 in the subsample (the host counts them: sub_items()).  The subsample passes of
// normalize_kernel's nested iteration read 1 / every of the bytes.
constexpr int SUB_CHUNK_LOG2 = 8;

template <bool SUB>
__device__ __forceinline__ void accumulate_moments(const float *__restrict__ tau, size_t n, const Trial &tr, double (&s)[5],
                                                   size_t every = 1, size_t items = 0)
{
#pragma unroll
    for (int k = 0; k < 5; ++k) s[k] = 0.0;
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t gsz  = (size_t)gridDim.x * blockDim.x;
    size_t head = ((16 - ((uintptr_t)tau & 15)) & 15) >> 2;
    if (head > n) head = n;
    const size_t n4 = SUB ? items : (n - head) >> 2;
    const float4 *t4 = reinterpret_cast<const float4 *>(tau + head);
    // item -> float4 index: the identity, or chunk (x >> 8) of the subsample = chunk (x >> 8) * every of tau
    auto at = [&](size_t x) -> size_t {
        return SUB ? ((((x >> SUB_CHUNK_LOG2) * every) << SUB_CHUNK_LOG2) | (x & ((1u << SUB_CHUNK_LOG2) - 1))) : x;
    };
    // fp32 inside a group of up to four float4 (16 pixels), double above: one cvt + DADD per moment and group
    float q[5] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
    auto add4 = [&](const float4 &t) {
        float pa = flux_of(t.x, tr), pb = flux_of(t.y, tr), pc = flux_of(t.z, tr), pd = flux_of(t.w, tr);
        q[0] += (pa + pb) + (pc + pd);
#pragma unroll
        for (int k = 1; k < 5; ++k) {
            pa *= t.x; pb *= t.y; pc *= t.z; pd *= t.w;
            q[k] += (pa + pb) + (pc + pd);
        }
    };
    size_t i = gtid;
    for (; i + 3 * gsz < n4; i += 4 * gsz) {
        const float4 t0 = __ldg(t4 + at(i)), t1 = __ldg(t4 + at(i + gsz)), t2 = __ldg(t4 + at(i + 2 * gsz)),
                     t3 = __ldg(t4 + at(i + 3 * gsz));
#pragma unroll
        for (int k = 0; k < 5; ++k) q[k] = 0.0f;
        add4(t0); add4(t1); add4(t2); add4(t3);
#pragma unroll
        for (int k = 0; k < 5; ++k) s[k] += (double)q[k];
    }
    for (; i < n4; i += gsz) {
        const float4 t0 = __ldg(t4 + at(i));
#pragma unroll
        for (int k = 0; k < 5; ++k) q[k] = 0.0f;
        add4(t0);
#pragma unroll
        for (int k = 0; k < 5; ++k) s[k] += (double)q[k];
    }
    if (SUB) return;                                     // the unaligned edges are not part of the subsample
    const size_t tail0 = head + (n4 << 2);
    const size_t n_edge = head + (n - tail0);
    for (size_t e = gtid; e < n_edge; e += gsz) {
        const size_t i = e < head ? e : tail0 + (e - head);
        const float t = tau[i];
        float p = flux_of(t, tr);
#pragma unroll
        for (int k = 0; k < 5; ++k) { s[k] += (double)p; p *= t; }
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// block-wide sum of NV doubles per thread; result valid in every thread of warp 0 (and written by thread 0)
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double *sh /* [NV][warps] */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        v[k] = warp_sum(v[k]);
        if (lane == 0) sh[k * 32 + warp] = v[k];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double x = lane < nw ? sh[k * 32 + lane] : 0.0;
            v[k] = warp_sum(x);
        }
    }
    __syncthreads();
}

struct NormArgs {
    const float *tau;
    size_t       n;
    const double *rowm;        // per-sightline plain moments [n_rows][5] written by the tau kernels, or NULL
    size_t       n_rows;
    size_t       sub_every;    // > 1: nested iteration -- converge on every sub_every-th 4 KiB chunk of tau first
    size_t       sub_items;    // float4 in that subsample
    double       sub_tol;      // relative tolerance of the subsample's own root
    double       f_target, rel_tol;
    int          max_iter;
    double      *partials;     // [2][gridDim.x][5], gridDim.x <= SM count
    double      *result;       // [0] A, [1] <F> at A, [2] passes over all of tau (incl. the row-moment pass), [3] status,
                               // [4] subsample passes, [5] 1 if the A = 0 pass read the row moments
};

// The iteration, nested (reading C14):
//   ROWS  the A = 0 pass from the tau kernels' per-sightline moments, if the caller has them (40 B per sightline);
//   SUB   the whole root iteration on a SUBSAMPLE of tau (1 / sub_every of the bytes per pass) to sub_tol: the mean flux
//         of 1/32 of 1e9 pixels already fixes A to ~1e-4, and a heavy-tailed tau (max 1e6 x mean on the lognormal fields)
//         makes the first steps from A = 0 short, so this is where most passes go;
//   FULL  passes over ALL of tau from the subsample's root: the first one's fifth-order step lands within ~1e-15 of the
//         root of the FULL mean (|h| ~ 1e-4 A), its quartic-vs-cubic truncation estimate proves it, and the iteration
//         stops -- normally ONE pass over tau instead of 3-5.
// The result is the root of the mean over all pixels in every case: the subsample only supplies the starting point,
// the stopping rule is the full iteration's own.
constexpr int NORM_SUB_MAX = 12;                         // subsample passes before giving up on its convergence
enum { PH_ROWS = 0, PH_SUB = 1, PH_FULL = 2 };

__global__ void __launch_bounds__(NORM_THREADS, 1) normalize_kernel(const NormArgs a)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double sh[5 * 32];
    __shared__ lya_root_state st;
    __shared__ int s_phase, s_full, s_sub, s_finished;
    if (threadIdx.x == 0) {
        const bool sub = a.sub_every > 1 && a.sub_items > 0;
        s_phase = a.rowm ? PH_ROWS : (sub ? PH_SUB : PH_FULL);
        s_full = s_sub = s_finished = 0;
        if (s_phase == PH_SUB) lya_root_reset(&st, a.f_target, a.sub_tol, 4.0 * (double)a.sub_items);
        else                   lya_root_reset(&st, a.f_target, a.rel_tol, (double)a.n);
    }
    __syncthreads();

    for (int pass = 0;; ++pass) {
        const int phase = s_phase;
        const Trial tr = make_trial(st.a);
        double s[5];
        if (phase == PH_ROWS) {
            // A = 0: the tilted moments are the plain moments sum tau^k, which the tau kernels left per sightline
            // (40 B per sightline instead of 4 B per pixel); fixed thread -> row assignment, so bit-reproducible
#pragma unroll
            for (int k = 0; k < 5; ++k) s[k] = 0.0;
            for (size_t r = (size_t)blockIdx.x * blockDim.x + threadIdx.x; r < a.n_rows; r += (size_t)gridDim.x * blockDim.x)
#pragma unroll
                for (int k = 0; k < 5; ++k) s[k] += __ldcs(a.rowm + 5 * r + k);
        } else if (phase == PH_SUB) {
            accumulate_moments<true>(a.tau, a.n, tr, s, a.sub_every, a.sub_items);
        } else {
            accumulate_moments<false>(a.tau, a.n, tr, s);
        }
        block_sum<5>(s, sh);
        double *part = a.partials + (size_t)(pass & 1) * gridDim.x * 5;
        if (threadIdx.x == 0)
#pragma unroll
            for (int k = 0; k < 5; ++k) part[5 * blockIdx.x + k] = s[k];
        grid.sync();
        // every block: identical fixed-order reduction of all partials
        double t[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (unsigned b = threadIdx.x; b < gridDim.x; b += blockDim.x)
#pragma unroll
            for (int k = 0; k < 5; ++k) t[k] += __ldcg(part + 5 * b + k);
        block_sum<5>(t, sh);
        if (threadIdx.x == 0) {
            const double a_before = st.a;
            lya_root_step_moments(&st, t);
            const bool sub = a.sub_every > 1 && a.sub_items > 0;
            if (phase == PH_SUB) {
                s_sub += 1;
                if (st.done || s_sub >= NORM_SUB_MAX) {  // the subsample's root (or the best it got): start of the full passes
                    const double a0 = (st.status == LYA_OK && st.a > 0.0 && st.a < 1.0e30) ? st.a : a_before;
                    lya_root_reset(&st, a.f_target, a.rel_tol, (double)a.n);
                    st.a = a0;
                    s_phase = PH_FULL;
                }
            } else {
                s_full += 1;
                if (st.done) {
                    s_finished = 1;
                } else if (s_full >= a.max_iter) {
                    st.status = LYA_ENOCONV; st.done = 1; s_finished = 1;
                } else if (phase == PH_ROWS) {
                    s_phase = sub ? PH_SUB : PH_FULL;
                    if (sub) {                           // the subsample has its own pixel count and tolerance
                        const double a0 = st.a;
                        lya_root_reset(&st, a.f_target, a.sub_tol, 4.0 * (double)a.sub_items);
                        st.a = a0;
                    }
                }
            }
        }
        __syncthreads();
        if (s_finished) break;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        a.result[0] = st.a;
        a.result[1] = st.f_at_a;
        a.result[2] = (double)s_full;
        a.result[3] = (double)st.status;
        a.result[4] = (double)s_sub;
        a.result[5] = a.rowm ? 1.0 : 0.0;
    }
}

struct TrialSet { Trial t[LYA_MAX_TRIALS]; };

template <int K>
__global__ void __launch_bounds__(RED_THREADS) partial_sums_kernel(const float *__restrict__ tau, size_t n,
                                                                   const TrialSet ts, double *partials)
{
    __shared__ double sh[2 * K * 32];
    Trial tr[K];
#pragma unroll
    for (int k = 0; k < K; ++k) tr[k] = ts.t[k];
    double s0[K], s1[K], s[2 * K];
    accumulate<K>(tau, n, tr, s0, s1);
#pragma unroll
    for (int k = 0; k < K; ++k) { s[k] = s0[k]; s[K + k] = s1[k]; }
    block_sum<2 * K>(s, sh);
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < 2 * K; ++k) partials[(size_t)blockIdx.x * 2 * K + k] = s[k];
}

__global__ void __launch_bounds__(RED_THREADS) moment_sums_kernel(const float *__restrict__ tau, size_t n, const Trial tr,
                                                                 double *partials, size_t sub_every, size_t sub_items)
{
    __shared__ double sh[5 * 32];
    double s[5];
    if (sub_every > 1) accumulate_moments<true>(tau, n, tr, s, sub_every, sub_items);
    else               accumulate_moments<false>(tau, n, tr, s);
    block_sum<5>(s, sh);
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < 5; ++k) partials[(size_t)blockIdx.x * 5 + k] = s[k];
}

// per-sightline plain moments -> per-block partials (lya_row_moment_sums: the A = 0 pass of a sharded S4)
__global__ void __launch_bounds__(RED_THREADS) row_sums_kernel(const double *__restrict__ rowm, size_t n_rows, double *partials)
{
    __shared__ double sh[5 * 32];
    double s[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (size_t r = (size_t)blockIdx.x * blockDim.x + threadIdx.x; r < n_rows; r += (size_t)gridDim.x * blockDim.x)
#pragma unroll
        for (int k = 0; k < 5; ++k) s[k] += __ldcs(rowm + 5 * r + k);
    block_sum<5>(s, sh);
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < 5; ++k) partials[(size_t)blockIdx.x * 5 + k] = s[k];
}

// one block: fixed-order sum of the per-block partials -> out[0 .. nv)
__global__ void __launch_bounds__(RED_THREADS) finish_sums_kernel(const double *partials, int n_blocks, int nv,
                                                                  double *out)
{
    __shared__ double sh[32];
    for (int k = 0; k < nv; ++k) {
        double v[1] = {0.0};
        for (int b = threadIdx.x; b < n_blocks; b += blockDim.x) v[0] += partials[(size_t)b * nv + k];
        block_sum<1>(v, sh);
        if (threadIdx.x == 0) out[k] = v[0];
    }
}

__global__ void __launch_bounds__(256) flux_kernel(const float *tau, size_t n, Trial tr, float *flux)
{
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t gsz  = (size_t)gridDim.x * blockDim.x;
    size_t head = ((16 - ((uintptr_t)tau & 15)) & 15) >> 2;
    if (head > n) head = n;
    const bool vec = (((uintptr_t)(flux + head)) & 15) == 0;
    const size_t n4 = vec ? (n - head) >> 2 : 0;
    const float4 *t4 = reinterpret_cast<const float4 *>(tau + head);
    float4 *f4 = reinterpret_cast<float4 *>(flux + head);
#pragma unroll 2
    for (size_t i = gtid; i < n4; i += gsz) {
        const float4 t = __ldcs(t4 + i);
        float4 f;
        f.x = flux_of(t.x, tr); f.y = flux_of(t.y, tr); f.z = flux_of(t.z, tr); f.w = flux_of(t.w, tr);
        __stcs(f4 + i, f);
    }
    const size_t tail0 = head + (n4 << 2);
    const size_t n_edge = head + (n - tail0);
    for (size_t e = gtid; e < n_edge; e += gsz) {
        const size_t i = e < head ? e : tail0 + (e - head);
        flux[i] = flux_of(tau[i], tr);
    }
}

// S5 and the flux PDF in one pass: F is written as by flux_kernel and binned as by
// flux_pdf_kernel (observe.cu) -- private per-thread histograms hist[bin][thread] in shared memory, the bin
// decision by pdf_bin.h's exact thresholds (reading O4) -- so the counts are bit-identical to lya_flux followed
// by lya_flux_pdf, with 8 B instead of 12 B of traffic per pixel.
constexpr int FPDF_THREADS = 128;

__global__ void __launch_bounds__(FPDF_THREADS) flux_pdf_fused_kernel(const float *tau, size_t n, Trial tr, float *flux,
                                                                      const __grid_constant__ PdfEdges edges,
                                                                      unsigned long long *counts, unsigned long long *host,
                                                                      unsigned int *ticket, int reps)
{
    extern __shared__ unsigned int hist[];               // [n_bins][FPDF_THREADS], then n_bins + 1 thresholds
    const int n_bins = edges.n_bins;
    float *s_thr = reinterpret_cast<float *>(hist + n_bins * FPDF_THREADS);
    for (int t = threadIdx.x; t < n_bins * FPDF_THREADS; t += FPDF_THREADS) hist[t] = 0u;
    for (int t = threadIdx.x; t <= n_bins; t += FPDF_THREADS) s_thr[t] = edges.thr[t];
    __syncthreads();
    unsigned int *mine = hist + threadIdx.x;
    const float f_lo = edges.f_lo, inv_width = edges.inv_width, eps = edges.eps, ome = edges.one_minus_eps;
    auto bin = [&](float f) { atomicAdd(mine + lya_pdf_bin(f, s_thr, n_bins, f_lo, inv_width, eps, ome) * FPDF_THREADS, 1u); };
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t gsz  = (size_t)gridDim.x * blockDim.x;
    size_t head = ((16 - ((uintptr_t)tau & 15)) & 15) >> 2;
    if (head > n) head = n;
    const bool vec = (((uintptr_t)(flux + head)) & 15) == 0;
    const size_t n4 = vec ? (n - head) >> 2 : 0;
    const float4 *t4 = reinterpret_cast<const float4 *>(tau + head);
    float4 *f4 = reinterpret_cast<float4 *>(flux + head);
#pragma unroll 2
    for (size_t i = gtid; i < n4; i += gsz) {
        const float4 t = __ldcs(t4 + i);
        float4 f;
        f.x = flux_of(t.x, tr); f.y = flux_of(t.y, tr); f.z = flux_of(t.z, tr); f.w = flux_of(t.w, tr);
        __stcs(f4 + i, f);
        bin(f.x); bin(f.y); bin(f.z); bin(f.w);
    }
    const size_t tail0 = head + (n4 << 2);
    const size_t n_edge = head + (n - tail0);
    for (size_t e = gtid; e < n_edge; e += gsz) {
        const size_t i = e < head ? e : tail0 + (e - head);
        const float f = flux_of(tau[i], tr);
        flux[i] = f;
        bin(f);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int b = warp; b < n_bins; b += FPDF_THREADS / 32) {
        unsigned int sum = 0;
        for (int t = lane; t < FPDF_THREADS; t += 32) sum += hist[b * FPDF_THREADS + t];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0 && sum) atomicAdd(counts + (blockIdx.x % reps) * n_bins + b, (unsigned long long)sum);
    }
    lya_publish_last_cta(counts, n_bins, host, ticket, reps);
}

// float4 in the subsample "every `every`-th chunk of 256 float4 of the aligned body of tau" (0: no subsample)
size_t sub_items_of(const float *tau, size_t n, size_t every)
{
    size_t head = ((16 - ((uintptr_t)tau & 15)) & 15) >> 2;
    if (head > n) head = n;
    const size_t n4 = (n - head) >> 2;
    if (every <= 1 || n4 == 0) return 0;
    const size_t n_ch = (n4 + 255) >> SUB_CHUNK_LOG2, k_sub = (n_ch + every - 1) / every;
    const size_t last = ((k_sub - 1) * every) << SUB_CHUNK_LOG2;          // first float4 of the last subsample chunk
    const size_t len_last = n4 - last < 256 ? n4 - last : 256;
    return ((k_sub - 1) << SUB_CHUNK_LOG2) + len_last;
}

int red_grid(lya_ctx *ctx, size_t n, int per_sm)
{
    size_t want = (n / 4 + RED_THREADS - 1) / RED_THREADS;
    if (want < 1) want = 1;
    size_t cap = (size_t)ctx->sm_count * per_sm;
    if (cap > LYA_MAX_RED_BLOCKS) cap = LYA_MAX_RED_BLOCKS;
    return (int)(want < cap ? want : cap);
}

}  // namespace

lya_status lya_run_normalize(lya_ctx *ctx, const float *tau, size_t n, const double *rowm, size_t n_rows,
                             double f_target, double rel_tol, int max_iter, double *a_out, double *f_out, int *iters)
{
    if (!ctx->coop_ok) return lya_fail(ctx, LYA_ECUDA, "device does not support cooperative launch");
    if (ctx->norm_occ == 0) {                              // asked once per ctx: the answer cannot change
        int per_sm = 0;
        LYA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, normalize_kernel, NORM_THREADS, 0));
        ctx->norm_occ = per_sm < 1 ? -1 : per_sm;
    }
    if (ctx->norm_occ < 1) return lya_fail(ctx, LYA_ECUDA, "normalize_kernel: zero occupancy");
    // the four result doubles go straight to the pinned host mirror (mapped under UVA): no copy to enqueue
    // nested iteration for grids beyond norm_sub_min pixels (lya_set_normalize_subsample); the subsample's own root is
    // only a starting point, so its tolerance is loose: its statistical distance from the full root is ~1e-4 anyway
    const size_t every = (ctx->norm_sub_every > 1 && n >= ctx->norm_sub_min) ? ctx->norm_sub_every : 1;
    const size_t items = sub_items_of(tau, n, every);
    NormArgs a{tau, n, rowm, n_rows, items ? every : 1, items, 1.0e-3 > rel_tol ? 1.0e-3 : rel_tol,
               f_target, rel_tol, max_iter, ctx->d_partials, ctx->h_pinned};
    size_t want = (n / 4 + NORM_THREADS - 1) / NORM_THREADS;           // at least one float4 per thread
    if (want < 1) want = 1;
    const int grid = (int)(want < (size_t)ctx->sm_count ? want : (size_t)ctx->sm_count);
    void *args[] = {(void *)&a};
    LYA_CUDA(ctx, cudaLaunchCooperativeKernel((void *)normalize_kernel, dim3(grid), dim3(NORM_THREADS), args, 0,
                                              ctx->stream));
    ctx->launches++;
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (a_out) *a_out = ctx->h_pinned[0];
    if (f_out) *f_out = ctx->h_pinned[1];
    if (iters) *iters = (int)ctx->h_pinned[2];
    ctx->norm_stats[0] = ctx->h_pinned[2];                 // lya_last_normalize_stats
    ctx->norm_stats[1] = ctx->h_pinned[4];
    ctx->norm_stats[2] = ctx->h_pinned[5];
    ctx->norm_stats[3] = 4.0 * (double)items;
    lya_status st = (lya_status)(int)ctx->h_pinned[3];
    if (st == LYA_ENOROOT) return lya_fail(ctx, st, "lya_normalize_mean_flux: no A > 0 reaches f_target");
    if (st == LYA_ENOCONV) return lya_fail(ctx, st, "lya_normalize_mean_flux: max_iter reached");
    return st;
}

lya_status lya_run_partial_sums(lya_ctx *ctx, const float *tau, size_t n, const double *a_trial, int k,
                                double *sums, double *dsums)
{
    TrialSet ts;
    for (int i = 0; i < LYA_MAX_TRIALS; ++i) ts.t[i] = make_trial(i < k ? a_trial[i] : 0.0);
    int grid = red_grid(ctx, n, 8);
    double *part = ctx->d_partials;
    switch (k) {
#define LYA_PS_CASE(K) case K: partial_sums_kernel<K><<<grid, RED_THREADS, 0, ctx->stream>>>(tau, n, ts, part); break;
        LYA_PS_CASE(1) LYA_PS_CASE(2) LYA_PS_CASE(3) LYA_PS_CASE(4)
        LYA_PS_CASE(5) LYA_PS_CASE(6) LYA_PS_CASE(7) LYA_PS_CASE(8)
#undef LYA_PS_CASE
        default: return lya_fail(ctx, LYA_EINVAL, "lya_flux_partial_sums: k must be 1..8");
    }
    finish_sums_kernel<<<1, RED_THREADS, 0, ctx->stream>>>(part, grid, 2 * k, ctx->h_pinned);   // mapped pinned memory
    ctx->launches += 2;
    LYA_CUDA(ctx, cudaGetLastError());
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < k; ++i) {
        sums[i] = ctx->h_pinned[i];
        if (dsums) dsums[i] = ctx->h_pinned[k + i];
    }
    return LYA_OK;
}

lya_status lya_launch_flux(lya_ctx *ctx, const float *tau, size_t n, double a, float *flux)
{
    size_t want = (n / 4 + 255) / 256;
    if (want < 1) want = 1;
    // about 12 float4 per thread, never fewer CTAs than 8 per SM: measured best on 256^3 (8 CTAs/SM), 512^3
    // (64-128 per SM: 99 % of the copy bandwidth) and 1024^3 (256-1024 per SM: 99-101 %; 8 per SM gave 92 %)
    size_t cap = (size_t)ctx->sm_count * 8;
    if (cap < want / 12) cap = want / 12;
    int grid = (int)(want < cap ? want : cap);
    flux_kernel<<<grid, 256, 0, ctx->stream>>>(tau, n, make_trial(a), flux);
    ctx->launches++;
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}

lya_status lya_run_moment_sums(lya_ctx *ctx, const float *tau, size_t n, double a_trial, size_t every, double *sums5,
                               uint64_t *n_sub)
{
    const size_t items = sub_items_of(tau, n, every);
    if (n_sub) *n_sub = every > 1 ? 4 * items : n;
    if (every > 1 && items == 0) {                         // nothing in the subsample (fewer than 4 aligned pixels)
        for (int i = 0; i < 5; ++i) sums5[i] = 0.0;
        return LYA_OK;
    }
    const int grid = red_grid(ctx, every > 1 ? 4 * items : n, 8);
    moment_sums_kernel<<<grid, RED_THREADS, 0, ctx->stream>>>(tau, n, make_trial(a_trial), ctx->d_partials, every, items);
    finish_sums_kernel<<<1, RED_THREADS, 0, ctx->stream>>>(ctx->d_partials, grid, 5, ctx->h_pinned);   // mapped pinned memory
    ctx->launches += 2;
    LYA_CUDA(ctx, cudaGetLastError());
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < 5; ++i) sums5[i] = ctx->h_pinned[i];
    return LYA_OK;
}

lya_status lya_run_row_moment_sums(lya_ctx *ctx, const double *rowm, size_t n_rows, double *sums5)
{
    size_t want = (n_rows + RED_THREADS - 1) / RED_THREADS, cap = (size_t)ctx->sm_count * 4;
    const int grid = (int)(want < cap ? want : cap);
    row_sums_kernel<<<grid, RED_THREADS, 0, ctx->stream>>>(rowm, n_rows, ctx->d_partials);
    finish_sums_kernel<<<1, RED_THREADS, 0, ctx->stream>>>(ctx->d_partials, grid, 5, ctx->h_pinned);   // mapped pinned memory
    ctx->launches += 2;
    LYA_CUDA(ctx, cudaGetLastError());
    LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < 5; ++i) sums5[i] = ctx->h_pinned[i];
    return LYA_OK;
}

lya_status lya_run_flux_with_pdf(lya_ctx *ctx, const float *tau, size_t n, double a, float *flux, int n_bins,
                                 double f_lo, double width, uint64_t *counts, double *pdf)
{
    unsigned long long *d_counts = reinterpret_cast<unsigned long long *>(ctx->d_stats);
    unsigned long long *host = reinterpret_cast<unsigned long long *>(ctx->h_pinned + LYA_PINNED_STATS);
    if (n > 0) {
        PdfEdges edges;
        lya_pdf_edges(n_bins, f_lo, width, &edges);
        const size_t smem = (size_t)n_bins * FPDF_THREADS * sizeof(unsigned int) + (size_t)(n_bins + 1) * sizeof(float);
        int per_sm = 0;
        lya_status st = lya_kernel_occupancy(ctx, (const void *)flux_pdf_fused_kernel, FPDF_THREADS, smem, &per_sm);
        if (st != LYA_OK) return st;
        if (per_sm < 1) return lya_fail(ctx, LYA_EINVAL, "lya_flux_with_pdf: too many bins for shared memory");
        size_t want = (n / 4 + FPDF_THREADS - 1) / FPDF_THREADS;
        if (want < 1) want = 1;
        const size_t cap = (size_t)ctx->sm_count * per_sm;
        st = lya_stats_begin(ctx, n_bins);
        if (st != LYA_OK) return st;
        // the last CTA to finish writes the totals straight to the pinned mirror and re-zeroes the device counters
        flux_pdf_fused_kernel<<<(int)(want < cap ? want : cap), FPDF_THREADS, smem, ctx->stream>>>(
            tau, n, make_trial(a), flux, edges, d_counts, host, ctx->d_sched + 4, lya_stats_replicas(n_bins, n, 16));
        ctx->launches++;
        st = lya_stats_end(ctx);
        if (st != LYA_OK) return st;
    } else {
        for (int b = 0; b < n_bins; ++b) host[b] = 0;
    }
    for (int b = 0; b < n_bins; ++b) {
        if (counts) counts[b] = host[b];
        if (pdf) pdf[b] = n ? (double)host[b] / ((double)n * width) : 0.0;
    }
    return LYA_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// lya_flux_moment_sums_static: the five tilted moments of S4 for callers that may not allocate -- code
// under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  The per-block partials, which every other
// reduction of this file keeps in ctx->d_partials (cudaMalloc'ed by lya_create), live in the file-scope array below:
// LYA_STATIC_MAX_BLOCKS x 5 doubles = 655,360 B of device memory held by every GPU that loads the library, until exit.
// Block b owns the FIXED pixel range [b, b + 1) * LYA_STATIC_PIX_PER_BLOCK, so the result does not depend on the SM
// count, and the largest input is LYA_STATIC_MAX_PIX = 16384 * 65536 = 2^30 pixels (config 4's whole grid).
// Every partial the finishing kernel reads is written by the same call first: nothing has to start at zero.  All calls
// on a device share the array: calls that overlap on the GPU (different streams, no ordering) race.
// ---------------------------------------------------------------------------------------------------------------------
#define LYA_STATIC_PIX_PER_BLOCK 65536
#define LYA_STATIC_MAX_BLOCKS    16384

static __device__ __align__(256) double lya_static_partials[(size_t)LYA_STATIC_MAX_BLOCKS * 5];

namespace {

__global__ void __launch_bounds__(RED_THREADS) static_moment_sums_kernel(const float *__restrict__ tau, size_t n, const Trial tr,
                                                                        double *partials)
{
    __shared__ double sh[5 * 32];
    const size_t lo = (size_t)blockIdx.x * LYA_STATIC_PIX_PER_BLOCK;
    const size_t hi = lo + LYA_STATIC_PIX_PER_BLOCK < n ? lo + LYA_STATIC_PIX_PER_BLOCK : n;
    double s[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    float q[5];
    auto add1 = [&](float t) {
        float p = flux_of(t, tr);
#pragma unroll
        for (int k = 0; k < 5; ++k) { q[k] += p; p *= t; }
    };
    auto flush = [&]() {                                 // fp32 inside a group of up to 16 pixels, double above
#pragma unroll
        for (int k = 0; k < 5; ++k) { s[k] += (double)q[k]; q[k] = 0.0f; }
    };
#pragma unroll
    for (int k = 0; k < 5; ++k) q[k] = 0.0f;
    if (((uintptr_t)tau & 15) == 0) {                    // lo is a multiple of 4 pixels: 128-bit loads
        const float4 *t4 = reinterpret_cast<const float4 *>(tau + lo);
        const size_t n4 = (hi - lo) >> 2;
        size_t i = threadIdx.x;
        for (; i + 3 * RED_THREADS < n4; i += 4 * RED_THREADS) {
            const float4 t0 = __ldg(t4 + i), t1 = __ldg(t4 + i + RED_THREADS), t2 = __ldg(t4 + i + 2 * RED_THREADS),
                         t3 = __ldg(t4 + i + 3 * RED_THREADS);
            add1(t0.x); add1(t0.y); add1(t0.z); add1(t0.w);
            add1(t1.x); add1(t1.y); add1(t1.z); add1(t1.w);
            add1(t2.x); add1(t2.y); add1(t2.z); add1(t2.w);
            add1(t3.x); add1(t3.y); add1(t3.z); add1(t3.w);
            flush();
        }
        for (; i < n4; i += RED_THREADS) {
            const float4 t0 = __ldg(t4 + i);
            add1(t0.x); add1(t0.y); add1(t0.z); add1(t0.w);
            flush();
        }
        for (size_t e = lo + (n4 << 2) + threadIdx.x; e < hi; e += RED_THREADS) { add1(tau[e]); flush(); }
    } else {
        for (size_t e = lo + threadIdx.x; e < hi; e += RED_THREADS) { add1(tau[e]); flush(); }
    }
    block_sum<5>(s, sh);
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < 5; ++k) partials[(size_t)blockIdx.x * 5 + k] = s[k];
}

// device address of lya_static_partials per device (the array's name is only a host-side stand-in in host code)
constexpr int STATIC_MAX_DEVICES = 64;
double *g_static_addr[STATIC_MAX_DEVICES];

}  // namespace

extern "C" lya_status lya_flux_moment_sums_static(lya_ctx *ctx, const float *tau, size_t n_pix, double a_trial, double *sums5)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if ((n_pix > 0 && (!tau || ((uintptr_t)tau & 3))) || !sums5 || ((uintptr_t)sums5 & 7))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums_static: null or misaligned pointer");
    if (!(a_trial >= 0.0) || !(a_trial < 1.0e30))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums_static: trial A must be finite and >= 0");
    if (n_pix > (size_t)LYA_STATIC_MAX_PIX)
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums_static: n_pix exceeds LYA_STATIC_MAX_PIX (2^30 pixels: the static "
                                         "scratch holds 16384 blocks of 65536 pixels); split the input or use lya_flux_moment_sums");
    if (ctx->device < 0 || ctx->device >= STATIC_MAX_DEVICES)
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_moment_sums_static: device index beyond 63");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    double *part = g_static_addr[ctx->device];
    if (!part) {                                         // set-up, once per device, with that device current
        LYA_CUDA(ctx, cudaGetSymbolAddress((void **)&part, lya_static_partials));
        g_static_addr[ctx->device] = part;               // (two threads racing here store the same address)
    }
    const int grid = (int)((n_pix + LYA_STATIC_PIX_PER_BLOCK - 1) / LYA_STATIC_PIX_PER_BLOCK);
    if (grid > 0) static_moment_sums_kernel<<<grid, RED_THREADS, 0, ctx->stream>>>(tau, n_pix, make_trial(a_trial), part);
    finish_sums_kernel<<<1, RED_THREADS, 0, ctx->stream>>>(part, grid, 5, sums5);        // n_pix == 0: five zeros
    ctx->launches += grid > 0 ? 2 : 1;
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}
