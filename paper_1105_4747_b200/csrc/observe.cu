// observe.cu -- the paper's instrument model on rows of transmitted flux:
// circular Gaussian convolution in velocity, flux-conserving resampling onto wider (or narrower) bins,
// additive noise N(0,1)/(S/N) from caller-supplied unit draws.  DESIGN.md readings O1-O3.
//
//   Fc(i)  = sum_k g(k) F(i-k),  g(k) ~ exp(-(k dv)^2 / 2 sigma^2) over the nearest periodic image,
//            normalised by the discrete sum; taps beyond 5 sigma are dropped (5.7e-7 of the kernel: |error| <= 5.7e-7)
//   Fb(m)  = (1/B) integral over [m B, (m+1) B) of the piecewise-constant Fc       (B = bin / dv in pixels)
//   out    = Fb + unit_noise / snr
//
// HBM-bound: 4 B read per pixel, 4 (+4 noise) B per output bin.  One CTA stages one row (with its periodic
// halo) in shared memory; the convolution is register-tiled -- a thread owns 4 consecutive outputs, walks the
// inputs with one conflict-free LDS.128 per 4 inputs and two broadcast LDS.128 of taps, 16 FFMA per step --
// so even a 60-tap kernel stays near the memory roofline; the rebinning reads the convolved row from shared
// memory with bin edges in double.
#include <math.h>

#include "lya_internal.h"
#include "pdf_bin.h"

namespace {

struct ObsArgs {
    const float *flux, *noise, *taps;     // taps: device, wp[0 .. L+10], wp[t+3] = g(Kr - t), zero padded
    float       *out;
    size_t       n_rows;
    int          n, n4;                   // pixels per row; rounded up to a multiple of 4
    int          Kl, Kr, KO, L;           // taps on either side, left halo KO >= Kr; L = KO + Kl (< 0: no convolution)
    int          nb;                      // output bins per row
    int          rebin;                   // 0: out has n pixels, no resampling
    unsigned long long bin_fx;            // B = bin / dv [pixels] in 32.32 fixed point
    float        inv_bin_f;               // 1 / B
    float        inv_snr;                 // 0: no noise
    const int4  *bins;                    // lean kernel: per output bin {i0, i1, bits(w_first), bits(w_last)}, or
    int          bins3;                   // (bins3, bins <= 2 pixels wide) {i0, bits(w0), bits(w1), bits(w2)}
};

// A CTA works on batches of D rows.  NV = float4 loads per thread and row (n4 <= 4 * NV * blockDim.x).  The
// NEXT batch is fetched into registers, and the CURRENT batch's noise draws are, before the current batch is
// convolved, so D * NV 128-bit loads per thread are in flight during all the arithmetic (HBM latency x
// bandwidth needs ~10 MB in flight on B200).
// s_in[d][h] = F_d[(h - KO) mod n], h < n + L, with KO >= Kr the left halo (a multiple of 4 in FAST mode, so
// that a thread's four pixels go to shared memory as one aligned STS.128 and the halo pixels -- at most one
// per thread and row -- are fetched separately); taps wp[t + 3] = g(KO - t), zero where KO - t is outside
// [-Kl, Kr].
constexpr int OBS_NBR = 4;                               // noise draws per thread and row held in registers

template <int NV, int D, bool FAST>
__global__ void __launch_bounds__(256) observe_rows_kernel(const ObsArgs a)
{
    extern __shared__ __align__(16) float sm[];
    const int n = a.n, n4 = a.n4;
    const int halo = a.L >= 0 ? a.L : 0;
    const int in_len = n4 + ((halo + 3) & ~3) + 8;       // staged inputs incl. halo and zero padding
    float *s_in = sm;                                    // [D][in_len]
    float *s_c  = sm + D * in_len;                       // [D][n4] convolved rows
    float *s_w  = s_c + D * n4;                          // taps, L + 11 floats rounded up to 4
    const int w_len = ((halo + 11) + 3) & ~3;
    const bool conv = a.L >= 0;
    const int T = blockDim.x, tid = threadIdx.x;

    if (conv)
        for (int t = tid; t < w_len; t += T) s_w[t] = t < halo + 11 ? a.taps[t] : 0.0f;
    for (int h = tid; h < D * in_len; h += T) s_in[h] = 0.0f;       // zero padding beyond n + halo
    if (!conv)
        for (int h = tid; h < D * n4; h += T) s_c[h] = 0.0f;

    float4 reg[D][NV];
    float hreg[D];                                       // FAST: this thread's halo pixel (tid < L)
    float nzr[D][OBS_NBR];
    auto fetch = [&](size_t row0) {                      // rows row0 .. row0+D-1 -> registers
#pragma unroll
        for (int d = 0; d < D; ++d) {
            const size_t row = row0 + d;
            hreg[d] = 0.0f;
#pragma unroll
            for (int q = 0; q < NV; ++q) reg[d][q] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (row >= a.n_rows) continue;
            const float *src = a.flux + row * (size_t)n;
#pragma unroll
            for (int q = 0; q < NV; ++q) {
                const int p = 4 * (tid + q * T);
                if (p < n) {
                    if (FAST) reg[d][q] = __ldcs(reinterpret_cast<const float4 *>(src + p));
                    else {
                        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                        v.x = __ldcs(src + p);
                        if (p + 1 < n) v.y = __ldcs(src + p + 1);
                        if (p + 2 < n) v.z = __ldcs(src + p + 2);
                        if (p + 3 < n) v.w = __ldcs(src + p + 3);
                        reg[d][q] = v;
                    }
                }
            }
            if (FAST && conv && tid < a.L)               // left halo h < KO: F[n - KO + h]; right: F[h - KO]
                hreg[d] = __ldg(src + (tid < a.KO ? n - a.KO + tid : tid - a.KO));
        }
    };
    auto put = [&](float *si, float *sc, int i, float v) {   // generic: pixel i -> body and halo copies
        if (i >= n) return;
        if (!conv) { sc[i] = v; return; }
        si[i + a.KO] = v;
        if (i < a.Kl) si[n + a.KO + i] = v;
        if (i >= n - a.KO) si[i - (n - a.KO)] = v;
    };

    size_t row0 = (size_t)blockIdx.x * D;
    if (row0 < a.n_rows) fetch(row0);
    for (; row0 < a.n_rows; row0 += (size_t)gridDim.x * D) {
        __syncthreads();                                 // previous batch's s_in / s_c consumed
#pragma unroll
        for (int d = 0; d < D; ++d) {
            float *si = s_in + d * in_len, *sc = s_c + d * n4;
#pragma unroll
            for (int q = 0; q < NV; ++q) {
                const int p = 4 * (tid + q * T);
                if (FAST) {
                    if (p < n) *reinterpret_cast<float4 *>((conv ? si + a.KO : sc) + p) = reg[d][q];
                } else {
                    put(si, sc, p, reg[d][q].x); put(si, sc, p + 1, reg[d][q].y);
                    put(si, sc, p + 2, reg[d][q].z); put(si, sc, p + 3, reg[d][q].w);
                }
            }
            if (FAST && conv && tid < a.L) si[tid < a.KO ? tid : n + tid] = hreg[d];
        }
        // loads issued now stay in flight during the convolution: the next batch, and this batch's noise
        if (row0 + (size_t)gridDim.x * D < a.n_rows) fetch(row0 + (size_t)gridDim.x * D);
        if (a.noise) {
#pragma unroll
            for (int d = 0; d < D; ++d)
#pragma unroll
                for (int k = 0; k < OBS_NBR; ++k) {
                    const int m = tid + k * T;
                    nzr[d][k] = (row0 + d < a.n_rows && m < a.nb) ? __ldcs(a.noise + (row0 + d) * (size_t)a.nb + m) : 0.0f;
                }
        }
        __syncthreads();
        if (conv) {
            for (int item = tid; item < D * (n4 >> 2); item += T) {
                const int d = item / (n4 >> 2), i0 = 4 * (item - d * (n4 >> 2));
                const float *si = s_in + d * in_len + i0;
                float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f, acc3 = 0.f;
                // out(i0 + r) = sum_t wt[t] s_in[i0 + r + t]; with u = r + t the weight of input u is wp[u - r + 3]
#pragma unroll 2
                for (int u = 0; u <= a.L + 3; u += 4) {
                    const float4 x  = *reinterpret_cast<const float4 *>(si + u);
                    const float4 wa = *reinterpret_cast<const float4 *>(s_w + u);       // wp[u .. u+3]
                    const float4 wb = *reinterpret_cast<const float4 *>(s_w + u + 4);   // wp[u+4 .. u+7]
                    // input c (= x.c) and output r use wp[u + c - r + 3]
                    acc0 = fmaf(wa.w, x.x, acc0); acc0 = fmaf(wb.x, x.y, acc0); acc0 = fmaf(wb.y, x.z, acc0); acc0 = fmaf(wb.z, x.w, acc0);
                    acc1 = fmaf(wa.z, x.x, acc1); acc1 = fmaf(wa.w, x.y, acc1); acc1 = fmaf(wb.x, x.z, acc1); acc1 = fmaf(wb.y, x.w, acc1);
                    acc2 = fmaf(wa.y, x.x, acc2); acc2 = fmaf(wa.z, x.y, acc2); acc2 = fmaf(wa.w, x.z, acc2); acc2 = fmaf(wb.x, x.w, acc2);
                    acc3 = fmaf(wa.x, x.x, acc3); acc3 = fmaf(wa.y, x.y, acc3); acc3 = fmaf(wa.z, x.z, acc3); acc3 = fmaf(wa.w, x.w, acc3);
                }
                *reinterpret_cast<float4 *>(s_c + d * n4 + i0) = make_float4(acc0, acc1, acc2, acc3);
            }
            __syncthreads();
        }

#pragma unroll
        for (int d = 0; d < D; ++d) {
            if (row0 + d >= a.n_rows) break;
            const float *sc = s_c + d * n4;
            float *dst = a.out + (row0 + d) * (size_t)a.nb;
            int k = 0;
            for (int m = tid; m < a.nb; m += T, ++k) {
                float v;
                if (a.rebin) {
                    // bin [lo, hi) in pixel units as 32.32 fixed point (bin_fx = B 2^32 rounded: the edges are
                    // off by < m 2^-33 pixels): partial first and last pixel, whole pixels in between
                    const unsigned long long lo = (unsigned long long)m * a.bin_fx, hi1 = lo + a.bin_fx - 1ull;
                    const int i0 = (int)(lo >> 32);
                    int i1 = (int)(hi1 >> 32);                                   // ceil(hi) - 1
                    if (i1 > n - 1) i1 = n - 1;
                    const float f_lo = (float)(unsigned int)lo * 2.3283064365386963e-10f;           // frac(lo)
                    const float f_hi = ((float)(unsigned int)hi1 + 1.0f) * 2.3283064365386963e-10f; // hi - i1
                    float acc;
                    if (i1 <= i0) {
                        acc = (f_hi - f_lo) * sc[i0];
                    } else {
                        acc = (1.0f - f_lo) * sc[i0];
#pragma unroll 1
                        for (int i = i0 + 1; i < i1; ++i) acc += sc[i];
                        acc = fmaf(f_hi, sc[i1], acc);
                    }
                    v = acc * a.inv_bin_f;
                } else {
                    v = sc[m];
                }
                if (a.noise) {
                    float z = 0.0f;
                    if (k < OBS_NBR) {
#pragma unroll
                        for (int kk = 0; kk < OBS_NBR; ++kk) if (kk == k) z = nzr[d][kk];
                    } else {
                        z = __ldcs(a.noise + (row0 + d) * (size_t)a.nb + m);
                    }
                    v = fmaf(z, a.inv_snr, v);
                }
                __stcs(dst + m, v);
            }
        }
    }
}

// ---- the lean kernel: the common case (16-byte aligned rows, n % 4 == 0, at most LT + 1 <= 125 taps incl. the
// alignment padding, at most four float4 per thread and row: rows up to 4096 pixels).  Same data flow as above, but the instruction count per
// pixel is roughly halved: the taps arrive as a __grid_constant__ kernel parameter, so with the tap loop fully
// unrolled every FFMA takes its weight straight from the constant bank and every LDS.128 of inputs has an
// immediate offset (17 instructions per 16 FFMA instead of 26); and the bin geometry of the rebinning, which
// is the same for every row, comes from a table built once on the host (bins[m] = first pixel, last pixel,
// weight of the first and of the last pixel) and kept in shared memory.
// packed FP32 pairs (sm_100a: fma.rn.f32x2 = FFMA2, one issue slot for two fused multiply-adds)
constexpr int OBS_PACKED_LT = 40;                        // beyond this the weight pairs no longer fit in registers
__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float sum2(unsigned long long v)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
    return lo + hi;
}

struct __align__(16) ObsTaps {
    float wp[136];                                       // wp[t + 3] = g(KO - t); zero outside the real taps
    float wq[136];                                       // wq[k] = wp[k + 1]: every (wp[k], wp[k + 1]) pair is 8-byte aligned in one of the two
};
// (wp[k], wp[k + 1]) as one 64-bit operand, k known at compile time
#define OBS_WPAIR(k) (((k) & 1) ? pack2(tp.wq[(k) - 1], tp.wq[(k)]) : pack2(tp.wp[(k)], tp.wp[(k) + 1]))

template <int LT, int NV>                                // LT >= L, multiple of 4: taps t = 0 .. LT; NV float4 per thread
__global__ void __launch_bounds__(256) observe_rows_lean_kernel(const ObsArgs a, const __grid_constant__ ObsTaps tp)
{
    extern __shared__ __align__(16) float sm[];
    const int n = a.n, T = blockDim.x, tid = threadIdx.x;
    const int in_len = n + LT + 8;
    float *s_in = sm;                                    // s_in[h] = F[(h - KO) mod n], zero beyond n + L
    float *s_c  = sm + in_len;                           // convolved row, n floats (+ 4 zeros for the 3-tap rebin)
    int4  *s_b  = reinterpret_cast<int4 *>(s_c + n + 4); // bin table, nb entries (rebin only)
    for (int h = tid; h < in_len; h += T) s_in[h] = 0.0f;
    if (tid < 4) s_c[n + tid] = 0.0f;
    if (a.rebin)
        for (int m = tid; m < a.nb; m += T) s_b[m] = a.bins[m];

    float4 reg[NV];                                      // this thread's pixels 4 (tid + q T) .. + 3
    float hreg = 0.0f, nzr[OBS_NBR];
    // everything that does not depend on the row is computed once: offsets are 32-bit, the row pointers advance by a
    // constant stride (the per-row 64-bit multiplies and the lambdas' re-derived addresses were a third of the
    // instructions: profiles/r2_ncu_next_rows.md)
    const int nb = a.nb;
    const bool has_halo = tid < a.L;
    const int hsrc = tid < a.KO ? n - a.KO + tid : tid - a.KO;       // this thread's halo pixel and where it goes
    const int hdst = tid < a.KO ? tid : n + tid;
    const size_t row_step = gridDim.x;
    const float *src = a.flux + (size_t)blockIdx.x * n;               // row being fetched
    const float *nz  = a.noise ? a.noise + (size_t)blockIdx.x * nb : nullptr;   // row being written
    float *dst = a.out + (size_t)blockIdx.x * nb;
    const size_t src_step = row_step * n, out_step = row_step * nb;
    auto fetch = [&]() {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const int p = 4 * (tid + q * T);
            reg[q] = p < n ? __ldcs(reinterpret_cast<const float4 *>(src + p)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (has_halo) hreg = __ldg(src + hsrc);
        src += src_step;
    };
    size_t row = blockIdx.x;
    if (row < a.n_rows) fetch();
    for (; row < a.n_rows; row += row_step) {
        __syncthreads();                                 // previous row's s_in / s_c consumed
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const int p = 4 * (tid + q * T);
            if (p < n) *reinterpret_cast<float4 *>(s_in + a.KO + p) = reg[q];
        }
        if (has_halo) s_in[hdst] = hreg;
        if (row + row_step < a.n_rows) fetch();
        if (nz) {
#pragma unroll
            for (int k = 0; k < OBS_NBR; ++k) {
                const int m = tid + k * T;
                nzr[k] = m < nb ? __ldcs(nz + m) : 0.0f;
            }
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const int p = 4 * (tid + q * T);
            if (p < n) {
                const float *si = s_in + p;
                float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f, acc3 = 0.f;
                if constexpr (LT <= OBS_PACKED_LT) {
                    // packed FP32 (FFMA2): output r keeps an (even inputs, odd inputs) pair of partial sums, the
                    // input pairs (x, y) and (z, w) come straight out of the LDS.128 and the weight pairs
                    // (wp[k], wp[k + 1]) are loop-invariant registers: 8 FFMA2 per LDS.128 instead of 16 FFMA
                    unsigned long long c0 = 0ull, c1 = 0ull, c2 = 0ull, c3 = 0ull;
#pragma unroll
                    for (int u = 0; u < LT + 4; u += 4) {
                        const float4 x = *reinterpret_cast<const float4 *>(si + u);
                        const unsigned long long xy = pack2(x.x, x.y), zw = pack2(x.z, x.w);
                        c0 = ffma2(xy, OBS_WPAIR(u + 3), c0); c0 = ffma2(zw, OBS_WPAIR(u + 5), c0);
                        c1 = ffma2(xy, OBS_WPAIR(u + 2), c1); c1 = ffma2(zw, OBS_WPAIR(u + 4), c1);
                        c2 = ffma2(xy, OBS_WPAIR(u + 1), c2); c2 = ffma2(zw, OBS_WPAIR(u + 3), c2);
                        c3 = ffma2(xy, OBS_WPAIR(u + 0), c3); c3 = ffma2(zw, OBS_WPAIR(u + 2), c3);
                    }
                    acc0 = sum2(c0); acc1 = sum2(c1); acc2 = sum2(c2); acc3 = sum2(c3);
                } else {
#pragma unroll
                    for (int u = 0; u < LT + 4; u += 4) {    // input u and output r use wp[u - r + 3]
                        const float4 x = *reinterpret_cast<const float4 *>(si + u);
                        acc0 = fmaf(tp.wp[u + 3], x.x, acc0); acc0 = fmaf(tp.wp[u + 4], x.y, acc0); acc0 = fmaf(tp.wp[u + 5], x.z, acc0); acc0 = fmaf(tp.wp[u + 6], x.w, acc0);
                        acc1 = fmaf(tp.wp[u + 2], x.x, acc1); acc1 = fmaf(tp.wp[u + 3], x.y, acc1); acc1 = fmaf(tp.wp[u + 4], x.z, acc1); acc1 = fmaf(tp.wp[u + 5], x.w, acc1);
                        acc2 = fmaf(tp.wp[u + 1], x.x, acc2); acc2 = fmaf(tp.wp[u + 2], x.y, acc2); acc2 = fmaf(tp.wp[u + 3], x.z, acc2); acc2 = fmaf(tp.wp[u + 4], x.w, acc2);
                        acc3 = fmaf(tp.wp[u + 0], x.x, acc3); acc3 = fmaf(tp.wp[u + 1], x.y, acc3); acc3 = fmaf(tp.wp[u + 2], x.z, acc3); acc3 = fmaf(tp.wp[u + 3], x.w, acc3);
                    }
                }
                *reinterpret_cast<float4 *>(s_c + p) = make_float4(acc0, acc1, acc2, acc3);
            }
        }
        __syncthreads();

        // output bins m = tid + k T: the three rebinning modes are uniform over the launch, so each gets its own loop
        const float inv_snr = nz ? a.inv_snr : 0.0f;
        auto put = [&](int k, int m, float v) {
            if (nz) v = fmaf(k < OBS_NBR ? nzr[k < OBS_NBR ? k : 0] : __ldcs(nz + m), inv_snr, v);
            __stcs(dst + m, v);
        };
        if (a.bins3) {                                   // bins <= 2 pixels wide: three pixels {i0, w0, w1, w2}
#pragma unroll
            for (int k = 0; k < OBS_NBR; ++k) {
                const int m = tid + k * T;
                if (m < nb) {
                    const int4 e = s_b[m];
                    const float *c = s_c + e.x;
                    put(k, m, fmaf(__int_as_float(e.w), c[2], fmaf(__int_as_float(e.z), c[1], __int_as_float(e.y) * c[0])));
                }
            }
            for (int m = tid + OBS_NBR * T; m < nb; m += T) {
                const int4 e = s_b[m];
                const float *c = s_c + e.x;
                put(OBS_NBR, m, fmaf(__int_as_float(e.w), c[2], fmaf(__int_as_float(e.z), c[1], __int_as_float(e.y) * c[0])));
            }
        } else if (a.rebin) {                            // wide bins: first pixel, whole pixels, last pixel (weights carry 1/B)
            auto wide = [&](int m) -> float {
                const int4 e = s_b[m];
                if (e.y <= e.x) return __int_as_float(e.z) * s_c[e.x];
                float mid = 0.0f;
#pragma unroll 1
                for (int i = e.x + 1; i < e.y; ++i) mid += s_c[i];
                return fmaf(__int_as_float(e.w), s_c[e.y], fmaf(mid, a.inv_bin_f, __int_as_float(e.z) * s_c[e.x]));
            };
#pragma unroll
            for (int k = 0; k < OBS_NBR; ++k) {
                const int m = tid + k * T;
                if (m < nb) put(k, m, wide(m));
            }
            for (int m = tid + OBS_NBR * T; m < nb; m += T) put(OBS_NBR, m, wide(m));
        } else {
#pragma unroll
            for (int k = 0; k < OBS_NBR; ++k) {
                const int m = tid + k * T;
                if (m < nb) put(k, m, s_c[m]);
            }
            for (int m = tid + OBS_NBR * T; m < nb; m += T) put(OBS_NBR, m, s_c[m]);
        }
        dst += out_step;
        if (nz) nz += out_step;
    }
}

// ---- the lean kernel with EIGHT consecutive outputs per thread (packed path only: at most 41 tap slots; rows of
// n % 8 == 0 pixels, n / 8 <= 256 threads).  The convolution then needs (LT + 8) / 4 LDS.128 per eight outputs instead
// of (LT + 4) / 4 per four, fewer distinct weight pairs per pixel, and every per-thread cost (staging, row change,
// barriers, address set-up) is spread over twice as many pixels: 66 -> ~45 instructions per pixel for the BOSS-like
// instrument.  Lanes that own 8 pixels sit 32 bytes apart, which would make every LDS.128 of the staged row a 2-way
// bank conflict; so the row is staged SPLIT by 16-byte chunk parity -- even chunks (4 pixels each) in one array, odd
// chunks in another: a thread's window alternates between the two with immediate offsets, and within either array
// neighbouring lanes read neighbouring chunks.
// shared-memory loads by 32-bit shared address (the output loop below: no generic-to-shared conversion per access)
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float lds_f32(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ int4 lds_v4(unsigned addr)
{
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

struct __align__(16) ObsTaps8 {
    float wp[64];                                        // wp[t + 7] = g(KO - t); zero outside the real taps
    float wq[64];                                        // wq[k] = wp[k + 1]
};
#define OBS_WPAIR8(k) (((k) & 1) ? pack2(tp.wq[(k) - 1], tp.wq[(k)]) : pack2(tp.wp[(k)], tp.wp[(k) + 1]))

constexpr int OBS_NBR8 = 6;                              // noise draws per thread and row held in registers (8-pixel kernel)
template <int LT, int T>                                 // LT >= L, multiple of 4, <= OBS_PACKED_LT; T = blockDim.x
__global__ void __launch_bounds__(T) observe_rows_lean8_kernel(const ObsArgs a, const __grid_constant__ ObsTaps8 tp)
{
    extern __shared__ __align__(16) float sm[];
    const int n = a.n, tid = threadIdx.x, nb = a.nb;
    constexpr int NJ = (LT + 8) / 4;                     // chunks in a thread's window
    const int nch = ((n + LT + 12) >> 3) + 1;            // chunks per half of the staged row (logical length n + LT + 12)
    float4 *s_e = reinterpret_cast<float4 *>(sm);        // even chunks of s_in[h] = F[(h - KO) mod n], zero beyond n + L
    float4 *s_o = s_e + nch;                             // odd chunks
    float *s_c  = reinterpret_cast<float *>(s_o + nch);  // convolved row, n floats (+ 4 zeros for the 3-tap rebin)
    int4  *s_b  = reinterpret_cast<int4 *>(s_c + n + 4); // bin table, nb entries (rebin only)
    auto in_chunk = [&](int c) -> float4 * { return ((c & 1) ? s_o : s_e) + (c >> 1); };
    for (int h = tid; h < 2 * nch; h += T) s_e[h] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid < 4) s_c[n + tid] = 0.0f;
    if (a.rebin)
        for (int m = tid; m < nb; m += T) {
            int4 e = a.bins[m];
            if (a.bins3) e.x *= 4;                       // three-pixel bins: first pixel as a byte offset into s_c
            s_b[m] = e;
        }
    const unsigned sc_addr = smem_addr(s_c), sb_addr = smem_addr(s_b) + 16u * tid;
    // three-pixel bins: a thread serves the SAME bins tid + k T in every row, so their table entries live in registers
    // (the per-bin LDS.128 was 2.8 of the ~13 shared-memory wavefronts per 32 pixels; ncu: shared-memory pipe 74 %)
    int4 eb[OBS_NBR8];
#pragma unroll
    for (int k = 0; k < OBS_NBR8; ++k) {
        eb[k] = make_int4(0, 0, 0, 0);
        if (a.bins3 && tid + k * T < nb) {
            eb[k] = a.bins[tid + k * T];
            eb[k].x *= 4;
        }
    }

    const bool own = 8 * tid < n;                        // this thread owns pixels 8 tid .. 8 tid + 7
    const bool has_halo = tid < a.L;
    const int hsrc = tid < a.KO ? n - a.KO + tid : tid - a.KO;       // this thread's halo pixel and where it goes
    const int hdst = tid < a.KO ? tid : n + tid;
    float *hptr = reinterpret_cast<float *>(in_chunk(hdst >> 2)) + (hdst & 3);
    float4 *own0 = in_chunk((a.KO >> 2) + 2 * tid), *own1 = in_chunk((a.KO >> 2) + 2 * tid + 1);
    const float4 *we = s_e + tid, *wo = s_o + tid;       // window: chunk 2 tid + j is (j even) we[j / 2], (j odd) wo[j / 2]
    const size_t row_step = gridDim.x;
    const float *src = a.flux + (size_t)blockIdx.x * n;
    const float *nz  = a.noise ? a.noise + (size_t)blockIdx.x * nb : nullptr;
    float *dst = a.out + (size_t)blockIdx.x * nb;
    const size_t src_step = row_step * n, out_step = row_step * nb;
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
    float hreg = 0.0f, nzr[OBS_NBR8];
    auto fetch = [&]() {
        if (own) {
            r0 = __ldcs(reinterpret_cast<const float4 *>(src + 8 * tid));
            r1 = __ldcs(reinterpret_cast<const float4 *>(src + 8 * tid + 4));
        }
        if (has_halo) hreg = __ldg(src + hsrc);
        src += src_step;
    };
    size_t row = blockIdx.x;
    if (row < a.n_rows) fetch();
    for (; row < a.n_rows; row += row_step) {
        __syncthreads();                                 // previous row's staged row / s_c consumed
        if (own) { *own0 = r0; *own1 = r1; }
        if (has_halo) *hptr = hreg;
        if (row + row_step < a.n_rows) fetch();
        if (nz) {
#pragma unroll
            for (int k = 0; k < OBS_NBR8; ++k) {
                const int m = tid + k * T;
                nzr[k] = m < nb ? __ldcs(nz + m) : 0.0f;
            }
        }
        __syncthreads();
        if (own) {
            unsigned long long c[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) c[r] = 0ull;
#pragma unroll
            for (int j = 0; j < NJ; ++j) {               // input u = 4 j + {0..3} and output r use wp[u - r + 7]
                const float4 x = (j & 1) ? wo[j >> 1] : we[j >> 1];
                const unsigned long long xy = pack2(x.x, x.y), zw = pack2(x.z, x.w);
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    c[r] = ffma2(xy, OBS_WPAIR8(4 * j - r + 7), c[r]);
                    c[r] = ffma2(zw, OBS_WPAIR8(4 * j - r + 9), c[r]);
                }
            }
            float4 *d = reinterpret_cast<float4 *>(s_c + 8 * tid);
            d[0] = make_float4(sum2(c[0]), sum2(c[1]), sum2(c[2]), sum2(c[3]));
            d[1] = make_float4(sum2(c[4]), sum2(c[5]), sum2(c[6]), sum2(c[7]));
        }
        __syncthreads();

        const float inv_snr = nz ? a.inv_snr : 0.0f;
        auto put = [&](int k, int m, float v) {
            if (nz) v = fmaf(k < OBS_NBR8 ? nzr[k < OBS_NBR8 ? k : 0] : __ldcs(nz + m), inv_snr, v);
            __stcs(dst + m, v);
        };
        if (a.bins3) {                                   // bins <= 2 pixels wide: three pixels {byte offset, w0, w1, w2}
            float *dt = dst + tid;                       // every offset below is an immediate (T is a template parameter)
            const float *nt = nz ? nz + tid : nullptr;
#pragma unroll
            for (int k = 0; k < OBS_NBR8; ++k) {
                if (tid + k * T < nb) {
                    const int4 e = eb[k];
                    const unsigned ca = sc_addr + (unsigned)e.x;
                    float v = fmaf(__int_as_float(e.w), lds_f32(ca + 8), fmaf(__int_as_float(e.z), lds_f32(ca + 4), __int_as_float(e.y) * lds_f32(ca)));
                    if (nz) v = fmaf(nzr[k], inv_snr, v);
                    __stcs(dt + k * T, v);
                }
            }
            for (int m = tid + OBS_NBR8 * T; m < nb; m += T) {
                const int4 e = lds_v4(sb_addr + 16u * (m - tid));
                const unsigned ca = sc_addr + (unsigned)e.x;
                float v = fmaf(__int_as_float(e.w), lds_f32(ca + 8), fmaf(__int_as_float(e.z), lds_f32(ca + 4), __int_as_float(e.y) * lds_f32(ca)));
                if (nz) v = fmaf(__ldcs(nt + (m - tid)), inv_snr, v);
                __stcs(dt + (m - tid), v);
            }
        } else if (a.rebin) {                            // wide bins: first pixel, whole pixels, last pixel (weights carry 1/B)
            auto wide = [&](int m) -> float {
                const int4 e = s_b[m];
                if (e.y <= e.x) return __int_as_float(e.z) * s_c[e.x];
                float mid = 0.0f;
#pragma unroll 1
                for (int i = e.x + 1; i < e.y; ++i) mid += s_c[i];
                return fmaf(__int_as_float(e.w), s_c[e.y], fmaf(mid, a.inv_bin_f, __int_as_float(e.z) * s_c[e.x]));
            };
            for (int m = tid, k = 0; m < nb; m += T, ++k) put(k < OBS_NBR8 ? k : OBS_NBR8, m, wide(m));
        } else {
            for (int m = tid, k = 0; m < nb; m += T, ++k) put(k < OBS_NBR8 ? k : OBS_NBR8, m, s_c[m]);
        }
        dst += out_step;
        if (nz) nz += out_step;
    }
}

// ---- flux PDF: private per-thread histograms in shared memory (hist[bin][thread]: conflict-free, no atomics)
constexpr int PDF_THREADS = 128;

__global__ void __launch_bounds__(PDF_THREADS) flux_pdf_kernel(const float *__restrict__ flux, size_t n,
                                                               const __grid_constant__ PdfEdges edges,
                                                               unsigned long long *counts, unsigned long long *host,
                                                               unsigned int *ticket, int reps)
{
    extern __shared__ unsigned int hist[];               // [n_bins][PDF_THREADS], then n_bins + 1 thresholds
    const int n_bins = edges.n_bins;
    float *s_thr = reinterpret_cast<float *>(hist + n_bins * PDF_THREADS);
    for (int t = threadIdx.x; t < n_bins * PDF_THREADS; t += PDF_THREADS) hist[t] = 0u;
    for (int t = threadIdx.x; t <= n_bins; t += PDF_THREADS) s_thr[t] = edges.thr[t];
    __syncthreads();
    unsigned int *mine = hist + threadIdx.x;
    const float f_lo = edges.f_lo, inv_width = edges.inv_width, eps = edges.eps, ome = edges.one_minus_eps;
    auto add = [&](float f) { atomicAdd(mine + lya_pdf_bin(f, s_thr, n_bins, f_lo, inv_width, eps, ome) * PDF_THREADS, 1u); };
    const size_t gtid = (size_t)blockIdx.x * PDF_THREADS + threadIdx.x, gsz = (size_t)gridDim.x * PDF_THREADS;
    size_t head = ((16 - ((uintptr_t)flux & 15)) & 15) >> 2;
    if (head > n) head = n;
    const size_t n4 = (n - head) >> 2;
    const float4 *f4 = reinterpret_cast<const float4 *>(flux + head);
#pragma unroll 2
    for (size_t i = gtid; i < n4; i += gsz) {
        const float4 f = __ldcs(f4 + i);
        add(f.x); add(f.y); add(f.z); add(f.w);
    }
    const size_t tail0 = head + (n4 << 2), n_edge = head + (n - tail0);
    for (size_t e = gtid; e < n_edge; e += gsz) add(flux[e < head ? e : tail0 + (e - head)]);
    __syncthreads();
    // one warp per bin: sum the 128 private counters, one atomic per bin and CTA
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int b = warp; b < n_bins; b += PDF_THREADS / 32) {
        unsigned int s = 0;
        for (int t = lane; t < PDF_THREADS; t += 32) s += hist[b * PDF_THREADS + t];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0 && s) atomicAdd(counts + (blockIdx.x % reps) * n_bins + b, (unsigned long long)s);
    }
    lya_publish_last_cta(counts, n_bins, host, ticket, reps);
}

}  // namespace

extern "C" double lya_bin_kms_from_angstrom(double z, double dlambda_angstrom)
{
    return (LYA_C_CGS * 1.0e-5) * dlambda_angstrom / (1215.67 * (1.0 + z));
}

extern "C" int32_t lya_instrument_bins(int32_t n_pix, double dv_kms, const lya_instrument *inst)
{
    if (!inst || n_pix < 1 || !(dv_kms > 0.0)) return 0;
    if (!(inst->bin_kms > 0.0)) return n_pix;
    return (int32_t)floor((double)n_pix * dv_kms / inst->bin_kms + 1e-9);
}

extern "C" lya_status lya_observe_rows(lya_ctx *ctx, size_t n_rows, int32_t n_pix, double dv_kms,
                                       const lya_instrument *inst, const float *flux, const float *unit_noise,
                                       float *out)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!inst || (n_rows > 0 && (!flux || !out))) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: null pointer");
    if (n_pix < 1 || !(dv_kms > 0.0)) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: n_pix >= 1 and dv > 0 required");
    if ((((uintptr_t)flux | (uintptr_t)out | (uintptr_t)unit_noise) & 3) != 0)
        return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: pointers must be 4-byte aligned");
    if (n_rows > 0 && out == flux) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: out may not alias flux");
    if (inst->snr > 0.0 && !unit_noise) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: snr > 0 needs unit_noise");
    const int32_t nb = lya_instrument_bins(n_pix, dv_kms, inst);
    if (nb < 1) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: bin wider than the row");
    if (n_rows == 0) return LYA_OK;
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));

    ObsArgs a;
    memset(&a, 0, sizeof(a));
    a.flux = flux; a.noise = inst->snr > 0.0 ? unit_noise : nullptr; a.out = out;
    a.n_rows = n_rows; a.n = n_pix; a.n4 = (n_pix + 3) & ~3; a.nb = nb;
    a.rebin = inst->bin_kms > 0.0;
    const double bin_px = a.rebin ? inst->bin_kms / dv_kms : 1.0;
    if (bin_px < 1.0e-6) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: bin narrower than 1e-6 pixel");
    a.bin_fx = (unsigned long long)llrint(bin_px * 4294967296.0);
    a.inv_bin_f = (float)(1.0 / bin_px);
    a.inv_snr = inst->snr > 0.0 ? (float)(1.0 / inst->snr) : 0.0f;
    int threads = ((a.n4 / 4 + 31) / 32) * 32;
    threads = threads < 32 ? 32 : (threads > 256 ? 256 : threads);
    bool fast = (n_pix % 4 == 0) && (((uintptr_t)flux & 15) == 0);
    a.L = -1;
    if (inst->fwhm_kms > 0.0) {
        const double sigma_px = inst->fwhm_kms / (2.0 * sqrt(2.0 * log(2.0))) / dv_kms;
        // taps beyond 5 sigma dropped: the two tails hold erfc(5 / sqrt 2) = 5.7e-7 of the kernel, so |error| <= 5.7e-7 max F
        const double kd = ceil(5.0 * sigma_px);
        const int K = kd < 1.0 ? 1 : (kd > 1.0e6 ? 1000000 : (int)kd);
        a.Kl = K < (n_pix - 1) / 2 ? K : (n_pix - 1) / 2;
        a.Kr = K < n_pix / 2 ? K : n_pix / 2;
        const int ko4 = (a.Kr + 3) & ~3;
        fast = fast && ko4 <= n_pix && ko4 + a.Kl <= threads;
        a.KO = fast ? ko4 : a.Kr;
        a.L = a.KO + a.Kl;
        if (a.L > 8192) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: Gaussian wider than 4096 taps a side");
        const int n_t = a.L + 11;
        if (ctx->taps_cap < (size_t)n_t) {
            if (ctx->d_taps) cudaFree(ctx->d_taps);
            ctx->d_taps = nullptr; ctx->taps_cap = 0;
            free(ctx->h_taps);
            ctx->h_taps = (float *)malloc((size_t)(n_t + 64) * sizeof(float));
            if (!ctx->h_taps) return lya_fail(ctx, LYA_ENOMEM, "lya_observe_rows: host allocation failed");
            LYA_CUDA(ctx, cudaMalloc((void **)&ctx->d_taps, (size_t)(n_t + 64) * sizeof(float)));
            ctx->taps_cap = (size_t)n_t + 64;
            ctx->taps_key[0] = -1.0;
        }
        // the taps depend on (sigma, Kl, Kr, KO) only: a repeated call (the usual case: one instrument, many
        // slabs) finds them on the device already and needs neither a synchronisation nor a copy
        if (!(ctx->taps_key[0] == sigma_px && ctx->taps_key[1] == (double)a.Kl && ctx->taps_key[2] == (double)a.Kr &&
              ctx->taps_key[3] == (double)a.KO)) {
            // the stream may still be reading the previous call's taps: wait before overwriting the host copy
            LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            double sum = 0.0;
            for (int k = -a.Kl; k <= a.Kr; ++k) sum += exp(-0.5 * (double)k * k / (sigma_px * sigma_px));
            for (int t = 0; t < n_t; ++t) ctx->h_taps[t] = 0.0f;
            for (int t = a.KO - a.Kr; t <= a.L; ++t) {                  // offset k = KO - t in [-Kl, Kr]
                const double k = (double)(a.KO - t);
                ctx->h_taps[t + 3] = (float)(exp(-0.5 * k * k / (sigma_px * sigma_px)) / sum);
            }
            LYA_CUDA(ctx, cudaMemcpyAsync(ctx->d_taps, ctx->h_taps, (size_t)n_t * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
            ctx->taps_key[0] = sigma_px; ctx->taps_key[1] = a.Kl; ctx->taps_key[2] = a.Kr; ctx->taps_key[3] = a.KO;
        }
        a.taps = ctx->d_taps;
    }
    // ---- lean kernel for the common case
    const int nv_lean = (a.n4 / 4 + threads - 1) / threads;
    if (fast && a.L >= 0 && a.L <= 124 && nv_lean <= 4) {
        ObsTaps tp;
        memset(&tp, 0, sizeof(tp));
        for (int t = 0; t < a.L + 11; ++t) tp.wp[t] = ctx->h_taps[t];
        for (int t = 0; t < 135; ++t) tp.wq[t] = tp.wp[t + 1];
        if (a.rebin) {
            if (ctx->bins_cap < (size_t)nb) {
                if (ctx->d_bins) cudaFree(ctx->d_bins);
                ctx->d_bins = nullptr; ctx->bins_cap = 0;
                free(ctx->h_bins);
                ctx->h_bins = malloc((size_t)(nb + 64) * sizeof(int4));
                if (!ctx->h_bins) return lya_fail(ctx, LYA_ENOMEM, "lya_observe_rows: host allocation failed");
                LYA_CUDA(ctx, cudaMalloc(&ctx->d_bins, (size_t)(nb + 64) * sizeof(int4)));
                ctx->bins_cap = (size_t)nb + 64;
                ctx->bins_key[0] = -1.0;
            }
            a.bins3 = bin_px <= 2.0;
            if (!(ctx->bins_key[0] == bin_px && ctx->bins_key[1] == (double)n_pix && ctx->bins_key[2] == (double)nb)) {
                LYA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));         // previous call may still read h_bins
                int4 *hb = (int4 *)ctx->h_bins;
                a.bins3 = bin_px <= 2.0;
                for (int m = 0; m < nb; ++m) {                                  // bin [lo, hi) in pixel units (reading O2)
                    const double lo = (double)m * bin_px, hi = lo + bin_px;
                    int i0 = (int)floor(lo), i1 = (int)ceil(hi) - 1;
                    if (i1 > n_pix - 1) i1 = n_pix - 1;
                    int4 e;
                    if (a.bins3) {                                              // overlap of the bin with pixels i0, i0+1, i0+2
                        float wq[3];
                        for (int q = 0; q < 3; ++q) {
                            const double l = lo > (double)(i0 + q) ? lo : (double)(i0 + q);
                            const double h = hi < (double)(i0 + q + 1) ? hi : (double)(i0 + q + 1);
                            wq[q] = (h > l && i0 + q < n_pix) ? (float)((h - l) / bin_px) : 0.0f;
                        }
                        e.x = i0;
                        memcpy(&e.y, &wq[0], 4); memcpy(&e.z, &wq[1], 4); memcpy(&e.w, &wq[2], 4);
                    } else {
                        float wf, wl;
                        if (i1 <= i0) { i1 = i0; wf = (float)((hi - lo) / bin_px); wl = 0.0f; }
                        else { wf = (float)(((double)(i0 + 1) - lo) / bin_px); wl = (float)((hi - (double)i1) / bin_px); }
                        e.x = i0; e.y = i1;
                        memcpy(&e.z, &wf, 4); memcpy(&e.w, &wl, 4);
                    }
                    hb[m] = e;
                }
                LYA_CUDA(ctx, cudaMemcpyAsync(ctx->d_bins, hb, (size_t)nb * sizeof(int4), cudaMemcpyHostToDevice, ctx->stream));
                ctx->bins_key[0] = bin_px; ctx->bins_key[1] = n_pix; ctx->bins_key[2] = nb;
            }
            a.bins = (const int4 *)ctx->d_bins;
        }
        // LT: the smallest instantiated multiple of 4 that is >= L (every multiple of 4 up to 64, then 96, 124)
        const int LT = a.L <= 64 ? ((a.L + 3) & ~3) : (a.L <= 96 ? 96 : 124);
        // eight outputs per thread where the packed convolution applies and the row gives every thread eight pixels
        if (LT <= OBS_PACKED_LT && n_pix % 8 == 0 && n_pix >= 256 && n_pix <= 2048) {
            ObsTaps8 t8;
            memset(&t8, 0, sizeof(t8));
            for (int t = 0; t <= a.L + 7 && t + 7 < 64; ++t) t8.wp[t + 4] = ctx->h_taps[t];      // h_taps[t + 3] = g(KO - t)
            for (int t = 0; t < 63; ++t) t8.wq[t] = t8.wp[t + 1];
            void (*lean8)(const ObsArgs, const ObsTaps8) = nullptr;
            const int threads8 = ((n_pix / 8 + 31) / 32) * 32;
            const int t8c = threads8 <= 32 ? 32 : (threads8 <= 64 ? 64 : (threads8 <= 128 ? 128 : 256));   // instantiated block sizes
            switch (LT) {
#define LYA_LEAN8(N) case N: lean8 = t8c == 32 ? observe_rows_lean8_kernel<N, 32> : (t8c == 64 ? observe_rows_lean8_kernel<N, 64> \
                             : (t8c == 128 ? observe_rows_lean8_kernel<N, 128> : observe_rows_lean8_kernel<N, 256>)); break;
                LYA_LEAN8(0) LYA_LEAN8(4) LYA_LEAN8(8) LYA_LEAN8(12) LYA_LEAN8(16) LYA_LEAN8(20) LYA_LEAN8(24)
                LYA_LEAN8(28) LYA_LEAN8(32) LYA_LEAN8(36) LYA_LEAN8(40)
#undef LYA_LEAN8
            }
            const size_t nch = (((size_t)n_pix + LT + 12) >> 3) + 1;
            const size_t smem8 = 2 * nch * sizeof(float4) + ((size_t)n_pix + 4) * sizeof(float) + (a.rebin ? (size_t)nb * sizeof(int4) : 0);
            int per_sm8 = 0;
            lya_status st8 = lya_kernel_occupancy(ctx, (const void *)lean8, t8c, smem8, &per_sm8);
            if (st8 != LYA_OK) return st8;
            if (lean8 && per_sm8 >= 1 && a.L <= t8c) {
                const size_t cap8 = (size_t)ctx->sm_count * per_sm8;
                lean8<<<(int)(n_rows < cap8 ? n_rows : cap8), t8c, smem8, ctx->stream>>>(a, t8);
                ctx->launches++;
                LYA_CUDA(ctx, cudaGetLastError());
                return LYA_OK;
            }
        }
        void (*lean)(const ObsArgs, const ObsTaps) = nullptr;
        switch (LT) {
#define LYA_LEAN(N) case N: lean = nv_lean == 1 ? observe_rows_lean_kernel<N, 1> : (nv_lean == 2 ? observe_rows_lean_kernel<N, 2> : observe_rows_lean_kernel<N, 4>); break;
            LYA_LEAN(0) LYA_LEAN(4) LYA_LEAN(8) LYA_LEAN(12) LYA_LEAN(16) LYA_LEAN(20) LYA_LEAN(24) LYA_LEAN(28)
            LYA_LEAN(32) LYA_LEAN(36) LYA_LEAN(40) LYA_LEAN(44) LYA_LEAN(48) LYA_LEAN(52) LYA_LEAN(56) LYA_LEAN(60)
            LYA_LEAN(64) LYA_LEAN(96) LYA_LEAN(124)
#undef LYA_LEAN
        }
        const size_t smem_l = ((size_t)n_pix + LT + 8 + n_pix + 4) * sizeof(float) + (a.rebin ? (size_t)nb * sizeof(int4) : 0);
        int per_sm_l = 0;
        lya_status st_l = lya_kernel_occupancy(ctx, (const void *)lean, threads, smem_l, &per_sm_l);
        if (st_l != LYA_OK) return st_l;
        if (per_sm_l >= 1) {
            const size_t cap_l = (size_t)ctx->sm_count * per_sm_l;
            lean<<<(int)(n_rows < cap_l ? n_rows : cap_l), threads, smem_l, ctx->stream>>>(a, tp);
            ctx->launches++;
            LYA_CUDA(ctx, cudaGetLastError());
            return LYA_OK;
        }
    }
    const int nv = (a.n4 / 4 + threads - 1) / threads;                 // float4 per thread and row
    void (*kern)(const ObsArgs) = nullptr;
    int D = 1;
    if (nv <= 1)       kern = fast ? observe_rows_kernel<1, 1, true> : observe_rows_kernel<1, 1, false>;
    else if (nv <= 2)  kern = fast ? observe_rows_kernel<2, 1, true> : observe_rows_kernel<2, 1, false>;
    else if (nv <= 4)  kern = fast ? observe_rows_kernel<4, 1, true> : observe_rows_kernel<4, 1, false>;
    else if (nv <= 8)  kern = fast ? observe_rows_kernel<8, 1, true> : observe_rows_kernel<8, 1, false>;
    else if (nv <= 16) kern = fast ? observe_rows_kernel<16, 1, true> : observe_rows_kernel<16, 1, false>;
    else return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: more than 16384 pixels per row");
    const int halo = a.L >= 0 ? a.L : 0;
    const size_t smem = ((size_t)D * (a.n4 + ((halo + 3) & ~3) + 8) + (size_t)D * a.n4 + (((halo + 11) + 3) & ~3)) * sizeof(float);
    if (smem > (size_t)ctx->max_smem_optin) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: row too long for shared memory");
    int per_sm = 0;
    lya_status st_g = lya_kernel_occupancy(ctx, (const void *)kern, threads, smem, &per_sm);
    if (st_g != LYA_OK) return st_g;
    if (per_sm < 1) return lya_fail(ctx, LYA_EINVAL, "lya_observe_rows: row too long for shared memory");
    const size_t cap = (size_t)ctx->sm_count * per_sm;
    const size_t n_batches = (n_rows + D - 1) / D;
    const int grid = (int)(n_batches < cap ? n_batches : cap);
    kern<<<grid, threads, smem, ctx->stream>>>(a);
    ctx->launches++;
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}

extern "C" lya_status lya_flux_pdf(lya_ctx *ctx, const float *flux, size_t n, int32_t n_bins, double f_lo,
                                   double width, uint64_t *counts, double *pdf)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (n > 0 && (!flux || ((uintptr_t)flux & 3))) return lya_fail(ctx, LYA_EINVAL, "lya_flux_pdf: bad flux pointer");
    if (n_bins < 1 || n_bins > 256 || !(width > 0.0)) return lya_fail(ctx, LYA_EINVAL, "lya_flux_pdf: 1 <= n_bins <= 256 and width > 0 required");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    unsigned long long *d_counts = reinterpret_cast<unsigned long long *>(ctx->d_stats);
    unsigned long long *host = reinterpret_cast<unsigned long long *>(ctx->h_pinned + LYA_PINNED_STATS);
    if (n > 0) {
        PdfEdges edges;
        lya_pdf_edges(n_bins, f_lo, width, &edges);
        const size_t smem = (size_t)n_bins * PDF_THREADS * sizeof(unsigned int) + (size_t)(n_bins + 1) * sizeof(float);
        int per_sm = 0;
        lya_status st = lya_kernel_occupancy(ctx, (const void *)flux_pdf_kernel, PDF_THREADS, smem, &per_sm);
        if (st != LYA_OK) return st;
        if (per_sm < 1) return lya_fail(ctx, LYA_EINVAL, "lya_flux_pdf: too many bins for shared memory");
        size_t want = (n / 4 + PDF_THREADS - 1) / PDF_THREADS;
        if (want < 1) want = 1;
        const size_t cap = (size_t)ctx->sm_count * per_sm;
        st = lya_stats_begin(ctx, n_bins);
        if (st != LYA_OK) return st;
        // the last CTA to finish writes the totals straight to the pinned mirror and re-zeroes the device counters
        flux_pdf_kernel<<<(int)(want < cap ? want : cap), PDF_THREADS, smem, ctx->stream>>>(flux, n, edges, d_counts, host,
                                                                                           ctx->d_sched + 4, lya_stats_replicas(n_bins, n, 16));
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
