// power.cu -- 1D flux power spectrum along the line of sight, averaged over rows:
//   P(k_m) = (V/N^2) < |sum_i dF_i exp(-2 pi i m i / N)|^2 >,  dF = F / <F> - 1,  m = 0 .. N/2   (reading O5)
//
// One CTA transforms two rows at a time as ONE complex FFT (row A in the real part, row B in the imaginary
// part; X_A(m) = (Z(m) + conj Z(N-m))/2, X_B(m) = (Z(m) - conj Z(N-m))/(2i)).  The FFT is a Stockham
// autosort transform in 1-4 passes of radix 16 / 8 / 4: a thread loads R points (the first pass straight
// from global memory, coalesced), applies the pass twiddles (one table look-up, the powers by at most four
// complex products), does the R-point DFT in registers (radix-2 DIF with compile-time constants) and
// scatters the result to the other shared-memory buffer, whose index is padded by one slot in 16 so that the
// stride-R scatter of the first pass is bank-conflict free.  4 B read per pixel; N = 1024 makes 3 passes = 2
// shared-memory round trips per point (the radix-2 version this replaces made 10, with a barrier each).  The
// butterflies' complex additions are packed FP32 (add/sub.rn.f32x2) for rows of 512 pixels and more.
// The two rows never have to be separated: |X_A(m)|^2 + |X_B(m)|^2 = (|Z(m)|^2 + |Z(N-m)|^2) / 2, and only the sum
// over rows is wanted, so for the common sizes (256 ... 4096 pixels) the LAST pass keeps |Z(k)|^2 of its own outputs
// in double registers across all the CTA's row pairs -- no final store, no read-out pass, two barriers per pair
// instead of four -- and the host folds k and N - k once at the end.  Other sizes write the last pass to shared
// memory and read the pairs (m, N - m) out (accumulated in double per CTA).
// Rows of 256 ... 2048 pixels (configs 2-5) take flux_power_warp_kernel / _short_kernel instead: ONE WARP per transform (32 x 32
// in two register passes, 2048 as two such transforms by a radix-2 split shared by a team of two warps), the next row
// pair prefetched by one cp.async.bulk, no CTA barrier in the loop: 1.30 -> 0.88 ms on 1024^3, 1.36 -> 0.97 ms on
// 2048-pixel rows.
#include "lya_internal.h"
#include "pdf_bin.h"

namespace {

struct PowArgs {
    const float *flux;
    size_t       n_rows;
    int          n, log2n;
    int          n_pass, radix[4];
    float        inv_mean;
    double      *acc;          // device accumulators (n or n/2 + 1 doubles), zero on entry and left zero
    double      *host;         // mapped pinned mirror: the last CTA to finish writes the totals there
    unsigned int *ticket;
    int          n_acc;
    int          reps;         // replicas of the n_acc accumulators (lya_stats_replicas): CTA b adds into replica b % reps
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }
// complex add / subtract as one packed FP32 instruction each (sm_100a add/sub.rn.f32x2 = FADD2)
__device__ __forceinline__ float2 cadd(float2 a, float2 b)
{
    unsigned long long x, y, r;
    float2 o;
    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(b.x), "f"(b.y));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(x), "l"(y));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(o.x), "=f"(o.y) : "l"(r));
    return o;
}
__device__ __forceinline__ float2 csub(float2 a, float2 b)
{
    unsigned long long x, y, r;
    float2 o;
    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(b.x), "f"(b.y));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(x), "l"(y));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(o.x), "=f"(o.y) : "l"(r));
    return o;
}

// R-point DFT in registers, radix-2 decimation in frequency: the result for frequency t ends up in
// v[bitrev_R(t)].  All indices and twiddles are compile-time constants once unrolled.
// PACK: butterflies' complex add / subtract as FADD2 (measured: 1024-pixel rows 1.654 -> 1.580 ms, 256-pixel rows
// 2.5 % slower, so only rows of 512 pixels and more take it).
template <int R, bool PACK>
__device__ __forceinline__ void dft_regs(float2 (&v)[R])
{
    constexpr float C[8] = {1.0f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f,
                            0.0f, -0.38268343236508977f, -0.70710678118654752f, -0.92387953251128674f};
    constexpr float S[8] = {0.0f, 0.38268343236508977f, 0.70710678118654752f, 0.92387953251128674f,
                            1.0f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f};
#pragma unroll
    for (int len = R; len >= 2; len >>= 1) {
        const int half = len >> 1;
#pragma unroll
        for (int s = 0; s < R; s += len) {
#pragma unroll
            for (int p = 0; p < half; ++p) {
                const float2 a = v[s + p], b = v[s + p + half];
                v[s + p] = PACK ? cadd(a, b) : make_float2(a.x + b.x, a.y + b.y);
                const float2 d = PACK ? csub(a, b) : make_float2(a.x - b.x, a.y - b.y);
                const int q = p * (16 / len);              // W_len^p = exp(-2 pi i q / 16), q < 8
                if (q == 0)      v[s + p + half] = d;
                else if (q == 4) v[s + p + half] = make_float2(d.y, -d.x);          // times -i
                else             v[s + p + half] = cmul(d, make_float2(C[q], -S[q]));
            }
        }
    }
}

template <int R> __device__ __forceinline__ constexpr int bitrev(int t)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (t & 1); t >>= 1; }
    return r;
}

// One Stockham pass of radix R.  ns = product of the radices of the passes already done.
//   v[t] = in[j + t N/R] ;  v[t] *= exp(-2 pi i t k / (ns R)), k = j mod ns ;  V = DFT_R(v) ;
//   out[(j - k) R + k + t ns] = V[t]
// FIRST: `in` is global memory (two rows -> one complex sequence, dF = F inv_mean - 1).
// N_CT / NS_CT > 0: row length and ns known at compile time (the common sizes), which turns every shared-memory
// offset below into an immediate; 0: taken from the arguments.
template <int R, bool FIRST, int N_CT = 0, int NS_CT = 0, bool LAST = false>
__device__ __forceinline__ void stockham_pass(const PowArgs &a, const float *ra, const float *rb, bool has_b,
                                              const float2 *in, float2 *out, const float2 *tw, int ns_rt,
                                              double *pacc = nullptr)
{
    const int n = N_CT > 0 ? N_CT : a.n, m = n / R;
    const int ns = NS_CT > 0 ? NS_CT : ns_rt;
    // padded addresses are affine in t: pad16(j + t m) = pad16(j) + t (m + m/16) for m >= 16, and
    // pad16(j0 + t ns) = pad16(j0) + t os_a + (t >> 1) os_b with (os_a, os_b) = (ns + ns/16, 0) for ns >= 16,
    // (8, 1) for ns == 8 (j0 mod 16 < 8 there), (1, 0) for ns == 1 (j0 = j R)
    const int is = m + (m >> 4);
    const int os_a = ns >= 16 ? ns + (ns >> 4) : ns, os_b = ns == 8 ? 1 : 0;
    const int tstep = m / ns;
    for (int j = threadIdx.x; j < m; j += blockDim.x) {
        float2 v[R];
        if (FIRST) {
#pragma unroll
            for (int t = 0; t < R; ++t) {
                const float fa = fmaf(__ldcs(ra + j + t * m), a.inv_mean, -1.0f);
                const float fb = has_b ? fmaf(__ldcs(rb + j + t * m), a.inv_mean, -1.0f) : 0.0f;
                v[t] = make_float2(fa, fb);
            }
        } else if (m >= 16) {
            const float2 *ib = in + pad16(j);
#pragma unroll
            for (int t = 0; t < R; ++t) v[t] = ib[t * is];
        } else {
#pragma unroll
            for (int t = 0; t < R; ++t) v[t] = in[pad16(j + t * m)];
        }
        const int k = j & (ns - 1);
        if (!FIRST) {                                     // ns == 1 in the first pass: all twiddles are 1
            // w^t, w = exp(-2 pi i k / (ns R)) = tw[k (n / (ns R))]; powers by products of depth <= 4
            float2 w[R];
            w[1] = tw[k * tstep];
#pragma unroll
            for (int t = 2; t < R; ++t) w[t] = (t & 1) ? cmul(w[t - 1], w[1]) : cmul(w[t >> 1], w[t >> 1]);
#pragma unroll
            for (int t = 1; t < R; ++t) v[t] = cmul(v[t], w[t]);
        }
        dft_regs<R, (N_CT == 0 || N_CT >= 512)>(v);
        if (LAST) {                                       // m <= blockDim.x here: one trip, pacc[t] belongs to output j + t ns
#pragma unroll
            for (int t = 0; t < R; ++t) {
                const float2 z = v[bitrev<R>(t)];
                pacc[t] += (double)fmaf(z.x, z.x, z.y * z.y);
            }
            continue;
        }
        float2 *ob = out + pad16((j - k) * R + k);
        if (ns == 2 || ns == 4) {                         // never produced by the plans (radices 16 / 8 first)
#pragma unroll
            for (int t = 0; t < R; ++t) out[pad16((j - k) * R + k + t * ns)] = v[bitrev<R>(t)];
        } else {
#pragma unroll
            for (int t = 0; t < R; ++t) ob[t * os_a + (t >> 1) * os_b] = v[bitrev<R>(t)];
        }
    }
}

// radix of pass i for the sizes with a compile-time plan (0: no such pass)
__host__ __device__ constexpr int plan_radix(int n, int i)
{
    return n == 256 ? (i < 2 ? 16 : 0) : n == 512 ? (i < 3 ? 8 : 0) : n == 1024 ? (i == 0 ? 16 : (i < 3 ? 8 : 0))
         : n == 2048 ? (i < 2 ? 16 : (i == 2 ? 8 : 0)) : n == 4096 ? (i < 3 ? 16 : 0) : 0;
}

template <int N_CT, bool REP = false>                    // REP: replicated accumulators (short launches only; see lya_stats_replicas)
__global__ void __launch_bounds__(256) flux_power_kernel(const PowArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = N_CT > 0 ? N_CT : a.n, nh = n >> 1, npad = n + (n >> 4) + 1;
    double *pw  = reinterpret_cast<double *>(smem_raw);                    // [nh + 1] (+1 pad)
    float2 *bufA = reinterpret_cast<float2 *>(pw + nh + 2);                // [npad]
    float2 *bufB = bufA + npad;                                            // [npad]
    float2 *tw  = bufB + npad;                                             // [nh]: exp(-2 pi i q / n)
    const int tid = threadIdx.x, T = blockDim.x;

    for (int q = tid; q < nh; q += T) {
        float s, c;
        sincospif(2.0f * (float)q / (float)n, &s, &c);
        tw[q] = make_float2(c, -s);
    }
    for (int m = tid; m <= nh; m += T) pw[m] = 0.0;

    __syncthreads();                                       // tables built
    constexpr int RL = N_CT > 0 ? (plan_radix(N_CT, 2) > 0 ? plan_radix(N_CT, 2) : plan_radix(N_CT, 1)) : 1;
    double pacc[RL];                                       // compile-time plans: |Z(k)|^2 of this thread's last-pass outputs
#pragma unroll
    for (int t = 0; t < RL; ++t) pacc[t] = 0.0;
    const size_t n_pairs = (a.n_rows + 1) >> 1;
    for (size_t pair = blockIdx.x; pair < n_pairs; pair += gridDim.x) {
        const float *ra = a.flux + (2 * pair) * (size_t)n;
        const bool has_b = 2 * pair + 1 < a.n_rows;
        const float *rb = ra + n;
        // the buffer the first pass writes was last read in the previous pair's LAST pass (two-pass plans, and the
        // read-out of the run-time plans); with three passes a barrier already lies in between
        if constexpr (!(N_CT > 0 && plan_radix(N_CT, 2) > 0)) __syncthreads();
        float2 *src = bufB, *dst = bufA;
        if constexpr (N_CT > 0) {                          // compile-time plan: immediates everywhere
            constexpr int R0 = plan_radix(N_CT, 0), R1 = plan_radix(N_CT, 1), R2 = plan_radix(N_CT, 2);
            stockham_pass<R0, true, N_CT, 1>(a, ra, rb, has_b, nullptr, bufA, tw, 1);
            __syncthreads();                               // (also: the previous pair's last pass has read bufB / bufA)
            if constexpr (R2 > 0) {
                stockham_pass<R1, false, N_CT, R0>(a, ra, rb, has_b, bufA, bufB, tw, R0);
                __syncthreads();
                stockham_pass<R2, false, N_CT, R0 * R1, true>(a, ra, rb, has_b, bufB, nullptr, tw, R0 * R1, pacc);
            } else {
                stockham_pass<R1, false, N_CT, R0, true>(a, ra, rb, has_b, bufA, nullptr, tw, R0, pacc);
            }
            continue;
        } else {
            int ns = 1;
#pragma unroll 1
            for (int ps = 0; ps < a.n_pass; ++ps) {
                const int R = ps == 0 ? a.radix[0] : (ps == 1 ? a.radix[1] : (ps == 2 ? a.radix[2] : a.radix[3]));
                if (ps == 0) {
                    if (R == 16)     stockham_pass<16, true>(a, ra, rb, has_b, nullptr, dst, tw, 1);
                    else if (R == 8) stockham_pass<8, true>(a, ra, rb, has_b, nullptr, dst, tw, 1);
                    else             stockham_pass<4, true>(a, ra, rb, has_b, nullptr, dst, tw, 1);
                } else {
                    if (R == 16)     stockham_pass<16, false>(a, ra, rb, has_b, src, dst, tw, ns);
                    else if (R == 8) stockham_pass<8, false>(a, ra, rb, has_b, src, dst, tw, ns);
                    else             stockham_pass<4, false>(a, ra, rb, has_b, src, dst, tw, ns);
                }
                ns *= R;
                float2 *tmp = src; src = dst; dst = tmp;   // src now holds the newest data
                __syncthreads();
            }
        }
        const float2 *z = src;
        for (int m = tid; m <= nh; m += T) {
            const float2 p = z[pad16(m)], q = z[pad16((n - m) & (n - 1))];
            // X_A = (p + conj q)/2, X_B = (p - conj q)/(2i)
            const float ar = 0.5f * (p.x + q.x), ai = 0.5f * (p.y - q.y);
            const float br = 0.5f * (p.y + q.y), bi = 0.5f * (q.x - p.x);
            pw[m] += (double)(ar * ar + ai * ai) + (double)(br * br + bi * bi);
        }
    }
    if constexpr (N_CT > 0) {                              // output k = j + t ns of the last pass, j = tid < N / RL
        if (tid < N_CT / RL)
#pragma unroll
            for (int t = 0; t < RL; ++t) atomicAdd(a.acc + (REP ? (blockIdx.x % a.reps) * a.n_acc : 0) + tid + t * (N_CT / RL), pacc[t]);
        lya_publish_last_cta(a.acc, a.n_acc, a.host, a.ticket, REP ? a.reps : 1);
        return;
    }
    __syncthreads();
    for (int m = tid; m <= nh; m += T)
        if (pw[m] != 0.0) atomicAdd(a.acc + (REP ? (blockIdx.x % a.reps) * a.n_acc : 0) + m, pw[m]);
    lya_publish_last_cta(a.acc, a.n_acc, a.host, a.ticket, REP ? a.reps : 1);
}

// ---- one WARP per row pair, two passes, no CTA barrier (N1 x N2 points, multiples of 32; instantiated: 32 x 32) --------
// ncu on the kernel above (1024-pixel rows): issue slots 55 % busy, barrier stall 5.0 and long-scoreboard 3.0 cycles per
// issued instruction, half of the threads idle in the radix-16 passes; prefetching the next pair with cp.async changed
// nothing (1.30 -> 1.26 ms), so the limit is the pass -> barrier -> pass chain itself.  Here a warp owns a whole
// transform (Cooley-Tukey, n = n2 + N2 n1, k = k1 + N1 k2):
//   pass 1  lane holds x[n2 + N2 n1], n1 < N1, for its residues n2 = lane (+ 32): coalesced 128-byte loads, an N1-point
//           DFT in registers, the twiddles W_N^(n2 k1) from a per-CTA table [k1][n2], the result to the warp's private
//           exchange buffer [k1][n2] (row stride N2 + 1 float2: conflict-free both ways);
//   pass 2  lane holds Y[n2][k1], n2 < N2, for its k1 = lane (+ 32): an N2-point DFT in registers, |Z(k)|^2 added to
//           fp32 accumulators in registers -- flushed to the double device accumulators (atomicAdd) every 256 pairs and
//           at the end, so an fp32 accumulator never holds more than 256 terms.
// Only __syncwarp() orders the two passes; without the cp.async stage below every load of a pair (64 per lane at
// N = 1024) is in flight at once.
// mbarrier + 1-D bulk copy (TMA unit; SASS: SYNCS, UBLKCP): one lane moves a whole row pair, 8 N bytes, per instruction
__device__ __forceinline__ unsigned pw_smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(pw_smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(pw_smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(pw_smem_addr(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(pw_smem_addr(dst)), "l"(src), "r"(bytes), "r"(pw_smem_addr(bar)) : "memory");
}

template <int R, bool PACK>
__device__ __forceinline__ void dft_regs64(float2 (&v)[R])   // as dft_regs, twiddles W_64^q (R <= 64)
{
    constexpr float C[32] = {1.f, 0.99518472667219693f, 0.98078528040323043f, 0.95694033573220882f, 0.92387953251128674f,
        0.88192126434835505f, 0.83146961230254524f, 0.77301045336273699f, 0.70710678118654757f, 0.63439328416364549f,
        0.55557023301960229f, 0.47139673682599781f, 0.38268343236508984f, 0.29028467725446233f, 0.19509032201612833f,
        0.09801714032956077f, 0.f, -0.098017140329560645f, -0.19509032201612819f, -0.29028467725446216f,
        -0.38268343236508973f, -0.4713967368259977f, -0.55557023301960196f, -0.63439328416364538f, -0.70710678118654746f,
        -0.77301045336273699f, -0.83146961230254535f, -0.88192126434835494f, -0.92387953251128674f, -0.95694033573220882f,
        -0.98078528040323043f, -0.99518472667219682f};
    constexpr float S[32] = {0.f, 0.098017140329560604f, 0.19509032201612825f, 0.29028467725446233f, 0.38268343236508978f,
        0.47139673682599764f, 0.55557023301960218f, 0.63439328416364549f, 0.70710678118654746f, 0.77301045336273699f,
        0.83146961230254524f, 0.88192126434835494f, 0.92387953251128674f, 0.95694033573220894f, 0.98078528040323043f,
        0.99518472667219682f, 1.f, 0.99518472667219693f, 0.98078528040323043f, 0.95694033573220894f, 0.92387953251128674f,
        0.88192126434835505f, 0.83146961230254546f, 0.7730104533627371f, 0.70710678118654757f, 0.63439328416364549f,
        0.55557023301960218f, 0.47139673682599786f, 0.38268343236508989f, 0.29028467725446239f, 0.19509032201612861f,
        0.098017140329560826f};
#pragma unroll
    for (int len = R; len >= 2; len >>= 1) {
        const int half = len >> 1;
#pragma unroll
        for (int s = 0; s < R; s += len) {
#pragma unroll
            for (int p = 0; p < half; ++p) {
                const float2 a = v[s + p], b = v[s + p + half];
                v[s + p] = PACK ? cadd(a, b) : make_float2(a.x + b.x, a.y + b.y);
                const float2 d = PACK ? csub(a, b) : make_float2(a.x - b.x, a.y - b.y);
                const int q = p * (64 / len);              // W_len^p = exp(-2 pi i q / 64), q < 32
                if (q == 0)       v[s + p + half] = d;
                else if (q == 16) v[s + p + half] = make_float2(d.y, -d.x);          // times -i
                else              v[s + p + half] = cmul(d, make_float2(C[q], -S[q]));
            }
        }
    }
}

constexpr int PW_FLUSH = 256;                            // pairs between two flushes of the fp32 accumulators

// NT = N1 N2 is the transform a warp does in two passes.  SPLIT: rows of N = 2 NT pixels, by one radix-2 decimation
// in frequency at load time -- Z(2 k') = DFT_NT(z[m] + z[m + NT]), Z(2 k' + 1) = DFT_NT((z[m] - z[m + NT]) W_N^m) -- so
// the two halves are independent NT-point transforms whose outputs are final (no combining step): a TEAM of two warps
// shares one staged pair, warp h of the team takes half h, and only two 64-thread named barriers per pair tie them
// together (pair landed / pair read).  A serial version (one warp, both halves) fits only 8 warps per SM next to its
// 16 KiB stage buffers and measured 1.40 ms on 2048-pixel rows, no better than the CTA-per-pair kernel.
// STAGE (16-byte aligned flux; required by SPLIT): the NEXT pair streams into the stage buffer (ONE cp.async.bulk of 8 N
// bytes issued by one lane, completion counted on the unit's mbarrier)
// while the current one is transformed, so no warp waits out an HBM latency (1024-pixel rows: 0.99 -> 0.92 ms with
// LDGSTS, 0.88 ms with the bulk copy).
template <int N1, int N2, bool SPLIT, bool STAGE, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) flux_power_warp_kernel(const PowArgs a)
{
    constexpr int NT = N1 * N2, H = SPLIT ? 2 : 1, N = H * NT;
    constexpr int UNITS = WARPS / H;                     // row pairs in flight per CTA (a unit = a warp, or a team of two)
    constexpr int S1 = N2 / 32, S2 = N1 / 32;            // residues n2 (pass 1) / outputs k1 (pass 2) per lane
    constexpr int XS = N2 + 1;                           // exchange row stride [float2]
    static_assert(N1 % 32 == 0 && N2 % 32 == 0 && (STAGE || !SPLIT) && WARPS % H == 0 && UNITS <= 15, "unsupported plan");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int unit = SPLIT ? warp >> 1 : warp, h = SPLIT ? warp & 1 : 0;
    float2 *tw  = reinterpret_cast<float2 *>(smem_raw);  // [N1][N2]: W_NT^(n2 k1)
    float2 *tw2 = tw + NT;                               // SPLIT: [NT] inv_mean W_N^m
    float2 *ex  = tw2 + (SPLIT ? NT : 0) + warp * (N1 * XS);
    float *stg  = reinterpret_cast<float *>(tw2 + (SPLIT ? NT : 0) + WARPS * (N1 * XS)) + unit * (2 * N);
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(
        reinterpret_cast<float *>(tw2 + (SPLIT ? NT : 0) + WARPS * (N1 * XS)) + UNITS * (2 * N)) + unit;
    const bool issuer = STAGE && lane == 0 && h == 0;    // the one thread of a unit that talks to the copy unit
    auto stage = [&](size_t pair) {                      // rows 2 pair (and 2 pair + 1 if it exists): contiguous floats
        const unsigned bytes = (2 * pair + 1 < a.n_rows ? 2 * N : N) * (unsigned)sizeof(float);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the buffer was read through the generic proxy
        mbar_expect_tx(mbar, bytes);
        bulk_g2s(stg, a.flux + (2 * pair) * (size_t)N, bytes, mbar);
    };
    if (issuer) {
        mbar_init(mbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    auto unit_sync = [&]() {                             // the warps that share a stage buffer
        if (SPLIT) asm volatile("bar.sync %0, 64;" ::"r"(unit + 1) : "memory");
        else       __syncwarp();
    };
    for (int i = threadIdx.x; i < NT; i += WARPS * 32) {
        const int k1 = i / N2, n2 = i - k1 * N2;
        float sn, cs;
        sincospif(2.0f * (float)((k1 * n2) & (NT - 1)) / (float)NT, &sn, &cs);
        tw[i] = make_float2(cs, -sn);
        if (SPLIT) {
            sincospif(2.0f * (float)i / (float)N, &sn, &cs);
            tw2[i] = make_float2(cs * a.inv_mean, -sn * a.inv_mean);
        }
    }
    __syncthreads();
    float acc[S2][N2];
#pragma unroll
    for (int s = 0; s < S2; ++s)
#pragma unroll
        for (int t = 0; t < N2; ++t) acc[s][t] = 0.0f;
    double *mine = a.acc + (blockIdx.x % a.reps) * a.n_acc;   // this CTA's replica of the accumulators
    auto flush = [&]() {                                 // fp32 accumulators -> the device's doubles
#pragma unroll
        for (int s = 0; s < S2; ++s)
#pragma unroll
            for (int t = 0; t < N2; ++t) {               // transform output k' = k1 + N1 k2 is Z(H k' + h)
                atomicAdd(mine + H * ((lane + 32 * s) + N1 * t) + h, (double)acc[s][bitrev<N2>(t)]);
                acc[s][bitrev<N2>(t)] = 0.0f;
            }
    };
    const size_t n_pairs = (a.n_rows + 1) >> 1, step = (size_t)gridDim.x * UNITS;
    const float im = a.inv_mean;
    int since = 0;
    size_t pair = (size_t)blockIdx.x * UNITS + unit;
    if (issuer && pair < n_pairs) stage(pair);           // (the mbarrier was initialised before the __syncthreads above)
    unsigned phase = 0;
    for (; pair < n_pairs; pair += step) {
        const float *ra = STAGE ? stg : a.flux + (2 * pair) * (size_t)N, *rb = ra + N;
        const bool has_b = 2 * pair + 1 < a.n_rows;
        if (STAGE) {
            mbar_wait(mbar, phase);                      // this pair has landed (complete_tx on the unit's mbarrier)
            phase ^= 1u;
        }
#pragma unroll
        for (int s = 0; s < S1; ++s) {                   // pass 1 for residue n2 = lane + 32 s: points m = n2 + N2 t
            const int n2 = lane + 32 * s;
            float2 v[N1];
            if (!SPLIT) {
#pragma unroll
                for (int t = 0; t < N1; ++t) v[t].x = STAGE ? ra[n2 + N2 * t] : __ldcs(ra + n2 + N2 * t);
#pragma unroll
                for (int t = 0; t < N1; ++t) v[t].y = !has_b ? 0.0f : STAGE ? rb[n2 + N2 * t] : __ldcs(rb + n2 + N2 * t);
            } else {                                     // z[m] +- z[m + NT] of the raw fluxes (dF is applied below)
#pragma unroll
                for (int t = 0; t < N1; ++t) {
                    const int m = n2 + N2 * t;
                    const float xa = ra[m], ya = ra[m + NT], xb = has_b ? rb[m] : 0.0f, yb = has_b ? rb[m + NT] : 0.0f;
                    v[t] = h == 0 ? make_float2(xa + ya, xb + yb) : make_float2(xa - ya, xb - yb);
                }
            }
            if (STAGE && s == S1 - 1) {                  // the stage buffer has been read: fetch the next pair into it
                unit_sync();
                if (issuer && pair + step < n_pairs) stage(pair + step);
            }
            if (!SPLIT) {
#pragma unroll
                for (int t = 0; t < N1; ++t) v[t] = make_float2(fmaf(v[t].x, im, -1.0f), has_b ? fmaf(v[t].y, im, -1.0f) : 0.0f);
            } else if (h == 0) {
#pragma unroll
                for (int t = 0; t < N1; ++t) v[t] = make_float2(fmaf(v[t].x, im, -2.0f), has_b ? fmaf(v[t].y, im, -2.0f) : 0.0f);
            } else {
#pragma unroll
                for (int t = 0; t < N1; ++t) v[t] = cmul(v[t], tw2[n2 + N2 * t]);   // the -1 cancels; tw2 carries inv_mean
            }
            dft_regs64<N1, true>(v);
            ex[n2] = v[0];                               // k1 = 0: twiddle 1
#pragma unroll
            for (int k1 = 1; k1 < N1; ++k1) ex[k1 * XS + n2] = cmul(v[bitrev<N1>(k1)], tw[k1 * N2 + n2]);
        }
        __syncwarp();
#pragma unroll
        for (int s = 0; s < S2; ++s) {                   // pass 2 for output residue k1 = lane + 32 s
            const float2 *row = ex + (lane + 32 * s) * XS;
            float2 u[N2];
#pragma unroll
            for (int t = 0; t < N2; ++t) u[t] = row[t];
            dft_regs64<N2, true>(u);
#pragma unroll
            for (int t = 0; t < N2; ++t) acc[s][t] = fmaf(u[t].x, u[t].x, fmaf(u[t].y, u[t].y, acc[s][t]));
        }
        __syncwarp();                                    // the exchange buffer is free again
        if (++since == PW_FLUSH) { flush(); since = 0; }
    }
    // last flush through the CTA: every warp parks its fp32 accumulators in its own (now idle) exchange buffer, then the
    // CTA's threads add the warps' values per output in double, in a fixed order, and send ONE atomic per output and CTA
    // instead of one per warp -- all warps of the grid finish together and their atomics to the same N addresses serialise
    __syncthreads();
    float *park = reinterpret_cast<float *>(ex);         // [NT]: transform output k' = k1 + N1 k2
#pragma unroll
    for (int s = 0; s < S2; ++s)
#pragma unroll
        for (int t = 0; t < N2; ++t) park[(lane + 32 * s) + N1 * t] = acc[s][bitrev<N2>(t)];
    __syncthreads();
    const float *park0 = reinterpret_cast<const float *>(tw2 + (SPLIT ? NT : 0));
    for (int o = threadIdx.x; o < N; o += WARPS * 32) {  // output o = H k' + h comes from the warps H u + h, u < UNITS
        const float *src = park0 + (size_t)(o % H) * (2 * N1 * XS) + o / H;
        double sum = 0.0;
#pragma unroll
        for (int u = 0; u < UNITS; ++u) sum += (double)src[(size_t)u * H * (2 * N1 * XS)];
        atomicAdd(mine + o, sum);
    }
    lya_publish_last_cta(a.acc, a.n_acc, a.host, a.ticket, a.reps);
}

// The same design for SHORT rows (256 and 512 pixels = N1 x 32 with N1 = 8, 16): a warp step takes a BUNDLE of
// PPW = 32 / N1 consecutive row pairs -- 1024 complex points again, one bulk copy of 8 KiB -- so that the second pass
// still has a 32-point DFT for every lane: pass 1 runs PPW times (all lanes, an N1-point DFT each), pass 2 once, lane
// q N1 + k1 transforming output residue k1 of pair q.  Lanes of different pairs add into the same accumulators at flush.
template <int N1, bool STAGE, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) flux_power_warp_short_kernel(const PowArgs a)
{
    constexpr int N = N1 * 32, PPW = 32 / N1, RPB = 2 * PPW, XS = 33;   // RPB: rows per bundle
    static_assert(N1 == 8 || N1 == 16, "unsupported plan");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float2 *tw = reinterpret_cast<float2 *>(smem_raw);   // [N1][32]: W_N^(n2 k1)
    float2 *ex = tw + N + warp * (32 * XS);              // row q N1 + k1, column n2
    float *stg = reinterpret_cast<float *>(tw + N + WARPS * (32 * XS)) + warp * (RPB * N);
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(
        reinterpret_cast<float *>(tw + N + WARPS * (32 * XS)) + WARPS * (RPB * N)) + warp;
    const bool issuer = STAGE && lane == 0;
    auto stage = [&](size_t bundle) {                    // up to RPB consecutive rows: contiguous floats
        const size_t row0 = bundle * RPB;
        const unsigned rows = a.n_rows - row0 < (size_t)RPB ? (unsigned)(a.n_rows - row0) : (unsigned)RPB;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(mbar, rows * N * (unsigned)sizeof(float));
        bulk_g2s(stg, a.flux + row0 * N, rows * N * (unsigned)sizeof(float), mbar);
    };
    if (issuer) {
        mbar_init(mbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < N; i += WARPS * 32) {
        const int k1 = i >> 5, n2 = i & 31;
        float sn, cs;
        sincospif(2.0f * (float)((k1 * n2) & (N - 1)) / (float)N, &sn, &cs);
        tw[i] = make_float2(cs, -sn);
    }
    __syncthreads();
    float acc[32];
#pragma unroll
    for (int t = 0; t < 32; ++t) acc[t] = 0.0f;
    double *mine = a.acc + (blockIdx.x % a.reps) * a.n_acc;
    const int k1l = lane & (N1 - 1);                     // pass 2: this lane's output residue (of pair lane / N1)
    auto flush = [&]() {
#pragma unroll
        for (int t = 0; t < 32; ++t) {                   // output k = k1 + N1 k2
            atomicAdd(mine + k1l + N1 * t, (double)acc[bitrev<32>(t)]);
            acc[bitrev<32>(t)] = 0.0f;
        }
    };
    const size_t n_bundles = (a.n_rows + RPB - 1) / RPB, step = (size_t)gridDim.x * WARPS;
    const float im = a.inv_mean;
    int since = 0;
    size_t bundle = (size_t)blockIdx.x * WARPS + warp;
    if (issuer && bundle < n_bundles) stage(bundle);
    unsigned phase = 0;
    for (; bundle < n_bundles; bundle += step) {
        const size_t row0 = bundle * RPB;
        const float *base = STAGE ? stg : a.flux + row0 * N;
        if (STAGE) {
            mbar_wait(mbar, phase);
            phase ^= 1u;
        }
        float2 v[PPW][N1];
#pragma unroll
        for (int q = 0; q < PPW; ++q) {
            const bool has_a = row0 + 2 * q < a.n_rows, has_b = row0 + 2 * q + 1 < a.n_rows;
            const float *ra = base + (2 * q) * N, *rb = ra + N;
#pragma unroll
            for (int t = 0; t < N1; ++t) {
                const float xa = !has_a ? 0.0f : STAGE ? ra[lane + 32 * t] : __ldcs(ra + lane + 32 * t);
                const float xb = !has_b ? 0.0f : STAGE ? rb[lane + 32 * t] : __ldcs(rb + lane + 32 * t);
                v[q][t] = make_float2(has_a ? fmaf(xa, im, -1.0f) : 0.0f, has_b ? fmaf(xb, im, -1.0f) : 0.0f);
            }
        }
        if (STAGE) {                                     // the stage buffer has been read: fetch the next bundle into it
            __syncwarp();
            if (issuer && bundle + step < n_bundles) stage(bundle + step);
        }
#pragma unroll
        for (int q = 0; q < PPW; ++q) {                  // pass 1 of pair q: an N1-point DFT per lane (n2 = lane)
            dft_regs64<N1, true>(v[q]);
            float2 *e = ex + (q * N1) * XS + lane;
            e[0] = v[q][0];
#pragma unroll
            for (int k1 = 1; k1 < N1; ++k1) e[k1 * XS] = cmul(v[q][bitrev<N1>(k1)], tw[k1 * 32 + lane]);
        }
        __syncwarp();
        {                                                // pass 2: row `lane` of the exchange buffer
            const float2 *row = ex + lane * XS;
            float2 u[32];
#pragma unroll
            for (int t = 0; t < 32; ++t) u[t] = row[t];
            dft_regs64<32, true>(u);
#pragma unroll
            for (int t = 0; t < 32; ++t) acc[t] = fmaf(u[t].x, u[t].x, fmaf(u[t].y, u[t].y, acc[t]));
        }
        __syncwarp();
        if (++since == PW_FLUSH) { flush(); since = 0; }
    }
    __syncthreads();                                     // last flush through the CTA, as in flux_power_warp_kernel
    float *park = reinterpret_cast<float *>(ex);         // [PPW][N]: lanes of different pairs own the same outputs
#pragma unroll
    for (int t = 0; t < 32; ++t) park[(lane / N1) * N + k1l + N1 * t] = acc[bitrev<32>(t)];
    __syncthreads();
    const float *park0 = reinterpret_cast<const float *>(tw + N);
    for (int o = threadIdx.x; o < N; o += WARPS * 32) {
        double sum = 0.0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w)
#pragma unroll
            for (int q = 0; q < PPW; ++q) sum += (double)park0[(size_t)w * (2 * 32 * XS) + q * N + o];
        atomicAdd(mine + o, sum);
    }
    lya_publish_last_cta(a.acc, a.n_acc, a.host, a.ticket, a.reps);
}

}  // namespace

extern "C" lya_status lya_flux_power_rows(lya_ctx *ctx, size_t n_rows, int32_t n_pix, double dv_kms,
                                          const float *flux, double mean_flux, double *power)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!flux || ((uintptr_t)flux & 3) || !power) return lya_fail(ctx, LYA_EINVAL, "lya_flux_power_rows: null or misaligned pointer");
    if (n_rows < 1 || !(dv_kms > 0.0) || !(mean_flux > 0.0))
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_power_rows: n_rows >= 1, dv > 0 and mean_flux > 0 required");
    int log2n = 0;
    while ((1 << log2n) < n_pix) ++log2n;
    if (n_pix < 8 || n_pix > 8192 || (1 << log2n) != n_pix)
        return lya_fail(ctx, LYA_EINVAL, "lya_flux_power_rows: n_pix must be a power of two in [8, 8192]");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));
    const int nk = n_pix / 2 + 1;
    const bool folded = n_pix >= 256 && n_pix <= 4096;     // compile-time plans leave sum |Z(k)|^2, k < n_pix, to fold here
    const int n_acc = folded ? n_pix : nk;
    PowArgs a;
    memset(&a, 0, sizeof(a));
    a.flux = flux; a.n_rows = n_rows; a.n = n_pix; a.log2n = log2n;
    a.inv_mean = (float)(1.0 / mean_flux); a.acc = ctx->d_stats;
    a.host = ctx->h_pinned + LYA_PINNED_STATS; a.ticket = ctx->d_sched + 4; a.n_acc = n_acc; a.reps = n_rows * (size_t)n_pix <= ((size_t)1 << 25) ? lya_stats_replicas(n_acc, n_rows * (size_t)n_pix, 4) : 1;   // measured: 512^3 is slower with replicas
    // radices of the passes (log2: 4, 3, 2), largest first
    static const int plan[14][4] = {{0}, {0}, {0}, {3}, {4}, {3, 2}, {3, 3}, {4, 3}, {4, 4}, {3, 3, 3}, {4, 3, 3},
                                    {4, 4, 3}, {4, 4, 4}, {4, 4, 3, 2}};
    for (int i = 0; i < 4 && plan[log2n][i]; ++i) a.radix[a.n_pass++] = 1 << plan[log2n][i];
    const int npad = n_pix + (n_pix >> 4) + 1;
    size_t smem = (size_t)(nk + 1) * sizeof(double) + 2 * (size_t)npad * sizeof(float2) + (size_t)(n_pix / 2) * sizeof(float2);
    int threads = n_pix / 8;
    threads = threads < 32 ? 32 : (threads > 256 ? 256 : threads);
    void (*kern)(const PowArgs) = n_pix == 256 ? flux_power_kernel<256> : n_pix == 512 ? flux_power_kernel<512>
                                : n_pix == 1024 ? flux_power_kernel<1024> : n_pix == 2048 ? flux_power_kernel<2048>
                                : n_pix == 4096 ? flux_power_kernel<4096> : flux_power_kernel<0>;
    if (a.reps > 1)                                        // short launch: replicated accumulators
        kern = n_pix == 256 ? flux_power_kernel<256, true> : n_pix == 512 ? flux_power_kernel<512, true>
             : n_pix == 1024 ? flux_power_kernel<1024, true> : n_pix == 2048 ? flux_power_kernel<2048, true>
             : n_pix == 4096 ? flux_power_kernel<4096, true> : flux_power_kernel<0, true>;
    // rows of 1024 / 2048 pixels: one warp per row pair (flux_power_warp_kernel); 2048 needs 16-byte aligned flux
    int warp_kernel = 0;
    const bool al16 = ((uintptr_t)flux & 15) == 0;
    if (n_pix == 1024) {
        kern = al16 ? flux_power_warp_kernel<32, 32, false, true, 4, 3> : flux_power_warp_kernel<32, 32, false, false, 4, 3>;
        warp_kernel = 4;
        threads = 4 * 32;
        smem = (size_t)1024 * sizeof(float2) + 4 * (size_t)32 * 33 * sizeof(float2) + (al16 ? 4 * 2 * (size_t)1024 * sizeof(float) : 0) + 4 * sizeof(unsigned long long);
    } else if (n_pix == 256 || n_pix == 512) {             // bundles of 4 / 2 row pairs per warp step
        kern = n_pix == 256 ? (al16 ? flux_power_warp_short_kernel<8, true, 4, 3> : flux_power_warp_short_kernel<8, false, 4, 3>)
                            : (al16 ? flux_power_warp_short_kernel<16, true, 4, 3> : flux_power_warp_short_kernel<16, false, 4, 3>);
        warp_kernel = 4 * (1024 / n_pix);                  // row pairs per CTA step
        threads = 4 * 32;
        smem = (size_t)n_pix * sizeof(float2) + 4 * (size_t)32 * 33 * sizeof(float2) + (al16 ? 4 * 2 * (size_t)1024 * sizeof(float) : 0) + 4 * sizeof(unsigned long long);
    } else if (n_pix == 2048 && al16) {                    // 6 teams of two warps, one CTA per SM
        kern = flux_power_warp_kernel<32, 32, true, true, 12, 1>;
        warp_kernel = 6;
        smem = 2 * (size_t)1024 * sizeof(float2) + 12 * (size_t)32 * 33 * sizeof(float2) + 6 * 2 * (size_t)2048 * sizeof(float) + 6 * sizeof(unsigned long long);
        threads = 12 * 32;
    }
    int per_sm = 0;
    lya_status st = lya_kernel_occupancy(ctx, (const void *)kern, threads, smem, &per_sm);
    if (st != LYA_OK) return st;
    if (per_sm < 1) return lya_fail(ctx, LYA_ECUDA, "flux_power_kernel: zero occupancy");
    const size_t n_pairs = warp_kernel ? ((n_rows + 1) / 2 + warp_kernel - 1) / warp_kernel : (n_rows + 1) / 2, cap = (size_t)ctx->sm_count * per_sm;
    st = lya_stats_begin(ctx, n_acc);
    if (st != LYA_OK) return st;
    kern<<<(int)(n_pairs < cap ? n_pairs : cap), threads, smem, ctx->stream>>>(a);   // the last CTA writes the totals to a.host
    ctx->launches++;
    st = lya_stats_end(ctx);
    if (st != LYA_OK) return st;
    const double *host = a.host;
    const double scale = dv_kms / ((double)n_pix * (double)n_rows);        // V / N^2 / n_rows
    for (int m = 0; m < nk; ++m)                                           // |X_A|^2 + |X_B|^2 = (|Z(m)|^2 + |Z(N-m)|^2) / 2
        power[m] = (folded ? 0.5 * (host[m] + host[(n_pix - m) & (n_pix - 1)]) : host[m]) * scale;
    return LYA_OK;
}
