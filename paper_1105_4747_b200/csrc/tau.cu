// tau.cu -- S2 + S3: redshift-space optical depth along every sightline (Eq.6).
//
//   tau(i) = K sum_j nHI(j)/b(j) exp(-((v_H(i) - u(j))/b(j))^2),   u(j) = v_H(j) + v_pec(j),
//   v_H(i) - v_H(j) = (i-j) dv, nearest periodic image (period V = N dv; reading C7).
//
// Every (i,j) pair is evaluated (N^2 per sightline): the kernel is bound by MUFU.EX2 (16 /clk/SM, measured),
// and on sm_100a every extra FP32 instruction per pair costs MUFU rate long before the issue limit
// ("pair loop"), so the pair body is packed FP32 on two SOURCES at a time -- 1.9 issue slots
// + 1 MUFU per pair (see "the staged layout" below for the pairing) -- and one exponential in eight is a packed
// polynomial on the otherwise half-idle FMA pipe (ex2_poly2_neg), which lifts the bound to 16 / (1 - 1/8) per clk and SM:
//
//   staged per source cell j (once per sightline, in shared memory, four floats):
//       m_j = j + P_j          P_j = round(v_pec/dv), reduced mod N          (integer-valued float, exact)
//       w_j = (dv/b_j) sqrt(log2 e)                                          (so exp(-x^2) = ex2(-(x')^2))
//       g_j = -f_j w_j         f_j = v_pec/dv - round(v_pec/dv)  in [-1/2,1/2] (exact fma residual)
//       a_j = K 1e-5 nHI_j / b_j                                             (line-centre amplitude)
//   a thread owns R CONSECUTIVE pixels i_0 .. i_0+R-1; per source cell:
//       E   = (i_0 + R/2) - m_j (exact) ;  x_ref = fma(E, w_j, g_j)          (FADD2 + FFMA2 per 2 R pairs)
//       x_r = fma(r - R/2, w_j, x_ref)                                       (1 FFMA2 / FADD2, none for r = R/2)
//       e   = ex2(-x_r * x_r)  ;  acc_r = fma(a_j, e, acc_r)                 (FMUL2 + 2 MUFU + FFMA2)
//
// Keeping the integer part of the pixel separation exact is what holds the error at ~1e-6 for N = 2048
// (forming u_j and v_i in fp32 km/s loses 3 digits there); x_ref is at most R/2 cells away
// from the pixel it serves, so for every pair that contributes its rounding error is ulp(|x| + 2 w)/2.
//
// Periodic wrap without per-pair work: a warp owns a tile of 32*R consecutive pixels and walks the sources
// in UNWRAPPED order jj = c - N/2 ... c + N/2 - 1 around the tile centre c (two contiguous index segments),
// so i - jj is already the nearest image for every pair that can contribute.  That is valid when, for every
// source of the sightline, (N/2 - 16R - |P_j| - 1/2) w_j >= 11.3, i.e. a pair whose chosen image is not the
// nearest has ex2(-x^2) == 0 in fp32 (and < 2^-127 of a_j in the oracle's double).  The staging pass checks
// the condition; a sightline that fails it (tiny N, |v_pec| of order V) takes the general loop with a
// per-pair image choice.  Both loops evaluate all N^2 pairs.
//
// Mapping, sightlines along x (contiguous rows): a GROUP of G warps (G = 1 unless the row is too long for
// enough groups to fit in shared memory) owns one sightline at a time: it stages the row (four consecutive cells
// per thread from 128-bit loads) straight into its private cell slots, syncs only itself (named barrier / __syncwarp),
// sums its tiles and stores R consecutive tau values per lane (128-bit).  Groups never wait for each other,
// so the MUFU pipe always has warps in the pair loop while others stage; rows are handed out by a global
// atomic counter, which removes the wave-quantisation tail of a static partition (65,536 rows over
// ~6,000 resident warps would lose 8 %).
// Sightlines along y / z: a CTA gathers 8 (or fewer) neighbouring x at a time so that global accesses stay
// 32- or 16-byte segments, its 8 warps sum (sightline, tile) items, and tau goes back through a shared-memory
// tile; batches come from the same atomic counter.
//
// Variants behind lya_tau_sightlines_opt (template flags, same kernels): FUSED applies S1 (gas_cell.h) to delta
// while staging, so n_HI and b never exist in memory; WIN (LYA_TAU_WINDOWED) lets every lane walk only the
// 2 W + R sources around its own pixels (tile_window, over a row staged unwrapped with a periodic halo) --
// bit-identical output, 3 % of the pairs at N = 1024.  The epilogue can leave per-sightline moments sum tau^k for S4.
#include "gas_cell.h"
#include "lya_internal.h"

namespace {

constexpr int   TAU_WARPS   = 8;       // strided kernel: warps per CTA
constexpr int   TAU_THREADS = TAU_WARPS * 32;
constexpr float TAU_XCUT    = 11.3f;   // ex2.approx.ftz(-11.3^2) = 2^-127.7 is below 2^-126: flushed to exactly 0

struct TauArgs {
    const float *n_hi, *b, *v;
    float       *tau;
    int          n;           // pixels per sightline
    int          tiles;       // pixel tiles of 32*R per sightline
    int          vec;         // x-axis: tau rows are 16-byte aligned and n % 4 == 0
    int          vec_in;      // x-axis: the input rows are (128-bit staging loads)
    int          bsl;         // strided: x-width of a gathered batch (power of 2)
    int          bshift;      // log2(bsl)
    int          cstride;     // strided: float4 cells per staged sightline (n + pad)
    int          tstride;     // strided: floats per sightline of the tau tile (tiles*32*R + pad)
    long long    n_sl;        // x-axis: number of sightlines (rows)
    long long    n_batches;   // strided: number of gathered batches
    unsigned int *sched;      // [0] next row / batch to hand out; zeroed by the host before every launch
    // strided modes (axis 1, 2)
    int          nx;          // x extent
    int          nxb;         // ceil(nx / bsl)
    long long    outer_stride; // elements between consecutive "outer" indices (axis 1: ny*nx per iz; axis 2: nx per iy)
    long long    stride;      // elements between consecutive pixels of a sightline
    float        inv_dv_hi, inv_dv_lo;   // 1 / dv [s/km] as an fp32 pair (hi + lo = the double value)
    float        amp_scale;   // K * 1e-5  [so that a_j is dimensionless]
    float        w_scale;     // dv * sqrt(log2 e) [km/s]
    float        inv_n, n_f;  // 1/N, N
    float        xcut_over_w; // TAU_XCUT / w_scale: TAU_XCUT / w_j = b_j * xcut_over_w
    GasK         gas;         // FUSED (LYA_TAU_FROM_DENSITY): n_hi points at delta, S1 is done while staging
    unsigned long long *pairs; // device counter of (i,j) pairs evaluated
    double      *rowm;        // [sightline][5] plain moments sum_i tau_i^k, k = 0..4, of every sightline written (or NULL):
                              // S4's first pass (A = 0) without re-reading tau -- lya_normalize_mean_flux_rows
};

__device__ __forceinline__ float ex2_ftz(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// 1 / x to 1 ulp (MUFU.RCP) -- the IEEE division's slow-path branch kept the staging loop's loads from being batched
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// round to nearest integer on the FP32 pipe (valid for |x| < 2^22; MUFU/XU-pipe FRND would compete with ex2)
__device__ __forceinline__ float round_magic(float x)
{
    const float big = 12582912.0f;                     // 1.5 * 2^23
    return __fsub_rn(__fadd_rn(x, big), big);
}

// One source cell -> staged float4 (m, w, g, a).  Returns the cell's REACH in pixels, 11.3 / w_j + |P_j| + 1/2:
// a pixel further than that from the (unwrapped) cell index gets ex2(-x^2) == 0 exactly from it.  The maximum
// over a sightline decides between the fast and the general loop and sets the window of LYA_TAU_WINDOWED.
// All fp32: p = v_pec/dv is split as P + f with P = round(v * inv_dv_hi) and f = fma(v, inv_dv_hi, -P) +
// v * inv_dv_lo -- the fma forms the residual of the exact 48-bit product with ONE rounding of a number
// below 1, so f carries an absolute error < 1e-7 pixel however large P is.  Precondition |v_pec| < 2^22 dv
// (4e6 pixels; beyond it P is no longer an integer: the reach is set to +inf, which sends the sightline to the
// general path with a meaningless but finite displacement).  No FP64 and, apart from one reciprocal, no
// XU-pipe instruction (MUFU.RCP: 1 / b to 1 ulp).  jf = (float)j.  Reading C11: +v -> higher pixel index.
__device__ __forceinline__ float stage_cell(const TauArgs &a, float jf, float nh, float bb, float vv, float4 &out)
{
    const float P  = round_magic(vv * a.inv_dv_hi);
    const float f  = fmaf(vv, a.inv_dv_lo, fmaf(vv, a.inv_dv_hi, -P));
    // integer displacement reduced to [-N/2, N/2]; at an exact half-way point either image is nearest
    const float Pr = fmaf(-a.n_f, round_magic(P * a.inv_n), P);
    const float ib = rcp_approx(bb);
    const float w  = a.w_scale * ib;
    out.x = jf + Pr;
    out.y = w;
    out.z = -f * w;
    out.w = (a.amp_scale * nh) * ib;
    const float reach = fmaf(bb, a.xcut_over_w, fabsf(Pr) + 0.5078125f);   // 1/2 for |f|, 2^-7 for the roundings here
    return (fabsf(P) < 4194304.0f && reach >= 0.0f) ? reach : __int_as_float(0x7f800000);   // NaN -> +inf
}

template <bool FUSED>
__device__ __forceinline__ float stage_from_global(const TauArgs &a, float jf, size_t g, float4 &out)
{
    float nh, bb;
    if (FUSED) gas_cell(a.gas, __ldcs(a.n_hi + g), nh, bb);            // n_hi points at delta
    else { nh = __ldcs(a.n_hi + g); bb = __ldcs(a.b + g); }
    return stage_cell(a, jf, nh, bb, __ldcs(a.v + g), out);
}

// Four consecutive cells j .. j + 3 from 128-bit loads (rows 16-byte aligned, n % 4 == 0): a quarter of the load and
// address instructions, and -- with no branch in stage_cell -- the compiler issues all loads of an unrolled batch before
// the first conversion, so a thread waits for global memory once per batch instead of once per cell.
template <bool FUSED>
__device__ __forceinline__ void load4(const TauArgs &a, size_t g, float4 &nh, float4 &bb, float4 &vv)
{
    nh = __ldcs(reinterpret_cast<const float4 *>(a.n_hi + g));         // FUSED: delta
    if (!FUSED) bb = __ldcs(reinterpret_cast<const float4 *>(a.b + g));
    vv = __ldcs(reinterpret_cast<const float4 *>(a.v + g));
}
template <bool FUSED>
__device__ __forceinline__ float stage4(const TauArgs &a, float jf, float4 nh, float4 bb, const float4 &vv, float4 (&out)[4])
{
    if (FUSED) {
        const float4 d = nh;
        gas_cell(a.gas, d.x, nh.x, bb.x); gas_cell(a.gas, d.y, nh.y, bb.y);
        gas_cell(a.gas, d.z, nh.z, bb.z); gas_cell(a.gas, d.w, nh.w, bb.w);
    }
    float reach = stage_cell(a, jf, nh.x, bb.x, vv.x, out[0]);
    reach = fmaxf(reach, stage_cell(a, jf + 1.0f, nh.y, bb.y, vv.y, out[1]));
    reach = fmaxf(reach, stage_cell(a, jf + 2.0f, nh.z, bb.z, vv.z, out[2]));
    return fmaxf(reach, stage_cell(a, jf + 3.0f, nh.w, bb.w, vv.w, out[3]));
}

// ---- the staged layout: sources in PAIRS.  Cells 2p and 2p + 1 of a row share two float4 slots,
//     slot 2p     A = (m_2p, m_2p+1, w_2p, w_2p+1)        slot 2p + 1   B = (g_2p, g_2p+1, a_2p, a_2p+1)
// so that an LDS.128 of A and one of B hand the pair loop (m, m'), (w, w'), (g, g'), (a, a') as aligned 64-bit register
// pairs: the loop body is packed FP32 (sub/fma/mul.rn.f32x2: FADD2, FFMA2, FMUL2) on two SOURCES at a time -- for four
// pixels per lane 23 issue slots per 8 pairs instead of 36, which is what the windowed variant, short of issue slots,
// needs (profiles/r2_ncu_tau_windowed.md); each f32x2 lane is the scalar operation, bit for bit.  Every pixel keeps an
// (even sources, odd sources) pair of partial sums, added at the end; the full and the windowed walks both start at an
// even unwrapped source index, so they add the same terms in the same order and stay bit-identical (the window needs
// n % 4 == 0: whole pad groups in the halo; other rows take the full walk).
// Slots are stored at cpos(slot): plain for the full sum (every lane reads the same slot: broadcast).  For
// LYA_TAU_WINDOWED, where lane k reads slot s0 + R k, the row is stored UNWRAPPED with a periodic halo of TAU_HALO
// cells on either side (slot j + TAU_HALO holds slot j; the halo copies carry m -/+ N, so a walk across the ends
// needs no wrap logic at all) and with one pad slot per R slots, s + s / R: the lanes of an LDS.128 phase then sit
// (R + 1) float4 apart, and R + 1 being odd the eight of them fall into the eight different 16-byte bank groups
// (R = 1 needs no pad: neighbouring lanes share a pair).
constexpr int TAU_HALO = 64;           // multiple of 4; a sightline whose window does not fit takes the full loops

typedef unsigned long long f32x2;      // two packed floats (lo, hi) in one 64-bit register pair
__device__ __forceinline__ f32x2 pk(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpk(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

template <bool WIN, int R> __device__ __forceinline__ int cpos(int j)
{
    if (!WIN) return j;
    const int s = j + TAU_HALO;
    return R > 1 ? s + (R == 2 ? (s >> 1) : (s >> 2)) : s;
}
template <int R> __host__ __device__ constexpr int crow_len(int n, bool win)        // slots of one staged row
{
    const int ne = (n + 1) & ~1;                          // an odd row gets a dummy last cell (amplitude 0)
    return !win ? ne : (R > 1 ? (ne + 2 * TAU_HALO) + (R == 2 ? ((ne + 2 * TAU_HALO) >> 1) : ((ne + 2 * TAU_HALO) >> 2)) + 1
                              : ne + 2 * TAU_HALO);
}

// one staged cell -> its half of the pair's two slots (scalar stores: the strided gather and unaligned rows)
template <bool WIN, int R>
__device__ __forceinline__ void put_cell(float4 *cs, int j, const float4 &q)
{
    float *fa = reinterpret_cast<float *>(cs + cpos<WIN, R>(j & ~1)) + (j & 1);
    float *fb = reinterpret_cast<float *>(cs + cpos<WIN, R>((j & ~1) + 1)) + (j & 1);
    fa[0] = q.x; fa[2] = q.y; fb[0] = q.z; fb[2] = q.w;
}
// four consecutive cells j .. j + 3 (j % 4 == 0) -> four slots, 128-bit stores
template <bool WIN, int R>
__device__ __forceinline__ void put_cells4(float4 *cs, int j, const float4 (&q)[4])
{
    cs[cpos<WIN, R>(j)]     = make_float4(q[0].x, q[1].x, q[0].y, q[1].y);
    cs[cpos<WIN, R>(j + 1)] = make_float4(q[0].z, q[1].z, q[0].w, q[1].w);
    cs[cpos<WIN, R>(j + 2)] = make_float4(q[2].x, q[3].x, q[2].y, q[3].y);
    cs[cpos<WIN, R>(j + 3)] = make_float4(q[2].z, q[3].z, q[2].w, q[3].w);
}
// an odd row's dummy cell n: amplitude 0, finite width, so the pair it shares with cell n - 1 is harmless
template <bool WIN, int R>
__device__ __forceinline__ void put_dummy(float4 *cs, int n)
{
    if (n & 1) put_cell<WIN, R>(cs, n, make_float4(0.0f, 1.0f, 0.0f, 0.0f));
}
template <bool WIN, int R>
__device__ __forceinline__ float4 get_cell(const float4 *cs, int j)
{
    const float *fa = reinterpret_cast<const float *>(cs + cpos<WIN, R>(j & ~1)) + (j & 1);
    const float *fb = reinterpret_cast<const float *>(cs + cpos<WIN, R>((j & ~1) + 1)) + (j & 1);
    return make_float4(fa[0], fa[2], fb[0], fb[2]);
}

// LYA_TAU_WINDOWED: after the row is staged (and the group has synchronised), fill the halo: slot -t is slot N - t
// with m - N, slot N - 1 + t is slot t - 1 with m + N (t = 1 .. TAU_HALO); only the A slots (even) carry m.  N % 4 == 0
// here (tile_any), so source and destination slots have the same parity.  Rows shorter than the halo never take
// the window, so they skip this.
template <int R>
__device__ __forceinline__ void fill_halo(float4 *cs, int n, float n_f, int t0, int nthreads)
{
    if (n < TAU_HALO || (n & 3)) return;
    for (int t = t0; t < 2 * TAU_HALO; t += nthreads) {
        const bool left = t < TAU_HALO;
        const int src = left ? n - TAU_HALO + t : t - TAU_HALO;
        const int dst = left ? t - TAU_HALO : n + t - TAU_HALO;
        float4 q = cs[cpos<true, R>(src)];
        if (!(t & 1)) {                                   // exact: integer-valued floats far below 2^24
            q.x += left ? -n_f : n_f;
            q.y += left ? -n_f : n_f;
        }
        cs[cpos<true, R>(dst)] = q;
    }
}

// 2^(-q) for q >= 0 on the FMA pipe, two values at a time (degree-5 minimax polynomial on the fractional part, relative
// error 2.3e-7 in fp32 -- MUFU.EX2's own is 2^-22 = 2.4e-7 -- and the exponent put in by an integer multiply-add).
// q >= 127.5 gives exactly 0 (the scale factor's exponent is clamped), which is all the windowed variant relies on:
// the terms it skips have q >= 127.69.
__device__ __forceinline__ f32x2 ex2_poly2_neg(f32x2 q2)                 // 2^(-q), q >= 0
{
    const f32x2 magic = pk(12582912.0f, 12582912.0f);             // 1.5 * 2^23
    const f32x2 tn = sub2(magic, q2);                             // low mantissa bits = rint(-q)
    const f32x2 h  = add2(q2, sub2(tn, magic));                   // q + rint(-q) = -(fractional part) in [-1/2, 1/2], exact
    f32x2 p = fma2(pk(-1.327647245e-03f, -1.327647245e-03f), h, pk(9.675540961e-03f, 9.675540961e-03f));   // odd signs flipped
    p = fma2(p, h, pk(-5.550713092e-02f, -5.550713092e-02f));
    p = fma2(p, h, pk(2.402212024e-01f, 2.402212024e-01f));
    p = fma2(p, h, pk(-6.931469440e-01f, -6.931469440e-01f));
    p = fma2(p, h, pk(1.000000119e+00f, 1.000000119e+00f));
    float n0, n1;
    unpk(tn, n0, n1);
    // scale = 2^max(n, -127): bits (n + 127) << 23 with n + 127 = bits(tn) - (0x4B400000 - 127), clamped at 0 -> 0.0f
    const int k0 = max(__float_as_int(n0), 0x4B400000 - 127), k1 = max(__float_as_int(n1), 0x4B400000 - 127);
    const float s0 = __int_as_float((k0 - (0x4B400000 - 127)) << 23), s1 = __int_as_float((k1 - (0x4B400000 - 127)) << 23);
    return mul2(p, pk(s0, s1));
}

// Two sources (one pair of slots) against the R pixels of a lane: cref2 = (c, c) with c the reference pixel's
// (unwrapped) index, so E = c - m is the exact integer separation; acc2[r] = (sum over even, sum over odd sources).
// POLY: the exponentials of the lane's LAST pixel go to the FMA pipe (ex2_poly2) instead of the MUFU pipe.  The walks
// set POLY on every second source pair (odd pair index, an absolute property of the pair), so one exponential in
// eight leaves the pipe that bounds the kernel; the packed loop has the issue slots and the FMA cycles to spare
// (DESIGN.md section 6).  R < 4 (rows shorter than 128 pixels: launch-bound) never takes it.
template <int R, bool POLY>
__device__ __forceinline__ void pair_step(const float4 &A, const float4 &B, f32x2 cref2, f32x2 (&acc2)[R])
{
    constexpr int RH = R / 2;
    const f32x2 m2 = pk(A.x, A.y), w2 = pk(A.z, A.w), g2 = pk(B.x, B.y), a2 = pk(B.z, B.w);
    const f32x2 xr = fma2(sub2(cref2, m2), w2, g2);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        // x_r = (r - RH) w + x_ref, one rounding: +-1 as a packed add / subtract, the others as a packed fma
        const f32x2 x = (r == RH) ? xr : (r == RH + 1) ? add2(xr, w2) : (r == RH - 1) ? sub2(xr, w2)
                                       : fma2(pk((float)(r - RH), (float)(r - RH)), w2, xr);
        if (POLY && R >= 4 && r == R - 1) {
            acc2[r] = fma2(a2, ex2_poly2_neg(mul2(x, x)), acc2[r]);
        } else {
            float t0, t1;
            unpk(mul2(x, x), t0, t1);
            acc2[r] = fma2(a2, pk(ex2_ftz(-t0), ex2_ftz(-t1)), acc2[r]);
        }
    }
}

// Fast path, full sum: unwrapped walk over all n sources jj = start .. start + n - 1 around the tile centre (at
// most one wrap), no per-pair image logic.  Lane owns pixels i0 + lane*R + r.  The walk is in whole pairs of slots: a
// segment that would begin or end inside a pair takes the whole pair -- the extra source is then met at an image
// n/2 - 16R + 1 or more pixels from every pixel of the tile, where the validity condition makes its term exactly 0 --
// and an odd row's last pair holds a dummy cell of amplitude 0.  For n % 4 == 0 (the window's requirement) nothing is
// extra: start, j0 and n are even.
template <int R, bool PAD>
__device__ __forceinline__ void tile_fast(const float4 *__restrict__ cs, int n, int i0, int lane, float (&acc)[R])
{
    constexpr int RH = R / 2;                          // reference pixel of the lane
    const int start = i0 + 16 * R - (n >> 1);          // first unwrapped source index
    int j0 = start % n;
    if (j0 < 0) j0 += n;                               // slot holding jj = start
    const int off = start - j0;                        // jj = j + off on [j0, n), jj = j + off + n on [0, j0)
    float cref = (float)(i0 + lane * R + RH - off);
    f32x2 acc2[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc2[r] = 0ull;
#pragma unroll 1
    for (int seg = 0; seg < 2; ++seg) {
        const int lo = seg ? 0 : (j0 & ~1), hi = seg ? ((j0 + 1) & ~1) : ((n + 1) & ~1);
        const f32x2 cref2 = pk(cref, cref);
        int j = lo;
        if ((j & 2) && j < hi) {                          // odd pair index first: get onto a multiple of 4
            pair_step<R, true>(cs[cpos<PAD, R>(j)], cs[cpos<PAD, R>(j + 1)], cref2, acc2);
            j += 2;
        }
#pragma unroll 2
        for (; j + 2 < hi; j += 4) {
            pair_step<R, false>(cs[cpos<PAD, R>(j)], cs[cpos<PAD, R>(j + 1)], cref2, acc2);
            pair_step<R, true>(cs[cpos<PAD, R>(j + 2)], cs[cpos<PAD, R>(j + 3)], cref2, acc2);
        }
        if (j < hi) pair_step<R, false>(cs[cpos<PAD, R>(j)], cs[cpos<PAD, R>(j + 1)], cref2, acc2);
        cref -= (float)n;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        float lo, hi;
        unpk(acc2[r], lo, hi);
        acc[r] = lo + hi;
    }
}

// LYA_TAU_WINDOWED: every LANE walks only its own window jj = s0 .. around its R pixels (il = i0 + lane R): from
// s0 = il - W (W = the sightline's reach rounded up to a multiple of R; R = 1: rounded down to even) up to at least
// il + R - 1 + W, in whole pairs.  A source outside the window is further than its reach from all R pixels, so it would
// have added ex2(..) == 0 exactly; the sources kept are added in the same ascending order, into the same (even, odd)
// partial sums, with the same arithmetic (same reference pixel, the same exact integer separation E), so the result is
// bit-identical to tile_fast.  The row is stored unwrapped with a halo (cpos<true, R>), and s0 + TAU_HALO being a
// multiple of R the walk is whole pad groups: R consecutive slots, then one pad slot -- every LDS.128 offset is an
// immediate, there is no wrap test and no index arithmetic in the loop.  Returns the sources walked.
template <int R>
__device__ __forceinline__ int tile_window(const float4 *__restrict__ cs, int n, int i0, int lane, int W,
                                           float (&acc)[R])
{
    constexpr int RH = R / 2;
    constexpr int PG = R > 1 ? R : 2;                     // slots per pad group (R = 1: one pair, no pad)
    const int il = i0 + lane * R;
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0.0f;
    const int s0l = R > 1 ? il - W : (il - W) - ((il - W) & 1);
    const int groups = R > 1 ? (2 * W + R) / R : (il + W - s0l + 2) / 2;
    const int walked = groups * PG;                       // lane 0's count is the tile's (R = 1: +-1 between lanes)
    if (il >= n) return walked;                           // ragged last tile: this lane owns no pixel
    const float4 *q4 = cs + cpos<true, R>(s0l);           // slot of the first source; (s0l + TAU_HALO) % PG == 0
    const f32x2 cref2 = pk((float)(il + RH), (float)(il + RH));
    f32x2 acc2[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc2[r] = 0ull;
    // pair parity is absolute: s0l is a multiple of 4 for R = 4 (slots 0, 1 of a pad group: even pair; 2, 3: odd pair);
    // R < 4 never takes the polynomial
#pragma unroll 2
    for (int g = 0; g < groups; ++g) {
        pair_step<R, false>(q4[0], q4[1], cref2, acc2);
        if (PG == 4) pair_step<R, true>(q4[2], q4[3], cref2, acc2);
        q4 += R > 1 ? R + 1 : 2;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        float lo, hi;
        unpk(acc2[r], lo, hi);
        acc[r] = lo + hi;
    }
    return walked;
}

// General path: nearest image chosen per pair (tiny N, or |v_pec| comparable to the box).
template <int R, bool PAD>
__device__ __forceinline__ void tile_general(const float4 *__restrict__ cs, int n, float n_f, float inv_n, int i0,
                                             int lane, float (&acc)[R])
{
    float ci[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        acc[r] = 0.0f;
        ci[r]  = (float)(i0 + lane * R + r);
    }
#pragma unroll 2
    for (int j = 0; j < n; ++j) {
        const float4 q = get_cell<PAD, R>(cs, j);
        const float  f = -q.z / q.y;                    // fractional displacement (only picks the image)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float d0 = ci[r] - q.x;                     // exact integer
            float k  = rintf((d0 - f) * inv_n);
            float E  = fmaf(-n_f, k, d0);               // exact
            float x  = fmaf(E, q.y, q.z);
            float e  = ex2_ftz(-(x * x));
            acc[r]   = fmaf(q.w, e, acc[r]);
        }
    }
}

// one tile of one sightline: picks the loop from the sightline's reach; returns the sources walked per pixel
template <int R, bool WIN>
__device__ __forceinline__ int tile_any(const TauArgs &a, const float4 *cs, float reach, int i0, int lane,
                                        float (&acc)[R])
{
    const int n = a.n;
    if (!(reach <= (float)((n >> 1) - 16 * R))) {       // also catches +inf
        tile_general<R, WIN>(cs, n, a.n_f, a.inv_n, i0, lane, acc);
        return n;
    }
    if (WIN) {
        const int W = ((int)reach + R - 1) / R * R;         // floor(reach), then whole pad groups on either side
        if (W + R + 2 <= TAU_HALO && n >= TAU_HALO && !(n & 3)) return tile_window<R>(cs, n, i0, lane, W, acc);
    }
    tile_fast<R, WIN>(cs, n, i0, lane, acc);
    return n;
}

__device__ __forceinline__ void group_sync(int G, int bar_id)
{
    if (G == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(G * 32) : "memory");
}

// ---------------------------------------------------------------------------------------------------------
// Sightlines along x.  blockDim = 32 * G * gpc (gpc = groups per CTA).  Dynamic shared memory: per group n
// float4 cells, then per group one int4 control word {row, reach (float bits), next row, -}.
// (A variant that bulk-copied the next row into a raw buffer with cp.async.bulk + mbarrier while the current
// one was summed measured 4 % slower: profiles/r1_tau_prefetch_ab.md.  The row change here is plain coalesced
// loads; the other resident groups keep the MUFU pipe busy meanwhile.)
template <int R, bool FUSED, bool WIN>
__global__ void __launch_bounds__(1024, 1) tau_x_kernel(const TauArgs a, const int G, const int gpc)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grp = warp / G, wg = warp - grp * G;       // group in CTA, warp in group
    const int n = a.n;
    const int crow = crow_len<R>(n, WIN);                // float4 slots per staged row
    float4 *cells = reinterpret_cast<float4 *>(smem) + (size_t)grp * crow;
    volatile int *ctl = reinterpret_cast<volatile int *>(smem + (size_t)gpc * crow * sizeof(float4)) + 4 * grp;
    // per warp: four doubles, the running sum_i tau_i^k (k = 1..4) of the warp's tiles of the current row
    double *mom = reinterpret_cast<double *>(smem + (size_t)gpc * (crow * sizeof(float4) + 16)) + 4 * warp;
    const int bar_id = grp;      // named barrier of the group (G >= 2: at most 16 groups; no __syncthreads here)
    const int gl = wg * 32 + lane, gthreads = G * 32;    // thread index / count inside the group

    if (gl == 0) ctl[0] = (int)atomicAdd(&a.sched[0], 1u);
    group_sync(G, bar_id);

    for (;;) {
        const long long row = (unsigned int)ctl[0];
        if (row >= a.n_sl) break;
        const size_t g0 = (size_t)row * n;

        // ---- stage the row: (nHI, b, v_pec) [or delta, v_pec] -> (m, w, g, a) per cell; 128-byte coalesced loads
        float reach = 0.0f;
        if (a.vec_in) {                                  // four consecutive cells per thread and step, two steps in flight
            int j = 4 * gl;
            for (; j + 4 * gthreads < n; j += 8 * gthreads) {
                float4 nh0, bb0, vv0, nh1, bb1, vv1, q[4];
                load4<FUSED>(a, g0 + j, nh0, bb0, vv0);
                load4<FUSED>(a, g0 + j + 4 * gthreads, nh1, bb1, vv1);
                reach = fmaxf(reach, stage4<FUSED>(a, (float)j, nh0, bb0, vv0, q));
                put_cells4<WIN, R>(cells, j, q);
                reach = fmaxf(reach, stage4<FUSED>(a, (float)(j + 4 * gthreads), nh1, bb1, vv1, q));
                put_cells4<WIN, R>(cells, j + 4 * gthreads, q);
            }
            if (j < n) {
                float4 nh0, bb0, vv0, q[4];
                load4<FUSED>(a, g0 + j, nh0, bb0, vv0);
                reach = fmaxf(reach, stage4<FUSED>(a, (float)j, nh0, bb0, vv0, q));
                put_cells4<WIN, R>(cells, j, q);
            }
        } else {
            float jf = (float)gl;
#pragma unroll 4
            for (int j = gl; j < n; j += gthreads) {
                float4 q;
                reach = fmaxf(reach, stage_from_global<FUSED>(a, jf, g0 + j, q));
                put_cell<WIN, R>(cells, j, q);
                jf += (float)gthreads;
            }
            if (gl == 0) put_dummy<WIN, R>(cells, n);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) reach = fmaxf(reach, __shfl_xor_sync(0xffffffffu, reach, o));
        if (gl == 0) ctl[1] = 0;
        group_sync(G, bar_id);                           // cells complete, ctl[0] read
        if (G > 1 && lane == 0) atomicMax(const_cast<int *>(ctl + 1), __float_as_int(reach));   // reach >= 0
        if (gl == 0) ctl[2] = (int)atomicAdd(&a.sched[0], 1u);   // claim the next row early: latency hidden
        if (WIN) fill_halo<R>(cells, n, a.n_f, gl, gthreads);
        if (G > 1 || WIN) {
            group_sync(G, bar_id);
            reach = __int_as_float(G > 1 ? ctl[1] : __float_as_int(reach));
        }

        // ---- sum: the group's warps take the pixel tiles of the row
        int walked = 0;
        if (a.rowm && lane < 4) mom[lane] = 0.0;
        for (int tile = wg; tile < a.tiles; tile += G) {
            const int i0 = tile * 32 * R;
            float acc[R];
            walked = tile_any<R, WIN>(a, cells, reach, i0, lane, acc);
            const int i = i0 + lane * R;
            if (a.rowm) {                                // plain moments of the tile: fp32 over its 32 R pixels, double above
                float p[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float t = (i + r < n) ? acc[r] : 0.0f;
                    float q = t;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { p[k] += q; q *= t; }
                }
#pragma unroll
                for (int k = 0; k < 4; ++k)
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) p[k] += __shfl_xor_sync(0xffffffffu, p[k], o);
                __syncwarp();
                if (lane == 0)
#pragma unroll
                    for (int k = 0; k < 4; ++k) mom[k] += (double)p[k];
            }
            float *dst = a.tau + g0 + i;
            if (R == 4 && a.vec) {
                if (i < n) __stcs(reinterpret_cast<float4 *>(dst), make_float4(acc[0], acc[1], acc[2], acc[3]));
            } else if (R == 2 && a.vec) {
                if (i < n) __stcs(reinterpret_cast<float2 *>(dst), make_float2(acc[0], acc[1]));
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (i + r < n) dst[r] = acc[r];
            }
        }
        group_sync(G, bar_id);                           // cells consumed by every warp of the group
        if (gl == 0 && a.pairs) atomicAdd(a.pairs, (unsigned long long)n * (unsigned long long)walked);
        if (gl == 0 && a.rowm) {                         // the row's moments: the group's warps in fixed order
            double m[4] = {0.0, 0.0, 0.0, 0.0};
            const int nw = G < a.tiles ? G : a.tiles;    // warps that had a tile
            for (int w2 = 0; w2 < nw; ++w2)
#pragma unroll
                for (int k = 0; k < 4; ++k) m[k] += mom[4 * w2 + k];
            double *dst = a.rowm + 5 * (size_t)row;
            dst[0] = (double)n;
#pragma unroll
            for (int k = 0; k < 4; ++k) dst[1 + k] = m[k];
        }
        if (gl == 0) ctl[0] = ctl[2];
        group_sync(G, bar_id);
    }
}

// ---------------------------------------------------------------------------------------------------------
// Sightlines along y or z.  A CTA (8 warps) gathers bsl neighbouring x at a time so that global accesses are
// 4*bsl-byte segments (the sibling batches run at the same time on other CTAs, so L2 serves the rest of each
// sector), its warps sum (sightline, tile) items, and tau goes back through a shared-memory tile the same
// way.  Batches are handed out by the atomic counter; bsl is chosen so that >= 4 CTAs are resident per SM and
// one CTA's gather overlaps the others' pair loops.  cstride / tstride are padded so that neither the
// transposed staging stores nor the tile read-out have shared-memory bank conflicts.
template <int R, bool FUSED, bool WIN>
__global__ void __launch_bounds__(TAU_THREADS) tau_strided_kernel(const TauArgs a)
{
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ unsigned int s_batch;
    __shared__ int s_reach;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = a.n;
    const int cstride = a.cstride, tstride = a.tstride;
    float4 *cells = reinterpret_cast<float4 *>(smem);                                          // [bsl][cstride]
    float *ttile = reinterpret_cast<float *>(smem + (size_t)a.bsl * cstride * sizeof(float4)); // [bsl][tstride]

    if (tid == 0) s_batch = atomicAdd(&a.sched[0], 1u);
    __syncthreads();
    for (;;) {
        const long long batch = s_batch;
        if (batch >= a.n_batches) break;
        const long long outer = batch / a.nxb;
        const int xb = (int)(batch - outer * a.nxb);
        const int x0 = xb << a.bshift;
        const int nb = (a.nx - x0 < a.bsl) ? (a.nx - x0) : a.bsl;
        const long long base = outer * a.outer_stride + x0;   // element offset of (pixel 0, first x of the batch)

        float reach = 0.0f;
        if (tid == 0) s_reach = 0;
#pragma unroll 4
        for (int c = tid; c < (n << a.bshift); c += TAU_THREADS) {
            const int bx = c & (a.bsl - 1), j = c >> a.bshift;
            if (bx < nb) {
                float4 q;
                reach = fmaxf(reach, stage_from_global<FUSED>(a, (float)j, (size_t)(base + (long long)j * a.stride + bx), q));
                put_cell<WIN, R>(cells + bx * cstride, j, q);
            }
        }
        if (tid < nb) put_dummy<WIN, R>(cells + tid * cstride, n);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) reach = fmaxf(reach, __shfl_xor_sync(0xffffffffu, reach, o));
        __syncthreads();                                 // s_reach zeroed; s_batch read by everyone
        if (lane == 0) atomicMax(&s_reach, __float_as_int(reach));
        __syncthreads();                                 // cells complete
        reach = __int_as_float(s_reach);
        if (tid == 0) s_batch = atomicAdd(&a.sched[0], 1u);
        if (WIN) {
            for (int sl = warp; sl < nb; sl += TAU_WARPS) fill_halo<R>(cells + (size_t)sl * cstride, n, a.n_f, lane, 32);
            __syncthreads();
        }

        int walked = 0;
        const int items = nb * a.tiles;
        for (int item = warp; item < items; item += TAU_WARPS) {
            const int sl = item / a.tiles, tile = item - sl * a.tiles;
            const int i0 = tile * 32 * R;
            const float4 *cs = cells + (size_t)sl * cstride;
            float acc[R];
            walked = tile_any<R, WIN>(a, cs, reach, i0, lane, acc);
            const int i = i0 + lane * R;
            float *dst = ttile + (size_t)sl * tstride + i;     // tstride covers tiles * 32 * R: no bound check
            if (R == 4)      *reinterpret_cast<float4 *>(dst) = make_float4(acc[0], acc[1], acc[2], acc[3]);
            else if (R == 2) *reinterpret_cast<float2 *>(dst) = make_float2(acc[0], acc[1]);
            else             dst[0] = acc[0];
        }
        __syncthreads();                                 // cells consumed, tau tile complete, s_batch written
        if (tid == 0 && a.pairs) atomicAdd(a.pairs, (unsigned long long)nb * n * (unsigned long long)walked);
        if (a.rowm) {                                    // plain moments per sightline, read off the tau tile
            for (int sl = warp; sl < nb; sl += TAU_WARPS) {
                double m[4] = {0.0, 0.0, 0.0, 0.0};
                for (int j = lane; j < n; j += 32) {
                    const double t = (double)ttile[sl * tstride + j];
                    double q = t;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { m[k] += q; q *= t; }
                }
#pragma unroll
                for (int k = 0; k < 4; ++k)
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) m[k] += __shfl_xor_sync(0xffffffffu, m[k], o);
                if (lane == 0) {
                    double *dst = a.rowm + 5 * (size_t)(outer * a.nx + x0 + sl);
                    dst[0] = (double)n;
#pragma unroll
                    for (int k = 0; k < 4; ++k) dst[1 + k] = m[k];
                }
            }
        }
        for (int c = tid; c < (n << a.bshift); c += TAU_THREADS) {
            const int bx = c & (a.bsl - 1), j = c >> a.bshift;
            if (bx < nb) __stcs(a.tau + base + (long long)j * a.stride + bx, ttile[bx * tstride + j]);
        }
        __syncthreads();                                 // tile read out before the next batch's sums
    }

}

template <int R, bool FUSED, bool WIN>
lya_status launch_x(lya_ctx *ctx, const TauArgs &a)
{
    auto kern = tau_x_kernel<R, FUSED, WIN>;
    const size_t cap = (size_t)ctx->max_smem_optin;
    const size_t per_group = (size_t)crow_len<R>(a.n, WIN) * sizeof(float4) + 16;
    const size_t mom_bytes = 32 * 4 * sizeof(double);    // four running moments per warp (a.rowm)
    int groups = (int)((cap - mom_bytes) / per_group);   // groups that fit in one SM's shared memory
    if (groups < 1) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
    // G warps per group: as few as keep >= 24 warps resident, never more than the row has tiles
    int G = 1;
    while (G < 16 && G * (groups < 32 / G ? groups : 32 / G) < 24 && 2 * G <= a.tiles) G *= 2;
    if (groups > 32 / G) groups = 32 / G;
    if (G > 1 && groups > 16) groups = 16;               // 16 named barriers per CTA
    // one persistent CTA per SM; never more groups than rows
    long long want = (a.n_sl + ctx->sm_count - 1) / ctx->sm_count;
    if (groups > want) groups = (int)(want < 1 ? 1 : want);
    const size_t smem_bytes = (size_t)groups * per_group + mom_bytes;
    int resident = 0;
    lya_status st = lya_kernel_occupancy(ctx, (const void *)kern, 32 * G * groups, smem_bytes, &resident);
    if (st != LYA_OK) return st;
    if (resident < 1) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
    long long ctas = (a.n_sl + groups - 1) / groups;
    const int grid = (int)(ctas < ctx->sm_count ? ctas : ctx->sm_count);
    kern<<<grid, 32 * G * groups, smem_bytes, ctx->stream>>>(a, G, groups);
    ctx->launches++;
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}

template <int R, bool FUSED, bool WIN>
lya_status launch_strided(lya_ctx *ctx, const TauArgs &a, size_t smem_bytes)
{
    auto kern = tau_strided_kernel<R, FUSED, WIN>;
    int per_sm = 0;
    lya_status st = lya_kernel_occupancy(ctx, (const void *)kern, TAU_THREADS, smem_bytes, &per_sm);
    if (st != LYA_OK) return st;
    if (per_sm < 1) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
    long long cap = (long long)ctx->sm_count * per_sm;
    int grid = (int)(a.n_batches < cap ? a.n_batches : cap);
    kern<<<grid, TAU_THREADS, smem_bytes, ctx->stream>>>(a);
    ctx->launches++;
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}

}  // namespace

lya_status lya_launch_tau(lya_ctx *ctx, int axis, int nx, int ny, int nz_local,
                          const float *n_hi, const float *b, const float *v, float *tau,
                          double amp_scale, double dv_kms, unsigned flags, const float *gas5,
                          unsigned long long *d_pairs, double *d_rowm)
{
    const bool fused = (flags & LYA_TAU_FROM_DENSITY) != 0;
    const bool win = (flags & LYA_TAU_WINDOWED) != 0;
    TauArgs a;
    memset(&a, 0, sizeof(a));
    a.n_hi = n_hi; a.b = b; a.v = v; a.tau = tau;
    const int n = axis == 0 ? nx : (axis == 1 ? ny : nz_local);
    a.n = n;
    a.inv_dv_hi = (float)(1.0 / dv_kms);
    a.inv_dv_lo = (float)(1.0 / dv_kms - (double)a.inv_dv_hi);
    a.amp_scale = (float)amp_scale;
    a.w_scale   = (float)(dv_kms * 1.2011224087864498);   // sqrt(log2 e)
    a.n_f = (float)n;
    a.inv_n = 1.0f / (float)n;
    a.xcut_over_w = TAU_XCUT / a.w_scale;
    a.pairs = d_pairs;
    a.rowm = d_rowm;
    // the work counter is zeroed on the stream before EVERY launch: a launch that failed or was killed midway cannot
    // leave it armed and turn later launches on this ctx into no-ops
    LYA_CUDA(ctx, cudaMemsetAsync(ctx->d_sched, 0, 2 * sizeof(unsigned int), ctx->stream));
    if (fused) a.gas = GasK{gas5[0], gas5[1], gas5[2], gas5[3], gas5[4]};
    const int R = n >= 128 ? 4 : (n >= 64 ? 2 : 1);
    a.tiles = (n + 32 * R - 1) / (32 * R);
    const size_t smem_cap = (size_t)ctx->max_smem_optin;

    if (axis == 0) {
        a.n_sl = (long long)ny * nz_local;
        if (a.n_sl >= (1LL << 31)) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: more than 2^31 sightlines");
        a.vec = (n % 4 == 0) && (((uintptr_t)tau & 15) == 0);
        a.vec_in = (n % 4 == 0) && ((((uintptr_t)n_hi | (uintptr_t)v | (fused ? 0 : (uintptr_t)b)) & 15) == 0);
        a.sched = ctx->d_sched;
#define LYA_TAU_X(RR)                                                                                       \
    return win ? (fused ? launch_x<RR, true, true>(ctx, a) : launch_x<RR, false, true>(ctx, a))             \
               : (fused ? launch_x<RR, true, false>(ctx, a) : launch_x<RR, false, false>(ctx, a))
        switch (R) {
            case 1:  LYA_TAU_X(1);
            case 2:  LYA_TAU_X(2);
            default: LYA_TAU_X(4);
        }
#undef LYA_TAU_X
    }

    // strided: axis 1 (pixels along y, outer index iz) or axis 2 (pixels along z, outer index iy)
    a.nx = nx;
    a.stride = axis == 1 ? (long long)nx : (long long)nx * ny;
    a.outer_stride = axis == 1 ? (long long)nx * ny : (long long)nx;
    const long long n_outer = axis == 1 ? nz_local : ny;
    // per staged sightline: cstride float4 cells + tstride floats of tau tile; strides padded against bank
    // conflicts: cstride = 8/bsl (mod 8) float4s for the transposed STS.128, tstride = 32/bsl (mod 32) floats
    // for the read-out (both trivially fine for bsl = 1)
    auto pad_to = [](int v, int mod, int want) { return v + ((want - v % mod) % mod + mod) % mod; };
    auto strides = [&](int sh, int &cs, int &ts) {
        const int bs = 1 << sh;
        cs = pad_to(R == 4 ? crow_len<4>(n, win) : (R == 2 ? crow_len<2>(n, win) : crow_len<1>(n, win)), 8, (8 / bs) % 8);
        ts = pad_to(a.tiles * 32 * R, 32, (32 / bs) % 32);
    };
    auto need2 = [&](int sh) {
        int cs, ts;
        strides(sh, cs, ts);
        return ((size_t)cs * 16 + (size_t)ts * 4) << sh;
    };
    int bshift = 3;                                      // 32-byte segments if >= 4 CTAs still fit per SM
    while (bshift > 1 && 4 * (need2(bshift) + 1024) > smem_cap) --bshift;
    while (bshift > 0 && need2(bshift) > smem_cap) --bshift;
    if (need2(bshift) > smem_cap)
        return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
    a.bshift = bshift;
    a.bsl = 1 << bshift;
    strides(bshift, a.cstride, a.tstride);
    a.nxb = (nx + a.bsl - 1) / a.bsl;
    a.n_batches = n_outer * a.nxb;
    if (a.n_batches >= (1LL << 31)) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: more than 2^31 batches");
    a.sched = ctx->d_sched;
#define LYA_TAU_S(RR)                                                                                       \
    return win ? (fused ? launch_strided<RR, true, true>(ctx, a, need2(bshift))                             \
                        : launch_strided<RR, false, true>(ctx, a, need2(bshift)))                           \
               : (fused ? launch_strided<RR, true, false>(ctx, a, need2(bshift))                            \
                        : launch_strided<RR, false, false>(ctx, a, need2(bshift)))
    switch (R) {
        case 1:  LYA_TAU_S(1);
        case 2:  LYA_TAU_S(2);
        default: LYA_TAU_S(4);
    }
#undef LYA_TAU_S
}
