// tau.cu -- S2 + S3: redshift-space optical depth along every sightline (Eq.6).
//
//   tau(i) = K sum_j nHI(j)/b(j) exp(-((v_H(i) - u(j))/b(j))^2),   u(j) = v_H(j) + v_pec(j),
//   v_H(i) - v_H(j) = (i-j) dv, nearest periodic image (period V = N dv; reading C7).
//
// Every (i,j) pair is evaluated (N^2 per sightline): the kernel is bound by MUFU.EX2 (16 /clk/SM), so the
// pair body is kept at 4 FP32 instructions + 1 MUFU:
//
//   staged per source cell j (once per sightline, in shared memory, one float4):
//       m_j = j + P_j          P_j = round(v_pec/dv), reduced mod N          (integer-valued float, exact)
//       w_j = (dv/b_j) sqrt(log2 e)                                          (so exp(-x^2) = ex2(-(x')^2))
//       g_j = -f_j w_j         f_j = v_pec/dv - round(v_pec/dv)  in [-1/2,1/2] (computed in double)
//       a_j = K 1e-5 nHI_j / b_j                                             (line-centre amplitude)
//   per pair:  E = c_i - m_j (exact) ; x = fma(E, w_j, g_j) ; e = ex2(-x*x) ; acc = fma(a_j, e, acc)
//
// Keeping the integer part of the pixel separation exact is what holds the error at ~1e-6 for N = 2048
// (forming u_j and v_i in fp32 km/s loses 3 digits there).
//
// Periodic wrap without per-pair work: a warp owns a tile of 32*R consecutive pixels and walks the sources
// in UNWRAPPED order jj = c - N/2 ... c + N/2 - 1 around the tile centre c (two contiguous index segments),
// so i - jj is already the nearest image for every pair that can contribute.  That is valid when, for every
// source of the sightline, (N/2 - 16R - |P_j| - 1) w_j >= 12.5, i.e. a pair whose chosen image is not the
// nearest has ex2(-x^2) == 0 in fp32 (and < 2^-156 of a_j in the oracle's double).  The staging pass checks
// the condition; a batch that fails it (tiny N, |v_pec| of order V) takes the general loop with a per-pair
// image choice.  Both loops evaluate all N^2 pairs.
//
// Mapping: persistent CTAs (grid = k * SM count) loop over batches of B sightlines; a batch's nHI/b/v_pec
// rows are fetched by cp.async.bulk into a 2-stage shared-memory ring (mbarrier complete_tx) while the
// previous batch is being summed; the 8 warps of the CTA then take (sightline, pixel-tile) items, every
// lane reading the same staged cell (broadcast LDS.128) for R pixels.  Sightlines along y / z are gathered
// 8 (or fewer) neighbouring x at a time so that global accesses stay 32-byte segments, and tau goes back
// through a shared-memory tile the same way.
#include "lya_internal.h"

namespace {

constexpr int   TAU_WARPS   = 8;
constexpr int   TAU_THREADS = TAU_WARPS * 32;
constexpr float TAU_XCUT    = 12.5f;   // ex2(-12.5^2) = 2^-156: exactly 0 in fp32 (ftz)

struct TauArgs {
    const float *n_hi, *b, *v;
    float       *tau;
    int          n;           // pixels per sightline
    int          tiles;       // pixel tiles of 32*R per sightline
    int          bsl;         // sightlines per batch (x-axis) / x-width of a gathered batch (y,z; power of 2)
    int          bshift;      // log2(bsl) for the strided modes
    long long    n_sl;        // x-axis: number of sightlines (rows)
    long long    n_batches;
    // strided modes (axis 1, 2)
    int          nx;          // x extent
    int          nxb;         // ceil(nx / bsl)
    long long    outer_stride; // elements between consecutive "outer" indices (axis 1: ny*nx per iz; axis 2: nx per iy)
    long long    stride;      // elements between consecutive pixels of a sightline
    double       inv_dv;      // 1 / dv  [s/km]
    float        amp_scale;   // K * 1e-5  [cm^3 * km/s ... so that a_j is dimensionless]
    float        w_scale;     // dv * sqrt(log2 e) [km/s]
    float        inv_n, n_f;  // 1/N, N
};

__device__ __forceinline__ float ex2_ftz(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// One source cell -> staged float4 (m, w, g, a); returns 1 if the cell breaks the fast-path condition.
__device__ __forceinline__ int stage_cell(const TauArgs &a, int j, float nh, float bb, float vv, int half_span,
                                          float4 &out)
{
    double p  = (double)vv * a.inv_dv;                 // displacement in pixels (reading C11: +v -> higher index)
    double P  = rint(p);
    float  f  = (float)(p - P);                        // [-1/2, 1/2], full fp32 precision
    double Pr = P - (double)a.n * rint(P / (double)a.n);   // integer displacement reduced to [-N/2, N/2]
    float  w  = a.w_scale / bb;
    out.x = (float)((double)j + Pr);
    out.y = w;
    out.z = -f * w;
    out.w = a.amp_scale * nh / bb;
    float room = (float)(a.n >> 1) - (float)half_span - fabsf((float)Pr) - 1.0f;
    return !(room * w >= TAU_XCUT);
}

// Fast path: unwrapped walk around the tile centre, no per-pair image logic.
template <int R>
__device__ __forceinline__ void tile_fast(const float4 *__restrict__ cs, int n, int i0, int lane, float (&acc)[R])
{
    const int c     = i0 + 16 * R;
    const int start = c - (n >> 1);                    // first unwrapped source index
    int j0 = start % n;
    if (j0 < 0) j0 += n;                               // slot holding jj = start
    const int off = start - j0;                        // jj = j + off on [j0, n), jj = j + off + n on [0, j0)
    float cr[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        acc[r] = 0.0f;
        cr[r]  = (float)(i0 + lane + 32 * r - off);
    }
#pragma unroll 1
    for (int seg = 0; seg < 2; ++seg) {
        const int lo = seg ? 0 : j0, hi = seg ? j0 : n;
#pragma unroll 4
        for (int j = lo; j < hi; ++j) {
            const float4 q = cs[j];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                float E = cr[r] - q.x;
                float x = fmaf(E, q.y, q.z);
                float e = ex2_ftz(-(x * x));
                acc[r]  = fmaf(q.w, e, acc[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) cr[r] -= (float)n;
    }
}

// General path: nearest image chosen per pair (tiny N, or |v_pec| comparable to the box).
template <int R>
__device__ __forceinline__ void tile_general(const float4 *__restrict__ cs, int n, float n_f, float inv_n, int i0,
                                             int lane, float (&acc)[R])
{
    float ci[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        acc[r] = 0.0f;
        ci[r]  = (float)(i0 + lane + 32 * r);
    }
#pragma unroll 2
    for (int j = 0; j < n; ++j) {
        const float4 q = cs[j];
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

// MODE 0: x-axis, cp.async.bulk ring.  MODE 1: x-axis, plain loads (unaligned / N % 4 != 0).
// MODE 2: strided sightlines (y or z), gathered bsl neighbouring x at a time.
template <int R, int MODE>
__global__ void __launch_bounds__(TAU_THREADS) tau_kernel(const TauArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = a.n;
    const int cstride = (MODE == 2) ? n + 1 : n;        // +1 cell: conflict-free transposed staging
    float4 *cells = reinterpret_cast<float4 *>(smem);
    const size_t cells_bytes = (size_t)a.bsl * cstride * sizeof(float4);
    float *aux = reinterpret_cast<float *>(smem + cells_bytes);     // MODE 0: raw ring; MODE 2: tau tile
    const int per_arr = a.bsl * n;                                  // floats per raw array per stage
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem + cells_bytes + (size_t)6 * per_arr * sizeof(float));

    auto issue = [&](long long batch, int stage) {                  // MODE 0, one thread
        long long s0 = batch * a.bsl;
        int nb = (int)((a.n_sl - s0 < a.bsl) ? (a.n_sl - s0) : a.bsl);
        uint32_t bytes = (uint32_t)nb * n * 4u;
        float *dst = aux + (size_t)stage * 3 * per_arr;
        mbar_expect_tx(&mbar[stage], 3u * bytes);
        bulk_g2s(dst,               a.n_hi + s0 * n, bytes, &mbar[stage]);
        bulk_g2s(dst + per_arr,     a.b    + s0 * n, bytes, &mbar[stage]);
        bulk_g2s(dst + 2 * per_arr, a.v    + s0 * n, bytes, &mbar[stage]);
    };

    if (MODE == 0) {
        if (tid == 0) {
            mbar_init(&mbar[0], 1);
            mbar_init(&mbar[1], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        if (tid == 0 && (long long)blockIdx.x < a.n_batches) issue(blockIdx.x, 0);
    }

    int it = 0;
    for (long long batch = blockIdx.x; batch < a.n_batches; batch += gridDim.x, ++it) {
        int nb;                       // sightlines in this batch
        long long base = 0;           // strided: element offset of (pixel 0, first x of the batch)
        if (MODE == 2) {
            long long outer = batch / a.nxb;
            int xb = (int)(batch - outer * a.nxb);
            int x0 = xb << a.bshift;
            nb   = (a.nx - x0 < a.bsl) ? (a.nx - x0) : a.bsl;
            base = outer * a.outer_stride + x0;
        } else {
            long long s0 = batch * a.bsl;
            nb = (int)((a.n_sl - s0 < a.bsl) ? (a.n_sl - s0) : a.bsl);
        }

        // ---- stage the batch: (nHI, b, v_pec) -> (m, w, g, a) per cell
        int bad = 0;
        if (MODE == 0) {
            const int stage = it & 1;
            long long next = batch + gridDim.x;
            if (tid == 0 && next < a.n_batches) issue(next, stage ^ 1);
            mbar_wait(&mbar[stage], (uint32_t)((it >> 1) & 1));
            const float *raw = aux + (size_t)stage * 3 * per_arr;
            for (int c = tid; c < nb * n; c += TAU_THREADS) {
                int j = c % n;
                float4 q;
                bad |= stage_cell(a, j, raw[c], raw[per_arr + c], raw[2 * per_arr + c], 16 * R, q);
                cells[c] = q;
            }
        } else if (MODE == 1) {
            const long long g0 = batch * a.bsl * n;
            for (int c = tid; c < nb * n; c += TAU_THREADS) {
                int j = c % n;
                float4 q;
                bad |= stage_cell(a, j, __ldg(a.n_hi + g0 + c), __ldg(a.b + g0 + c), __ldg(a.v + g0 + c), 16 * R, q);
                cells[c] = q;
            }
        } else {
            for (int c = tid; c < (n << a.bshift); c += TAU_THREADS) {
                int bx = c & (a.bsl - 1), j = c >> a.bshift;
                if (bx < nb) {
                    long long g = base + (long long)j * a.stride + bx;
                    float4 q;
                    bad |= stage_cell(a, j, __ldg(a.n_hi + g), __ldg(a.b + g), __ldg(a.v + g), 16 * R, q);
                    cells[bx * cstride + j] = q;
                }
            }
        }
        bad = __syncthreads_or(bad);

        // ---- sum: warps take (sightline, pixel tile) items
        const int items = nb * a.tiles;
        for (int item = warp; item < items; item += TAU_WARPS) {
            const int sl = item / a.tiles, tile = item - sl * a.tiles;
            const int i0 = tile * 32 * R;
            const float4 *cs = cells + (size_t)sl * cstride;
            float acc[R];
            if (!bad) tile_fast<R>(cs, n, i0, lane, acc);
            else      tile_general<R>(cs, n, a.n_f, a.inv_n, i0, lane, acc);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                int i = i0 + lane + 32 * r;
                if (i < n) {
                    if (MODE == 2) aux[(i << a.bshift) + sl] = acc[r];
                    else           a.tau[(batch * a.bsl + sl) * n + i] = acc[r];
                }
            }
        }
        __syncthreads();                                 // cells (and the tau tile) complete / consumed
        if (MODE == 2) {
            for (int c = tid; c < (n << a.bshift); c += TAU_THREADS) {
                int bx = c & (a.bsl - 1), j = c >> a.bshift;
                if (bx < nb) a.tau[base + (long long)j * a.stride + bx] = aux[c];
            }
            __syncthreads();
        }
    }
}

template <int R, int MODE>
lya_status launch_rm(lya_ctx *ctx, const TauArgs &a, size_t smem_bytes)
{
    auto kern = tau_kernel<R, MODE>;
    LYA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
    int per_sm = 0;
    LYA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, TAU_THREADS, smem_bytes));
    if (per_sm < 1) return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
    long long cap = (long long)ctx->sm_count * per_sm;
    int grid = (int)(a.n_batches < cap ? a.n_batches : cap);
    kern<<<grid, TAU_THREADS, smem_bytes, ctx->stream>>>(a);
    ctx->launches++;
    LYA_CUDA(ctx, cudaGetLastError());
    return LYA_OK;
}

template <int MODE>
lya_status launch_m(lya_ctx *ctx, int R, const TauArgs &a, size_t smem_bytes)
{
    switch (R) {
        case 1:  return launch_rm<1, MODE>(ctx, a, smem_bytes);
        case 2:  return launch_rm<2, MODE>(ctx, a, smem_bytes);
        default: return launch_rm<4, MODE>(ctx, a, smem_bytes);
    }
}

}  // namespace

lya_status lya_launch_tau(lya_ctx *ctx, int axis, int nx, int ny, int nz_local,
                          const float *n_hi, const float *b, const float *v, float *tau,
                          double amp_scale, double dv_kms)
{
    TauArgs a;
    memset(&a, 0, sizeof(a));
    a.n_hi = n_hi; a.b = b; a.v = v; a.tau = tau;
    const int n = axis == 0 ? nx : (axis == 1 ? ny : nz_local);
    a.n = n;
    a.inv_dv    = 1.0 / dv_kms;
    a.amp_scale = (float)amp_scale;
    a.w_scale   = (float)(dv_kms * 1.2011224087864498);   // sqrt(log2 e)
    a.n_f = (float)n;
    a.inv_n = 1.0f / (float)n;
    const int R = n >= 128 ? 4 : (n >= 64 ? 2 : 1);
    a.tiles = (n + 32 * R - 1) / (32 * R);
    const size_t smem_cap = (size_t)ctx->max_smem_optin;

    if (axis == 0) {
        a.n_sl = (long long)ny * nz_local;
        int bsl = TAU_WARPS / a.tiles;
        if (bsl < 1) bsl = 1;
        if ((long long)bsl > a.n_sl) bsl = (int)a.n_sl;
        bool bulk = (n % 4 == 0) && ((((uintptr_t)n_hi | (uintptr_t)b | (uintptr_t)v) & 15) == 0);
        // shrink the batch if it would not fit (very long sightlines)
        auto need = [&](int bs, bool blk) {
            return (size_t)bs * n * 16 + (blk ? (size_t)bs * n * 24 + 16 : 0);
        };
        while (bsl > 1 && need(bsl, bulk) > smem_cap / 2) bsl >>= 1;
        if (bulk && need(bsl, true) > smem_cap) bulk = false;
        if (need(bsl, bulk) > smem_cap)
            return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
        a.bsl = bsl;
        a.n_batches = (a.n_sl + bsl - 1) / bsl;
        return bulk ? launch_m<0>(ctx, R, a, need(bsl, true)) : launch_m<1>(ctx, R, a, need(bsl, false));
    }

    // strided: axis 1 (pixels along y, outer index iz) or axis 2 (pixels along z, outer index iy)
    a.nx = nx;
    a.stride = axis == 1 ? (long long)nx : (long long)nx * ny;
    a.outer_stride = axis == 1 ? (long long)nx * ny : (long long)nx;
    const long long n_outer = axis == 1 ? nz_local : ny;
    int bshift = 3;
    auto need2 = [&](int sh) { return ((size_t)(n + 1) * 16 + (size_t)n * 4) << sh; };
    while (bshift > 0 && need2(bshift) > smem_cap / 2) --bshift;
    if (need2(bshift) > smem_cap)
        return lya_fail(ctx, LYA_EINVAL, "lya_tau_sightlines: sightline too long for shared memory");
    a.bshift = bshift;
    a.bsl = 1 << bshift;
    a.nxb = (nx + a.bsl - 1) / a.bsl;
    a.n_batches = n_outer * a.nxb;
    return launch_m<2>(ctx, R, a, need2(bshift));
}
