// fields.cu -- before the hot path: baryon density and peculiar velocity from a
// dark-matter density field.
//   Eq.1  delta_b(k) = delta_DM(k) / (1 + k^2 / k_F^2)
//   Eq.3  v_a(k)     = E_+ i k_a / k^2 delta_DM(k),  E_+ = H(z) f(z) / (1+z)   [km/s per comoving Mpc]
// One real-to-complex 3D FFT of delta_DM, then ONE k-space kernel for all requested outputs (8 B read once + 8 B
// written per output and half-spectrum mode, HBM-bound; the 1/N^3 of the unnormalised transforms is folded in) and
// one complex-to-real FFT per output.  The FFTs are cuFFT's (library primitive), resolved with dlopen at first use so that
// liblya.so itself does not depend on libcufft; everything else is this file.  Readings U1-U5: DESIGN.md 12.
#include <cufft.h>
#include <dlfcn.h>
#include <math.h>

#include <mutex>

#include "lya_internal.h"

namespace {

struct CufftApi {
    void *handle;
    cufftResult (*Plan3d)(cufftHandle *, int, int, int, cufftType);
    cufftResult (*SetStream)(cufftHandle, cudaStream_t);
    cufftResult (*ExecR2C)(cufftHandle, cufftReal *, cufftComplex *);
    cufftResult (*ExecC2R)(cufftHandle, cufftComplex *, cufftReal *);
    cufftResult (*Destroy)(cufftHandle);
};

CufftApi *cufft_api()
{
    static CufftApi api = {};
    static std::once_flag once;
    static bool ok = false;
    std::call_once(once, [] {                               // contexts of several host threads may race here
        const char *names[] = {"libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so.11",
                               "/usr/local/cuda/lib64/libcufft.so"};
        for (const char *nm : names)
            if ((api.handle = dlopen(nm, RTLD_NOW | RTLD_LOCAL))) break;
        if (api.handle) {
            api.Plan3d    = (decltype(api.Plan3d))dlsym(api.handle, "cufftPlan3d");
            api.SetStream = (decltype(api.SetStream))dlsym(api.handle, "cufftSetStream");
            api.ExecR2C   = (decltype(api.ExecR2C))dlsym(api.handle, "cufftExecR2C");
            api.ExecC2R   = (decltype(api.ExecC2R))dlsym(api.handle, "cufftExecC2R");
            api.Destroy   = (decltype(api.Destroy))dlsym(api.handle, "cufftDestroy");
        }
        ok = api.handle && api.Plan3d && api.SetStream && api.ExecR2C && api.ExecC2R && api.Destroy;
    });
    return ok ? &api : nullptr;
}

struct KArgs {
    const float2 *in;
    float2       *out[4];             // per output (0: Eq.1 filter; 1, 2, 3: Eq.3 velocity along x, y, z), NULL: not wanted
    int           nxh, nx, ny, nz;
    unsigned      rows_per_block;
    size_t        n_rows;             // ny * nz
    float         dkx, dky, dkz;       // 2 pi h / L_i [Mpc^-1]
    float         inv_kf2;             // 1 / k_F^2 (0: no filtering)
    float         scale0, scale_v;     // 1/N^3; E_+ / N^3
};

// One read of delta(k) (8 B per half-spectrum mode) serves EVERY requested output (8 B written each).  A block owns
// KS_ROWS consecutive (iz, iy) rows of nx/2 + 1 modes as one flat range, so that the odd row length does not leave
// most of a last trip idle (a block per row with 128 threads kept 257 modes busy 67 % of the time); a thread steps
// through the range by the block size and carries (ix, iy, iz) along, so there is no division in the loop.
constexpr int KS_THREADS = 256, KS_ROWS = 16;

__global__ void __launch_bounds__(KS_THREADS) kspace_kernel(const KArgs a)
{
    const size_t row0 = (size_t)blockIdx.x * a.rows_per_block;
    const size_t rows = a.n_rows - row0 < a.rows_per_block ? a.n_rows - row0 : a.rows_per_block;
    const unsigned count = (unsigned)rows * (unsigned)a.nxh;
    unsigned l = threadIdx.x;
    unsigned lr = l / (unsigned)a.nxh;
    int ix = (int)(l - lr * (unsigned)a.nxh);
    int iy = (int)((row0 + lr) % (size_t)a.ny), iz = (int)((row0 + lr) / (size_t)a.ny);
    const int step_r = KS_THREADS / a.nxh, step_x = KS_THREADS - step_r * a.nxh;   // one step = step_r rows + step_x modes
    const bool even_x = (a.nx & 1) == 0, even_y = (a.ny & 1) == 0, even_z = (a.nz & 1) == 0;
    const float2 *in = a.in + row0 * a.nxh;
    // two further loads are always in flight per thread: 64 resident warps x 8 B per lane are only 16 KB per SM
    // with one (ncu: long-scoreboard 15.7 stall cycles per issue, 61 % of the DRAM peak)
    float2 d1 = l + KS_THREADS < count ? __ldcs(in + l + KS_THREADS) : make_float2(0.f, 0.f);
    float2 d0 = l < count ? __ldcs(in + l) : make_float2(0.f, 0.f);
    for (; l < count; l += KS_THREADS) {
        const float2 d2 = l + 2 * KS_THREADS < count ? __ldcs(in + l + 2 * KS_THREADS) : make_float2(0.f, 0.f);
        const int my = iy < (a.ny + 1) / 2 ? iy : iy - a.ny;       // signed frequency, -n/2 at the Nyquist slot
        const int mz = iz < (a.nz + 1) / 2 ? iz : iz - a.nz;
        const float kx = a.dkx * (float)ix, ky = a.dky * (float)my, kz = a.dkz * (float)mz;
        const float k2 = fmaf(kx, kx, fmaf(ky, ky, kz * kz));
        const float2 d = d0;
        const size_t e = row0 * a.nxh + l;
        if (a.out[0]) {
            const float f = __fdividef(a.scale0, fmaf(k2, a.inv_kf2, 1.0f));       // 2 ulp: far inside the FFT's own error
            __stcs(a.out[0] + e, make_float2(d.x * f, d.y * f));
        }
        const float g = k2 > 0.0f ? __fdividef(a.scale_v, k2) : 0.0f;              // U4: no k = 0 mode
        if (a.out[1]) {
            const float c = (even_x && ix == a.nx / 2) ? 0.0f : g * kx;            // U4: no Nyquist plane of the axis
            __stcs(a.out[1] + e, make_float2(-d.y * c, d.x * c));                  // times i c
        }
        if (a.out[2]) {
            const float c = (even_y && iy == a.ny / 2) ? 0.0f : g * ky;
            __stcs(a.out[2] + e, make_float2(-d.y * c, d.x * c));
        }
        if (a.out[3]) {
            const float c = (even_z && iz == a.nz / 2) ? 0.0f : g * kz;
            __stcs(a.out[3] + e, make_float2(-d.y * c, d.x * c));
        }
        d0 = d1; d1 = d2;
        ix += step_x; iy += step_r;
        if (ix >= a.nxh) { ix -= a.nxh; ++iy; }
        while (iy >= a.ny) { iy -= a.ny; ++iz; }
    }
}

lya_status ensure_ws(lya_ctx *ctx, size_t bytes)
{
    if (ctx->ws_bytes >= bytes) return LYA_OK;
    if (ctx->ws) { cudaFree(ctx->ws); ctx->ws = nullptr; ctx->ws_bytes = 0; }
    if (cudaMalloc(&ctx->ws, bytes) != cudaSuccess) {
        cudaGetLastError();
        return lya_fail(ctx, LYA_ENOMEM, "lya_fields_from_dm: device workspace allocation failed");
    }
    ctx->ws_bytes = bytes;
    return LYA_OK;
}

}  // namespace

extern "C" lya_status lya_growth_rate(double z, double omega_m, double *f_out)
{
    if (!f_out || !(z > -1.0) || !(omega_m > 0.0) || !(omega_m <= 1.0)) return LYA_EINVAL;
    // D(a) ~ E(a) I(a), I = int_0^a dx / (x E(x))^3; with x = t^2 the integrand 2 t^4 / (Om + OL t^6)^1.5 is smooth
    const double a = 1.0 / (1.0 + z), ol = 1.0 - omega_m, T = sqrt(a);
    const int n = 4096;
    auto g = [&](double t) { const double t2 = t * t, t6 = t2 * t2 * t2; return 2.0 * t2 * t2 / pow(omega_m + ol * t6, 1.5); };
    double s = g(0.0) + g(T);
    for (int i = 1; i < n; ++i) s += (i & 1 ? 4.0 : 2.0) * g(T * i / n);
    const double I = s * T / (3.0 * n);
    const double E2 = omega_m / (a * a * a) + ol, E = sqrt(E2);
    *f_out = -1.5 * omega_m / (a * a * a) / E2 + a / pow(a * E, 3.0) / I;
    return LYA_OK;
}

extern "C" lya_status lya_fields_from_dm(lya_ctx *ctx, const lya_field_params *p, const float *delta_dm,
                                         float *delta_b, float *v_x, float *v_y, float *v_z)
{
    if (!ctx) return LYA_EINVAL;
    ctx->err[0] = 0;
    if (!p || !delta_dm) return lya_fail(ctx, LYA_EINVAL, "lya_fields_from_dm: null pointer");
    if (p->nx < 2 || p->ny < 1 || p->nz < 1 || !(p->box_mpch > 0.0) || !(p->h > 0.0) || !(p->z > -1.0) ||
        !(p->omega_m > 0.0) || !(p->omega_m <= 1.0))
        return lya_fail(ctx, LYA_EINVAL, "lya_fields_from_dm: bad parameters");
    float *outs[4] = {delta_b, v_x, v_y, v_z};
    for (int i = 0; i < 4; ++i) {
        if (outs[i] && (outs[i] == delta_dm || ((uintptr_t)outs[i] & 3))) return lya_fail(ctx, LYA_EINVAL, "lya_fields_from_dm: output aliases the input or is misaligned");
        for (int j = 0; j < i; ++j)
            if (outs[i] && outs[i] == outs[j]) return lya_fail(ctx, LYA_EINVAL, "lya_fields_from_dm: outputs alias each other");
    }
    CufftApi *fft = cufft_api();
    if (!fft) return lya_fail(ctx, LYA_ECUDA, "lya_fields_from_dm: libcufft not found (dlopen)");
    LYA_CUDA(ctx, cudaSetDevice(ctx->device));

    const int nxh = p->nx / 2 + 1;
    const size_t half = (size_t)p->nz * p->ny * nxh;
    ctx->forest_total = 0;                               // the shared workspace no longer holds lya_forest_host_begin's tau
    int n_out = 0;
    for (int i = 0; i < 4; ++i) n_out += outs[i] != nullptr;
    if (n_out == 0) return LYA_OK;
    // one spectrum buffer per output lets ONE k-space kernel serve them all from a single read of delta(k); if the
    // device cannot hold that many, two buffers and one kernel per output do
    int n_buf = n_out;
    lya_status st = LYA_OK;
    if (ctx->ws_bytes < (1 + (size_t)n_buf) * half * sizeof(float2) + 256) {
        size_t free_b = 0, total_b = 0;
        cudaMemGetInfo(&free_b, &total_b);
        if (free_b + ctx->ws_bytes < (1 + (size_t)n_buf) * half * sizeof(float2) + ((size_t)1 << 30)) n_buf = 1;
    }
    st = ensure_ws(ctx, (1 + (size_t)n_buf) * half * sizeof(float2) + 256);
    if (st != LYA_OK && n_buf > 1) { n_buf = 1; ctx->err[0] = 0; st = ensure_ws(ctx, 2 * half * sizeof(float2) + 256); }
    if (st != LYA_OK) return st;
    float2 *A = (float2 *)ctx->ws, *B = A + half;

    if (ctx->fft_dims[0] != p->nz || ctx->fft_dims[1] != p->ny || ctx->fft_dims[2] != p->nx) {
        if (ctx->fft_dims[0]) { fft->Destroy(ctx->fft_r2c); fft->Destroy(ctx->fft_c2r); ctx->fft_dims[0] = 0; }
        if (fft->Plan3d(&ctx->fft_r2c, p->nz, p->ny, p->nx, CUFFT_R2C) != CUFFT_SUCCESS)
            return lya_fail(ctx, LYA_ECUDA, "lya_fields_from_dm: cufftPlan3d(R2C) failed");
        if (fft->Plan3d(&ctx->fft_c2r, p->nz, p->ny, p->nx, CUFFT_C2R) != CUFFT_SUCCESS) {
            fft->Destroy(ctx->fft_r2c);
            return lya_fail(ctx, LYA_ECUDA, "lya_fields_from_dm: cufftPlan3d(C2R) failed");
        }
        ctx->fft_dims[0] = p->nz; ctx->fft_dims[1] = p->ny; ctx->fft_dims[2] = p->nx;
    }
    fft->SetStream(ctx->fft_r2c, ctx->stream);
    fft->SetStream(ctx->fft_c2r, ctx->stream);
    if (fft->ExecR2C(ctx->fft_r2c, const_cast<float *>(delta_dm), A) != CUFFT_SUCCESS)
        return lya_fail(ctx, LYA_ECUDA, "lya_fields_from_dm: cufftExecR2C failed");

    double f = 0.0;
    lya_growth_rate(p->z, p->omega_m, &f);
    const double zp1 = 1.0 + p->z;
    const double Hz = 100.0 * p->h * sqrt(p->omega_m * zp1 * zp1 * zp1 + 1.0 - p->omega_m);
    const double eplus = Hz * f / zp1;                                        // km/s per comoving Mpc (U1)
    const double n3 = (double)p->nx * p->ny * p->nz;
    const double dk = 2.0 * M_PI * p->h / p->box_mpch * (double)p->nx;        // 2 pi h / (cell size x n_i), per axis below
    KArgs a;
    memset(&a, 0, sizeof(a));
    a.in = A; a.nxh = nxh; a.nx = p->nx; a.ny = p->ny; a.nz = p->nz;
    a.n_rows = (size_t)p->ny * p->nz;
    a.rows_per_block = KS_ROWS;
    a.dkx = (float)(dk / p->nx); a.dky = (float)(dk / p->ny); a.dkz = (float)(dk / p->nz);
    a.inv_kf2 = p->k_filter_mpc > 0.0 ? (float)(1.0 / (p->k_filter_mpc * p->k_filter_mpc)) : 0.0f;
    a.scale0 = (float)(1.0 / n3);
    a.scale_v = (float)(eplus / n3);
    const size_t n_blocks = (a.n_rows + KS_ROWS - 1) / KS_ROWS;
    if (n_blocks > 0x7fffffffull || (size_t)KS_ROWS * nxh > 0x7fffffffull)
        return lya_fail(ctx, LYA_EINVAL, "lya_fields_from_dm: grid too large");
    if (n_buf == n_out) {                                  // one kernel, then the inverse transforms
        int slot = 0;
        for (int mode = 0; mode < 4; ++mode) a.out[mode] = outs[mode] ? B + (size_t)(slot++) * half : nullptr;
        kspace_kernel<<<(unsigned)n_blocks, KS_THREADS, 0, ctx->stream>>>(a);
        ctx->launches++;
        LYA_CUDA(ctx, cudaGetLastError());
        for (int mode = 0; mode < 4; ++mode)
            if (outs[mode] && fft->ExecC2R(ctx->fft_c2r, a.out[mode], outs[mode]) != CUFFT_SUCCESS)
                return lya_fail(ctx, LYA_ECUDA, "lya_fields_from_dm: cufftExecC2R failed");
        return LYA_OK;
    }
    for (int mode = 0; mode < 4; ++mode) {
        if (!outs[mode]) continue;
        for (int k = 0; k < 4; ++k) a.out[k] = k == mode ? B : nullptr;
        kspace_kernel<<<(unsigned)n_blocks, KS_THREADS, 0, ctx->stream>>>(a);
        ctx->launches++;
        LYA_CUDA(ctx, cudaGetLastError());
        if (fft->ExecC2R(ctx->fft_c2r, B, outs[mode]) != CUFFT_SUCCESS)
            return lya_fail(ctx, LYA_ECUDA, "lya_fields_from_dm: cufftExecC2R failed");
    }
    return LYA_OK;
}

// called by lya_destroy
void lya_fields_release(lya_ctx *ctx)
{
    CufftApi *fft = ctx->fft_dims[0] ? cufft_api() : nullptr;
    if (fft) { fft->Destroy(ctx->fft_r2c); fft->Destroy(ctx->fft_c2r); }
    ctx->fft_dims[0] = 0;
}
