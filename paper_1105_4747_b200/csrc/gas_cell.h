// gas_cell.h -- S1 per cell (Eq.4, Eq.5 with pivot, Doppler parameter), shared by gas.cu
// (lya_gas_from_density) and tau.cu (LYA_TAU_FROM_DENSITY: S1 fused into the staging of S3) so that both give
// bit-identical n_HI and b.
//
//   D   = 1 + delta                      Dt = min(D, pivot)
//   T   = T0 Dt^(gamma-1)                                              (Eq.5)
//   b   = sqrt(2 kB T / m_p) = b0 Dt^((gamma-1)/2)
//   nHI = nbarHI (T/T0)^-0.7 D^2 = nbarHI Dt^(-1.4 (gamma-1)/2) D^2    (Eq.4 with the local T: reading C4)
#pragma once

struct GasK {
    float nbar_hi;   // Eq.4 at delta = 0, T = T0 [cm^-3]
    float b0;        // km/s
    float h;         // (gamma-1)/2
    float e_n;       // -0.7 (gamma-1)
    float pivot;     // +inf when disabled
};

__device__ __forceinline__ void gas_cell(const GasK &k, float delta, float &n_hi, float &b)
{
    float D  = 1.0f + delta;
    float Dt = fminf(D, k.pivot);
    float l  = log2f(Dt);                       // full-precision log2 (the kernels stay HBM / MUFU.EX2 bound)
    b    = k.b0 * exp2f(k.h * l);
    n_hi = (k.nbar_hi * exp2f(k.e_n * l)) * (D * D);
}
