"""Upstream fields of arXiv:1105.4747, sections 2.1-2.2 -- TEST INFRASTRUCTURE, NOT PRODUCT.

    Eq.1   delta_b(k) = delta_DM(k) / (1 + k^2 / k_F^2)            Jeans / pressure filtering
    Eq.3   v(k) = E_+ i k / k^2 delta_DM(k),  E_+ = H(z) f D_+ / (1+z)
                         f = -dln D_+ / dln(1+z)                                   linear peculiar velocity

Plain numpy in double precision; the 3D FFT is the library primitive numpy.fft (a step, not the method).  Only
tests/ may import this module; it shares nothing with paper_1105_4747_b200/.

Readings: U1 the input delta_DM is the field ALREADY evolved to redshift z, so D_+ is
folded into it and E_+ reduces to H(z) f(z) / (1+z), in km/s per comoving Mpc; U2 k is the comoving wavevector
in Mpc^-1, k_i = 2 pi m_i h / L with signed integer m_i in [-N_i/2, N_i/2) and L in h^-1 Mpc; k_F is given in
the same units (paper: 6.5 Mpc^-1); U3 Fourier convention of numpy / cuFFT (forward e^{-ikx}), for which
continuity gives v(k) = +i a H f k/k^2 delta(k), i.e. the paper's sign; U4 the k = 0 mode of v is zero, and
so is the Nyquist plane of the component being differentiated (m_a = -N_a/2, whose i k_a would break the
Hermitian symmetry of a real field) -- Eq.1 keeps every mode; U5 the output velocity is the proper peculiar
velocity in km/s along +axis, the convention lya_tau_sightlines takes (C11).
"""
from __future__ import annotations

import numpy as np


def E_of_z(z: float, omega_m: float) -> float:
    return float(np.sqrt(omega_m * (1.0 + z) ** 3 + 1.0 - omega_m))


def growth_rate(z: float, omega_m: float) -> float:
    """f = dlnD/dlna for flat LCDM, from D(a) ~ H(a) int_0^a da' / (a' H(a'))^3 (Heath 1977), by quadrature."""
    from scipy.integrate import quad
    a = 1.0 / (1.0 + z)
    E = lambda x: np.sqrt(omega_m / x ** 3 + 1.0 - omega_m)
    integral, _ = quad(lambda x: 1.0 / (x * E(x)) ** 3, 0.0, a, epsabs=0.0, epsrel=1e-13)
    dlnE = -1.5 * omega_m / a ** 3 / E(a) ** 2
    return float(dlnE + a / (a * E(a)) ** 3 / integral)


def wavevectors(shape, box_mpch, h):
    """k_z, k_y, k_x [Mpc^-1, comoving] broadcastable over a [nz][ny][nx] grid; box_mpch = (Lz, Ly, Lx)."""
    ks = []
    for ax, (n, L) in enumerate(zip(shape, box_mpch)):
        m = np.fft.fftfreq(n, d=1.0 / n)                         # signed integers, -n/2 at the Nyquist slot
        k = 2.0 * np.pi * m * h / L
        sh = [1, 1, 1]
        sh[ax] = n
        ks.append(k.reshape(sh))
    return ks


def fields_from_dm(delta_dm, box_mpch, h, z, omega_m, k_filter_mpc):
    """Returns delta_b and (v_x, v_y, v_z) [km/s] in double.  box_mpch: scalar (cubic cells) or (Lz, Ly, Lx)."""
    d = np.asarray(delta_dm, dtype=np.float64)
    nz, ny, nx = d.shape
    if np.isscalar(box_mpch):
        box_mpch = (box_mpch * nz / nx, box_mpch * ny / nx, float(box_mpch))
    kz, ky, kx = wavevectors(d.shape, box_mpch, h)
    k2 = kz ** 2 + ky ** 2 + kx ** 2
    dk = np.fft.fftn(d)
    db = np.fft.ifftn(dk / (1.0 + k2 / k_filter_mpc ** 2)).real if k_filter_mpc > 0 else d.copy()
    eplus = 100.0 * h * E_of_z(z, omega_m) * growth_rate(z, omega_m) / (1.0 + z)     # km/s/Mpc
    k2s = np.where(k2 > 0, k2, 1.0)
    vs = []
    for ax, (k, n) in enumerate(((kx, nx), (ky, ny), (kz, nz))):
        fac = 1j * k / k2s
        fac = np.where(k2 > 0, fac, 0.0)
        if n % 2 == 0:                                            # U4: drop the Nyquist plane of this axis
            m = np.fft.fftfreq(n, d=1.0 / n)
            sh = [1, 1, 1]
            sh[2 - ax] = n
            fac = fac * (m != -n / 2).reshape(sh)
        vs.append(eplus * np.fft.ifftn(fac * dk).real)
    return db, tuple(vs)
