"""Pins of oracle/lya_fields_oracle.py (Eq.1 and Eq.3) against closed forms."""
import numpy as np
import pytest

from oracle import lya_fields_oracle as fo


def test_growth_rate_closed_forms():
    assert fo.growth_rate(0.0, 1.0) == pytest.approx(1.0, abs=1e-10)          # Einstein-de Sitter: D = a
    assert fo.growth_rate(5.0, 1.0) == pytest.approx(1.0, abs=1e-10)
    for z in (0.0, 1.0, 2.5):                                                  # Linder (2005): f ~ Omega_m(z)^0.55
        om_z = 0.3 * (1 + z) ** 3 / fo.E_of_z(z, 0.3) ** 2
        assert fo.growth_rate(z, 0.3) == pytest.approx(om_z ** 0.55, rel=6e-3)
    # against a finite difference of D(a) = E(a) int da'/(a' E)^3 done here by the trapezoid rule
    def D(a, om=0.3, n=200001):
        x = np.linspace(1e-8, a, n)
        y = 1.0 / (x * np.sqrt(om / x ** 3 + 1 - om)) ** 3
        return np.sqrt(om / a ** 3 + 1 - om) * np.sum(0.5 * (y[1:] + y[:-1]) * np.diff(x))
    a = 1 / 3.5
    f_fd = (np.log(D(a * 1.001)) - np.log(D(a / 1.001))) / (2 * np.log(1.001))
    assert fo.growth_rate(2.5, 0.3) == pytest.approx(f_fd, rel=1e-5)


def test_plane_wave_closed_forms():
    """delta = eps cos(k0 . x): delta_b = delta / (1 + k0^2/kF^2); v = -E+ eps sin(k0 . x) k0 / k0^2."""
    nz, ny, nx, L, h, z, om, kF = 16, 24, 32, 40.0, 0.7, 2.5, 0.3, 6.5
    mz, my, mx = 1, -2, 3
    zz, yy, xx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    phase = 2 * np.pi * (mz * zz / nz + my * yy / ny + mx * xx / nx)
    d = 0.1 * np.cos(phase)
    box = (L * nz / nx, L * ny / nx, L)
    k0 = np.array([2 * np.pi * mz * h / box[0], 2 * np.pi * my * h / box[1], 2 * np.pi * mx * h / box[2]])
    k0sq = (k0 ** 2).sum()
    db, (vx, vy, vz) = fo.fields_from_dm(d, L, h, z, om, kF)
    assert np.allclose(db, d / (1 + k0sq / kF ** 2), atol=1e-15)
    eplus = 100 * h * fo.E_of_z(z, om) * fo.growth_rate(z, om) / (1 + z)
    for v, k in ((vz, k0[0]), (vy, k0[1]), (vx, k0[2])):
        assert np.allclose(v, -eplus * 0.1 * np.sin(phase) * k / k0sq, atol=1e-12)


def test_continuity_and_zero_modes():
    """i k . v(k) = -E+ delta(k) for every mode off the Nyquist planes; mean(v) = 0; kF -> inf is the identity."""
    rng = np.random.default_rng(0)
    d = rng.normal(0, 1, (8, 12, 10))
    L, h, z, om = 25.0, 0.7, 3.0, 0.3
    db, (vx, vy, vz) = fo.fields_from_dm(d, L, h, z, om, 1e9)
    assert np.allclose(db, d, atol=1e-12)
    assert abs(vx.mean()) < 1e-12 and abs(vy.mean()) < 1e-12 and abs(vz.mean()) < 1e-12
    kz, ky, kx = fo.wavevectors(d.shape, (L * 8 / 10, L * 12 / 10, L), h)
    div = 1j * (kx * np.fft.fftn(vx) + ky * np.fft.fftn(vy) + kz * np.fft.fftn(vz))
    eplus = 100 * h * fo.E_of_z(z, om) * fo.growth_rate(z, om) / (1 + z)
    mzz, myy, mxx = np.meshgrid(np.fft.fftfreq(8, 1 / 8), np.fft.fftfreq(12, 1 / 12), np.fft.fftfreq(10, 1 / 10), indexing="ij")
    ok = (mzz != -4) & (myy != -6) & (mxx != -5) & ((mzz != 0) | (myy != 0) | (mxx != 0))
    assert np.allclose(div[ok], -eplus * np.fft.fftn(d)[ok], rtol=1e-10, atol=1e-9)


def test_filter_damps_small_scales_only():
    rng = np.random.default_rng(1)
    d = rng.normal(0, 1, (16, 16, 16))
    db, _ = fo.fields_from_dm(d, 10.0, 0.7, 3.0, 0.3, 6.5)
    P, Pb = np.abs(np.fft.fftn(d)) ** 2, np.abs(np.fft.fftn(db)) ** 2
    kz, ky, kx = fo.wavevectors(d.shape, (10.0, 10.0, 10.0), 0.7)
    k2 = kz ** 2 + ky ** 2 + kx ** 2
    assert np.allclose(Pb, P / (1 + k2 / 6.5 ** 2) ** 2, rtol=1e-10)
    assert db.mean() == pytest.approx(d.mean(), abs=1e-14)                       # k = 0 untouched
