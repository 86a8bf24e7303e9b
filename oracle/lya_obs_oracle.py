"""ctypes wrapper of oracle/lya_obs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.

Instrument model, flux PDF and 1D flux power spectrum
 in plain double precision.  Only tests/ may import this module; it shares nothing with
paper_1105_4747_b200/.  Argument marshalling only: the arithmetic is in lya_obs_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lya_obs_oracle.c")
_LIB = os.path.join(_HERE, "liblya_obs_oracle.so")
_lib = None

C_KMS = 299792.458            # speed of light [km/s]
LYA_ANGSTROM = 1215.67        # rest wavelength of Lyman alpha [Angstrom]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-std=c99", "-O2", "-fno-fast-math", "-ffp-contract=off", "-shared", "-fPIC",
                        "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"], check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, fp = C.POINTER(C.c_double), C.POINTER(C.c_float)
        L.obs_convolve_rows.argtypes = [C.c_int32, C.c_size_t, C.c_double, C.c_double, dp, dp]
        L.obs_n_bins.argtypes = [C.c_int32, C.c_double, C.c_double]
        L.obs_n_bins.restype = C.c_int32
        L.obs_rebin_rows.argtypes = [C.c_int32, C.c_size_t, C.c_double, C.c_double, dp, dp]
        L.obs_add_noise.argtypes = [C.c_size_t, C.c_double, dp, fp, dp]
        L.obs_flux_pdf.argtypes = [fp, C.c_size_t, C.c_int32, C.c_double, C.c_double,
                                   C.POINTER(C.c_uint64), dp]
        L.obs_flux_pdf_edge.argtypes = [C.c_int32, C.c_double, C.c_double]
        L.obs_flux_pdf_edge.restype = C.c_double
        L.obs_flux_power.argtypes = [C.c_int32, C.c_size_t, C.c_double, dp, C.c_double, dp]
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def bin_kms_from_angstrom(z: float, dlambda: float) -> float:
    """Velocity width of a wavelength bin at the observed Lyman-alpha wavelength 1215.67 (1+z) Angstrom."""
    return C_KMS * dlambda / (LYA_ANGSTROM * (1.0 + z))


def convolve_rows(F, dv_kms: float, fwhm_kms: float) -> np.ndarray:
    F = _d(F)
    out = np.empty_like(F)
    rc = lib().obs_convolve_rows(F.shape[-1], F.size // F.shape[-1], dv_kms, fwhm_kms, _p(F, C.c_double),
                                 _p(out, C.c_double))
    assert rc == 0
    return out


def n_bins(n_pix: int, dv_kms: float, bin_kms: float) -> int:
    return int(lib().obs_n_bins(n_pix, dv_kms, bin_kms))


def rebin_rows(Fc, dv_kms: float, bin_kms: float) -> np.ndarray:
    Fc = _d(Fc)
    n = Fc.shape[-1]
    out = np.empty(Fc.shape[:-1] + (n_bins(n, dv_kms, bin_kms),), dtype=np.float64)
    rc = lib().obs_rebin_rows(n, Fc.size // n, dv_kms, bin_kms, _p(Fc, C.c_double), _p(out, C.c_double))
    assert rc == 0
    return out


def add_noise(Fb, snr: float, unit_noise) -> np.ndarray:
    Fb = _d(Fb)
    out = np.empty_like(Fb)
    un = None if unit_noise is None else np.ascontiguousarray(unit_noise, dtype=np.float32)
    rc = lib().obs_add_noise(Fb.size, snr, _p(Fb, C.c_double), None if un is None else _p(un, C.c_float),
                             _p(out, C.c_double))
    assert rc == 0
    return out


def observe_rows(F, dv_kms: float, fwhm_kms: float, bin_kms: float, snr: float, unit_noise=None) -> np.ndarray:
    """The whole instrument model in the paper's order: convolve, resample, add noise."""
    return add_noise(rebin_rows(convolve_rows(F, dv_kms, fwhm_kms), dv_kms, bin_kms), snr, unit_noise)


def flux_pdf(F, nbins: int = 21, f_lo: float = -0.025, width: float = 0.05):
    F = np.ascontiguousarray(F, dtype=np.float32).ravel()
    counts = np.zeros(nbins, dtype=np.uint64)
    pdf = np.zeros(nbins, dtype=np.float64)
    rc = lib().obs_flux_pdf(_p(F, C.c_float), F.size, nbins, f_lo, width, _p(counts, C.c_uint64),
                            _p(pdf, C.c_double))
    assert rc == 0
    return counts, pdf


def flux_pdf_edge(b: int, f_lo: float = -0.025, width: float = 0.05) -> float:
    """Lower edge of bin b as the oracle compares against it."""
    return float(lib().obs_flux_pdf_edge(b, f_lo, width))


def flux_power(F, dv_kms: float, mean_flux: float) -> np.ndarray:
    F = _d(F)
    n = F.shape[-1]
    P = np.empty(n // 2 + 1, dtype=np.float64)
    rc = lib().obs_flux_power(n, F.size // n, dv_kms, _p(F, C.c_double), mean_flux, _p(P, C.c_double))
    assert rc == 0
    return P
