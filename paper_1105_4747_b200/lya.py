"""ctypes binding of the C-ABI library include/lya.h (paper_1105_4747_b200/liblya.so).

Argument marshalling only: every step of the hot path (S1 gas state, S2+S3 tau, S4 normalisation, S5 flux;
PAPER.md:70-92) runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream.  There is
no CPU fallback: if the library is missing it is built with nvcc, and if that fails, or no CUDA device is
present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

from . import build as _build

OK, EINVAL, ECUDA, ENOROOT, ENOCONV, ENOMEM = range(6)
TAU_WINDOWED, TAU_FROM_DENSITY = 1, 2


class LyaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"lya status {status}: {msg}")
        self.status = status


class CParams(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("box_mpch", C.c_double), ("z", C.c_double), ("omega_m", C.c_double), ("h", C.c_double),
                ("omega_b_h2", C.c_double), ("gamma_m12", C.c_double), ("y_he", C.c_double),
                ("T0", C.c_double), ("gamma", C.c_double), ("delta_pivot", C.c_double)]


class CScalars(C.Structure):
    _fields_ = [("n_pix", C.c_int32)] + [(k, C.c_double) for k in
                ("Ez", "Hz", "dR_cm", "dv_kms", "V_kms", "b0_kms", "nbarH", "nbarHI", "K", "tau0", "tauGP")]


class CInstrument(C.Structure):
    _fields_ = [("fwhm_kms", C.c_double), ("bin_kms", C.c_double), ("snr", C.c_double)]


class CFieldParams(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("box_mpch", C.c_double),
                ("h", C.c_double), ("z", C.c_double), ("omega_m", C.c_double), ("k_filter_mpc", C.c_double)]


class CNormalizeStats(C.Structure):
    _fields_ = [("tau_passes", C.c_int32), ("sub_passes", C.c_int32), ("row_pass", C.c_int32), ("n_sub", C.c_uint64)]


class CRootState(C.Structure):
    _fields_ = [("f_target", C.c_double), ("rel_tol", C.c_double), ("n_pix", C.c_double),
                ("lo", C.c_double), ("hi", C.c_double), ("a", C.c_double), ("f_at_a", C.c_double),
                ("iters", C.c_int32), ("done", C.c_int32), ("status", C.c_int32), ("finishing", C.c_int32)]


@dataclass
class Params:
    """The paper's free parameters (include/lya.h: lya_params)."""
    nx: int
    ny: int
    nz: int
    box_mpch: float
    z: float
    T0: float
    gamma: float
    omega_m: float = 0.3
    h: float = 0.7
    omega_b_h2: float = 0.024
    gamma_m12: float = 1.0
    y_he: float = 0.24
    delta_pivot: float = 10.0

    @classmethod
    def from_workload(cls, w) -> "Params":
        return cls(nx=w.n, ny=w.n, nz=w.n, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma,
                   omega_m=w.omega_m, h=w.h, omega_b_h2=w.omega_b_h2, gamma_m12=w.gamma_m12,
                   y_he=w.y_he, delta_pivot=w.delta_pivot)

    def c(self) -> CParams:
        return CParams(self.nx, self.ny, self.nz, self.box_mpch, self.z, self.omega_m, self.h,
                       self.omega_b_h2, self.gamma_m12, self.y_he, self.T0, self.gamma, self.delta_pivot)


EXPORTS = ("lya_version", "lya_status_string", "lya_scalars_from_params", "lya_create", "lya_destroy",
           "lya_last_error", "lya_sm_count", "lya_gas_from_density", "lya_tau_sightlines",
           "lya_normalize_mean_flux", "lya_flux_partial_sums", "lya_root_init", "lya_root_update",
           "lya_flux", "lya_forest_host", "lya_launch_count", "lya_measure_mufu_peak",
           "lya_bin_kms_from_angstrom", "lya_instrument_bins", "lya_observe_rows", "lya_flux_pdf",
           "lya_flux_power_rows", "lya_tau_sightlines_opt", "lya_growth_rate", "lya_fields_from_dm", "lya_flux_moment_sums",
           "lya_root_update_moments", "lya_flux_with_pdf", "lya_forest_host_begin", "lya_forest_moment_sums",
           "lya_forest_host_finish", "lya_measure_hbm_peak", "lya_normalize_mean_flux_rows", "lya_row_moment_sums",
           "lya_set_normalize_subsample", "lya_last_normalize_stats", "lya_flux_moment_sums_sub",
           "lya_forest_moment_sums_sub", "lya_flux_moment_sums_static")

STATIC_MAX_PIX = 1 << 30                                 # LYA_STATIC_MAX_PIX of include/lya.h

_lib = None


def lib() -> C.CDLL:
    """Load (building if stale) liblya.so and declare the signatures of include/lya.h."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, fp, dp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    pp, sp = C.POINTER(CParams), C.POINTER(CScalars)
    L.lya_version.restype = C.c_int
    L.lya_status_string.restype = C.c_char_p
    L.lya_status_string.argtypes = [C.c_int]
    L.lya_scalars_from_params.argtypes = [pp, C.c_int, sp]
    L.lya_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    L.lya_destroy.argtypes = [vp]
    L.lya_destroy.restype = None
    L.lya_last_error.argtypes = [vp]
    L.lya_last_error.restype = C.c_char_p
    L.lya_sm_count.argtypes = [vp]
    L.lya_launch_count.argtypes = [vp]
    L.lya_launch_count.restype = C.c_uint64
    L.lya_gas_from_density.argtypes = [vp, pp, fp, C.c_size_t, fp, fp]
    L.lya_tau_sightlines.argtypes = [vp, pp, C.c_int, C.c_int32, fp, fp, fp, fp]
    L.lya_tau_sightlines_opt.argtypes = [vp, pp, C.c_int, C.c_int32, C.c_uint, fp, fp, fp, fp, C.POINTER(C.c_uint64), vp]
    L.lya_normalize_mean_flux_rows.argtypes = [vp, fp, C.c_size_t, vp, C.c_size_t, C.c_double, C.c_double, C.c_int, dp, dp, ip]
    L.lya_row_moment_sums.argtypes = [vp, vp, C.c_size_t, dp]
    L.lya_normalize_mean_flux.argtypes = [vp, fp, C.c_size_t, C.c_double, C.c_double, C.c_int, dp, dp, ip]
    L.lya_flux_partial_sums.argtypes = [vp, fp, C.c_size_t, dp, C.c_int, dp, dp]
    L.lya_root_init.argtypes = [C.POINTER(CRootState), C.c_double, C.c_double, C.c_double]
    L.lya_root_update.argtypes = [C.POINTER(CRootState), C.c_double, C.c_double]
    L.lya_flux_moment_sums.argtypes = [vp, fp, C.c_size_t, C.c_double, dp]
    L.lya_flux_moment_sums_static.argtypes = [vp, fp, C.c_size_t, C.c_double, vp]
    L.lya_root_update_moments.argtypes = [C.POINTER(CRootState), dp]
    L.lya_flux_moment_sums_sub.argtypes = [vp, fp, C.c_size_t, C.c_double, C.c_int32, dp, C.POINTER(C.c_uint64)]
    L.lya_forest_moment_sums_sub.argtypes = [vp, C.c_double, C.c_int32, dp, C.POINTER(C.c_uint64)]
    L.lya_set_normalize_subsample.argtypes = [vp, C.c_int32, C.c_size_t]
    L.lya_last_normalize_stats.argtypes = [vp, C.POINTER(CNormalizeStats)]
    L.lya_flux.argtypes = [vp, fp, C.c_size_t, C.c_double, fp]
    L.lya_forest_host.argtypes = [vp, pp, C.c_int, C.c_int32, fp, fp, C.c_double, C.c_double, C.c_int,
                                  fp, fp, dp, dp, ip]
    L.lya_forest_host_begin.argtypes = [vp, pp, C.c_int, C.c_int32, fp, fp, fp]
    L.lya_forest_moment_sums.argtypes = [vp, C.c_double, dp]
    L.lya_forest_host_finish.argtypes = [vp, C.c_double, fp]
    L.lya_measure_mufu_peak.argtypes = [vp, dp]
    L.lya_measure_hbm_peak.argtypes = [vp, C.c_size_t, dp]
    L.lya_growth_rate.argtypes = [C.c_double, C.c_double, dp]
    L.lya_fields_from_dm.argtypes = [vp, C.POINTER(CFieldParams), fp, fp, fp, fp, fp]
    L.lya_bin_kms_from_angstrom.argtypes = [C.c_double, C.c_double]
    L.lya_bin_kms_from_angstrom.restype = C.c_double
    L.lya_instrument_bins.argtypes = [C.c_int32, C.c_double, C.POINTER(CInstrument)]
    L.lya_instrument_bins.restype = C.c_int32
    L.lya_observe_rows.argtypes = [vp, C.c_size_t, C.c_int32, C.c_double, C.POINTER(CInstrument), fp, fp, fp]
    L.lya_flux_pdf.argtypes = [vp, fp, C.c_size_t, C.c_int32, C.c_double, C.c_double, C.POINTER(C.c_uint64), dp]
    L.lya_flux_with_pdf.argtypes = [vp, fp, C.c_size_t, C.c_double, fp, C.c_int32, C.c_double, C.c_double,
                                    C.POINTER(C.c_uint64), dp]
    L.lya_flux_power_rows.argtypes = [vp, C.c_size_t, C.c_int32, C.c_double, fp, C.c_double, dp]
    _lib = L
    return L


def bin_kms_from_angstrom(z: float, dlambda: float) -> float:
    return float(lib().lya_bin_kms_from_angstrom(z, dlambda))


def growth_rate(z: float, omega_m: float) -> float:
    f = C.c_double()
    if lib().lya_growth_rate(z, omega_m, C.byref(f)) != OK:
        raise LyaError(EINVAL, "lya_growth_rate: bad arguments")
    return f.value


def scalars(p: Params, axis: int = 0) -> dict:
    """Host-only: the derived scalars of one sightline direction (no GPU needed)."""
    s, cp = CScalars(), p.c()
    st = lib().lya_scalars_from_params(C.byref(cp), axis, C.byref(s))
    if st != OK:
        raise LyaError(st, "lya_scalars_from_params: bad parameters")
    return {k: getattr(s, k) for k, _ in CScalars._fields_}


def _dev(t: torch.Tensor, name: str):
    if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name}: contiguous float32 CUDA tensor required")
    return t.data_ptr() or None                          # an empty tensor has no storage: NULL


def _host(t: torch.Tensor | None, name: str):
    if t is None:
        return None
    if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name}: contiguous float32 host tensor required")
    return t.data_ptr()


class Context:
    """One lya_ctx bound to a CUDA device and to torch's current stream on it."""

    def __init__(self, device: int | None = None, stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise LyaError(ECUDA, "no CUDA device: this library has no CPU path")
        self.device = torch.cuda.current_device() if device is None else int(device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        st = lib().lya_create(C.byref(self._h), self.device, C.c_void_p(self.stream.cuda_stream))
        if st != OK:
            raise LyaError(st, "lya_create failed")

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:      # _lib is None only at interpreter shutdown
            _lib.lya_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, st: int, allow=()):
        if st != OK and st not in allow:
            raise LyaError(st, lib().lya_last_error(self._h).decode())
        return st

    @property
    def sm_count(self) -> int:
        return lib().lya_sm_count(self._h)

    @property
    def launch_count(self) -> int:
        return int(lib().lya_launch_count(self._h))

    def measure_mufu_peak(self) -> float:
        """MUFU.EX2 results per second of this device (the tau kernel's roofline denominator)."""
        r = C.c_double()
        self._check(lib().lya_measure_mufu_peak(self._h, C.byref(r)))
        return r.value

    def measure_hbm_peak(self, n_bytes: int = 1 << 32) -> float:
        """GB/s (read + written bytes) of the library's own 128-bit streaming copy kernel over n_bytes."""
        r = C.c_double()
        self._check(lib().lya_measure_hbm_peak(self._h, n_bytes, C.byref(r)))
        return r.value

    # S1
    def gas_from_density(self, p: Params, delta: torch.Tensor, n_hi=None, b_kms=None):
        n_hi = torch.empty_like(delta) if n_hi is None else n_hi
        b_kms = torch.empty_like(delta) if b_kms is None else b_kms
        cp = p.c()
        self._check(lib().lya_gas_from_density(self._h, C.byref(cp), _dev(delta, "delta"), delta.numel(),
                                               _dev(n_hi, "n_hi"), _dev(b_kms, "b_kms")))
        return n_hi, b_kms

    # S2 + S3
    def tau_sightlines(self, p: Params, axis: int, n_hi, b_kms, v_pec, tau=None, nz_local=None):
        tau = torch.empty_like(n_hi) if tau is None else tau
        nz_local = n_hi.shape[0] if nz_local is None else nz_local
        if n_hi.numel() != nz_local * p.ny * p.nx or b_kms.numel() != n_hi.numel() or \
                v_pec.numel() != n_hi.numel() or tau.numel() != n_hi.numel():
            raise ValueError("tau_sightlines: arrays must be [nz_local][ny][nx]")
        cp = p.c()
        self._check(lib().lya_tau_sightlines(self._h, C.byref(cp), axis, nz_local, _dev(n_hi, "n_hi"),
                                             _dev(b_kms, "b_kms"), _dev(v_pec, "v_pec"), _dev(tau, "tau")))
        return tau

    def tau_sightlines_opt(self, p: Params, axis: int, v_pec, n_hi=None, b_kms=None, delta=None, windowed=False,
                           tau=None, nz_local=None, count_pairs=False, row_moments=None):
        """delta given -> S1 fused into the staging; windowed -> only contributing sources.
        row_moments: float64 CUDA tensor [sightlines][5] that receives the per-sightline plain moments of tau.
        Returns tau, or (tau, pairs evaluated) with count_pairs."""
        first = delta if delta is not None else n_hi
        flags = (TAU_WINDOWED if windowed else 0) | (TAU_FROM_DENSITY if delta is not None else 0)
        tau = torch.empty_like(first) if tau is None else tau
        nz_local = first.shape[0] if nz_local is None else nz_local
        if first.numel() != nz_local * p.ny * p.nx or v_pec.numel() != first.numel() or tau.numel() != first.numel():
            raise ValueError("tau_sightlines_opt: arrays must be [nz_local][ny][nx]")
        if row_moments is not None:
            n_ax = (p.nx, p.ny, p.nz)[axis]
            if not (row_moments.is_cuda and row_moments.dtype == torch.float64 and row_moments.is_contiguous()
                    and row_moments.numel() == 5 * (first.numel() // n_ax)):
                raise ValueError("row_moments: contiguous float64 CUDA tensor [sightlines][5] required")
        cp = p.c()
        pairs = C.c_uint64()
        self._check(lib().lya_tau_sightlines_opt(
            self._h, C.byref(cp), axis, nz_local, flags, _dev(first, "n_hi/delta"),
            None if delta is not None else _dev(b_kms, "b_kms"), _dev(v_pec, "v_pec"), _dev(tau, "tau"),
            C.byref(pairs) if count_pairs else None, None if row_moments is None else row_moments.data_ptr()))
        return (tau, int(pairs.value)) if count_pairs else tau

    # S4
    def normalize_mean_flux(self, tau, f_target: float, rel_tol: float = 1e-7, max_iter: int = 60,
                            allow_noconv: bool = False, row_moments=None):
        """row_moments: what tau_sightlines_opt(row_moments=...) wrote for exactly this tau -- the A = 0 pass then
        reads them instead of tau.  Returns (A, f at A (model value), passes, status)."""
        a, f, it = C.c_double(), C.c_double(), C.c_int()
        if row_moments is None:
            rc = lib().lya_normalize_mean_flux(self._h, _dev(tau, "tau"), tau.numel(), f_target,
                                               rel_tol, max_iter, C.byref(a), C.byref(f), C.byref(it))
        else:
            rc = lib().lya_normalize_mean_flux_rows(self._h, _dev(tau, "tau"), tau.numel(), row_moments.data_ptr(),
                                                    row_moments.numel() // 5, f_target, rel_tol, max_iter,
                                                    C.byref(a), C.byref(f), C.byref(it))
        st = self._check(rc, allow=(ENOCONV,) if allow_noconv else ())
        return a.value, f.value, it.value, st

    def set_normalize_subsample(self, every: int, min_pix: int):
        """S4's nested iteration: subsample stride in 4 KiB chunks (<= 1: off) and the smallest n_pix that uses it."""
        self._check(lib().lya_set_normalize_subsample(self._h, every, min_pix))

    def last_normalize_stats(self) -> dict:
        st = CNormalizeStats()
        self._check(lib().lya_last_normalize_stats(self._h, C.byref(st)))
        return {k: int(getattr(st, k)) for k, _ in CNormalizeStats._fields_}

    def row_moment_sums(self, row_moments):
        s5 = (C.c_double * 5)()
        self._check(lib().lya_row_moment_sums(self._h, row_moments.data_ptr() or None, row_moments.numel() // 5, s5))
        return list(s5)

    def flux_partial_sums(self, tau, a_trials):
        k = len(a_trials)
        at = (C.c_double * k)(*a_trials)
        s, d = (C.c_double * k)(), (C.c_double * k)()
        self._check(lib().lya_flux_partial_sums(self._h, _dev(tau, "tau"), tau.numel(), at, k, s, d))
        return list(s), list(d)

    def flux_moment_sums(self, tau, a_trial: float):
        s5 = (C.c_double * 5)()
        self._check(lib().lya_flux_moment_sums(self._h, _dev(tau, "tau"), tau.numel(), a_trial, s5))
        return list(s5)

    def flux_moment_sums_static(self, tau, a_trial: float, out):
        """lya_flux_moment_sums_static: the five sums into `out` (5 float64 on the device, the caller's), asynchronous; the
        call allocates nothing (static device scratch; at most STATIC_MAX_PIX pixels; overlapping calls race)."""
        if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 5):
            raise TypeError("out: 5 contiguous float64 on the device required")
        self._check(lib().lya_flux_moment_sums_static(self._h, _dev(tau, "tau"), tau.numel(), a_trial, out.data_ptr()))
        return out

    def flux_moment_sums_sub(self, tau, a_trial: float, every: int):
        """The five tilted moments over every `every`-th 4 KiB chunk of tau; returns (sums5, pixels summed over)."""
        s5, ns = (C.c_double * 5)(), C.c_uint64()
        self._check(lib().lya_flux_moment_sums_sub(self._h, _dev(tau, "tau"), tau.numel(), a_trial, every, s5, C.byref(ns)))
        return list(s5), int(ns.value)

    # S5
    def flux(self, tau, a: float, out=None):
        out = torch.empty_like(tau) if out is None else out
        self._check(lib().lya_flux(self._h, _dev(tau, "tau"), tau.numel(), a, _dev(out, "flux")))
        return out

    # after F: instrument model, flux PDF, 1D flux power
    def observe_rows(self, flux, dv_kms: float, fwhm_kms: float = 0.0, bin_kms: float = 0.0, snr: float = 0.0,
                     unit_noise=None, out=None):
        """flux: [..., n_pix] rows.  Returns [n_rows, n_bins]."""
        n_pix = flux.shape[-1]
        n_rows = flux.numel() // n_pix
        inst = CInstrument(fwhm_kms, bin_kms, snr)
        nb = lib().lya_instrument_bins(n_pix, dv_kms, C.byref(inst))
        if nb < 1:
            raise LyaError(EINVAL, "observe_rows: bin wider than the row")
        out = torch.empty((n_rows, nb), dtype=torch.float32, device=flux.device) if out is None else out
        if out.numel() != n_rows * nb or (unit_noise is not None and unit_noise.numel() != n_rows * nb):
            raise ValueError("observe_rows: out / unit_noise must be [n_rows][n_bins]")
        self._check(lib().lya_observe_rows(self._h, n_rows, n_pix, dv_kms, C.byref(inst), _dev(flux, "flux"),
                                           None if unit_noise is None else _dev(unit_noise, "unit_noise"),
                                           _dev(out, "out")))
        return out

    def flux_pdf(self, flux, n_bins: int = 21, f_lo: float = -0.025, width: float = 0.05):
        import numpy as np
        counts = (C.c_uint64 * n_bins)()
        pdf = (C.c_double * n_bins)()
        self._check(lib().lya_flux_pdf(self._h, _dev(flux, "flux"), flux.numel(), n_bins, f_lo, width, counts, pdf))
        return np.array(counts, dtype=np.uint64), np.array(pdf, dtype=np.float64)

    def flux_with_pdf(self, tau, a: float, out=None, n_bins: int = 21, f_lo: float = -0.025, width: float = 0.05):
        """S5 and the flux PDF in one pass: returns (F, counts, pdf)."""
        import numpy as np
        out = torch.empty_like(tau) if out is None else out
        counts = (C.c_uint64 * n_bins)()
        pdf = (C.c_double * n_bins)()
        self._check(lib().lya_flux_with_pdf(self._h, _dev(tau, "tau"), tau.numel(), a, _dev(out, "flux"), n_bins,
                                            f_lo, width, counts, pdf))
        return out, np.array(counts, dtype=np.uint64), np.array(pdf, dtype=np.float64)

    def flux_power_rows(self, flux, dv_kms: float, mean_flux: float):
        import numpy as np
        n_pix = flux.shape[-1]
        P = (C.c_double * (n_pix // 2 + 1))()
        self._check(lib().lya_flux_power_rows(self._h, flux.numel() // n_pix, n_pix, dv_kms, _dev(flux, "flux"),
                                              mean_flux, P))
        return np.array(P, dtype=np.float64)

    # before the hot path: Eq.1 and Eq.3
    def fields_from_dm(self, delta_dm, box_mpch: float, h: float, z: float, omega_m: float, k_filter_mpc: float,
                       want=("delta_b", "v_x", "v_y", "v_z")):
        """delta_dm: [nz][ny][nx] CUDA fp32, box_mpch along x.  Returns a dict of the requested fields."""
        nz, ny, nx = delta_dm.shape
        fpar = CFieldParams(nx, ny, nz, box_mpch, h, z, omega_m, k_filter_mpc)
        out = {k: torch.empty_like(delta_dm) for k in want}
        ptr = lambda k: _dev(out[k], k) if k in out else None
        self._check(lib().lya_fields_from_dm(self._h, C.byref(fpar), _dev(delta_dm, "delta_dm"), ptr("delta_b"),
                                             ptr("v_x"), ptr("v_y"), ptr("v_z")))
        return out

    # S1..S5 from host buffers
    def forest_host(self, p: Params, axis: int, delta_h, v_pec_h, f_target: float, rel_tol: float = 1e-7,
                    max_iter: int = 60, slab_nz: int = 0, tau_h=None, flux_h=None):
        a, f, it = C.c_double(), C.c_double(), C.c_int()
        cp = p.c()
        self._check(lib().lya_forest_host(self._h, C.byref(cp), axis, slab_nz, _host(delta_h, "delta_h"),
                                          _host(v_pec_h, "v_pec_h"), f_target, rel_tol, max_iter,
                                          _host(tau_h, "tau_h"), _host(flux_h, "flux_h"),
                                          C.byref(a), C.byref(f), C.byref(it)))
        return a.value, f.value, it.value


def forest_host_sharded(ctx: Context, p: Params, axis: int, delta_h, v_pec_h, f_target: float, n_pix_global: int,
                        rel_tol: float = 1e-7, max_iter: int = 60, slab_nz: int = 0, tau_h=None, flux_h=None, group=None,
                        sub_every: int = 32):
    """S1..S5 from HOST buffers when every rank holds a z-slab of complete sightlines: lya_forest_host_begin on the
    local slab, S4 over ALL ranks' pixels (five moments per pass, one all-reduce, lya_root_update_moments -- the
    GLOBAL A of PAPER.md:92), lya_forest_host_finish.  Returns (A, f at A (model), passes over all of tau)."""
    cp = p.c()
    ctx._check(lib().lya_forest_host_begin(ctx._h, C.byref(cp), axis, slab_nz, _host(delta_h, "delta_h"),
                                           _host(v_pec_h, "v_pec_h"), _host(tau_h, "tau_h")))

    def sums(a, every):
        s5, ns = (C.c_double * 5)(), C.c_uint64()
        ctx._check(lib().lya_forest_moment_sums_sub(ctx._h, a, every, s5, C.byref(ns)))
        return list(s5), int(ns.value)

    A, f, it = normalize_mean_flux_sharded(ctx, None, f_target, n_pix_global, rel_tol, max_iter, group,
                                           kernel_sums=sums, sub_every=sub_every)
    ctx._check(lib().lya_forest_host_finish(ctx._h, A, _host(flux_h, "flux_h")))
    return A, f, it


def normalize_mean_flux_sharded(ctx: Context, tau_local, f_target: float, n_pix_global: int,
                                rel_tol: float = 1e-7, max_iter: int = 60, group=None, partial_sums=None,
                                row_moments=None, sub_every: int = 32, sub_min_pix: int = 1 << 24, kernel_sums=None,
                                stats: dict | None = None):
    """S4 when the pixels are sharded over ranks (z-slabs per GPU).

    Each pass: the five local tilted moments from lya_flux_moment_sums[_sub], one all-reduce of six doubles (the
    moments and the number of pixels they run over), then the library's scalar update lya_root_update_moments --
    identical on every rank, so all ranks hold the same A.  The passes are nested as in lya_normalize_mean_flux: the
    A = 0 pass from `row_moments` (the local tau's per-sightline plain moments, tau_sightlines_opt) if given; for
    n_pix_global >= sub_min_pix the whole iteration on every sub_every-th 4 KiB chunk of each rank's tau to 1e-3;
    then passes over all of tau from there until the full iteration's own stopping rule holds (normally one).
    `partial_sums` lets a CPU test (gloo) stand in for the kernel (no subsample then); the product path leaves it None.
    `kernel_sums(a, every) -> (sums5, pixels)` replaces lya_flux_moment_sums_sub (forest_host_sharded's resident tau).
    Returns (A, f at A (model value), passes over all of tau); `stats` receives the pass counts.
    """
    import torch.distributed as dist
    L = lib()

    def all_reduce(vals):
        buf = torch.tensor(vals, dtype=torch.float64)
        if dist.is_available() and dist.is_initialized():
            if dist.get_backend(group) == "nccl":
                buf = buf.cuda()
            dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
            buf = buf.cpu()
        return [float(x) for x in buf]

    def local_sums(a, every):
        if kernel_sums is not None:
            return kernel_sums(a, every)
        if a == 0.0 and every <= 1 and row_moments is not None:
            return ctx.row_moment_sums(row_moments), tau_local.numel()
        return ctx.flux_moment_sums_sub(tau_local, a, every)

    def new_state(tol, n_pix, a0=0.0):
        st = CRootState()
        if L.lya_root_init(C.byref(st), f_target, tol, float(n_pix)) != OK:
            raise LyaError(EINVAL, "lya_root_init: bad arguments")
        st.a = a0
        return st

    def update(st, sums5):
        rc = L.lya_root_update_moments(C.byref(st), (C.c_double * 5)(*sums5))
        if rc == ENOROOT:
            raise LyaError(rc, "no A > 0 reaches f_target")

    st = new_state(rel_tol, n_pix_global)
    n_full = n_sub_passes = n_sub_local = 0
    if partial_sums is not None:                         # CPU stand-in: plain loop, five moments or the two-sum rule
        while not st.done and st.iters < max_iter:
            got = partial_sums(st.a)
            if len(got) == 5:
                update(st, all_reduce(list(got)))
            else:
                s = all_reduce([got[0][0], got[1][0]])
                if L.lya_root_update(C.byref(st), s[0], s[1]) == ENOROOT:
                    raise LyaError(ENOROOT, "no A > 0 reaches f_target")
        return st.a, st.f_at_a, st.iters

    use_sub = sub_every > 1 and n_pix_global >= sub_min_pix
    if row_moments is not None or kernel_sums is not None or not use_sub:
        s5, _ = local_sums(0.0, 1)                       # the A = 0 pass (row moments when there are some)
        update(st, all_reduce(s5))
        n_full += 1
    if use_sub and not st.done:
        a0, ss = st.a, None
        while n_sub_passes < 12:
            s5, npx = local_sums(a0 if ss is None else ss.a, sub_every)
            n_sub_local = npx
            red = all_reduce(s5 + [float(npx)])
            if ss is None:
                if red[5] < 1.0:
                    break                                 # nothing in the subsample
                ss = new_state(max(1e-3, rel_tol), red[5], a0)
            rc = L.lya_root_update_moments(C.byref(ss), (C.c_double * 5)(*red[:5]))
            n_sub_passes += 1
            if rc != OK:
                ss = None
                break
            if ss.done:
                break
        if ss is not None and 0.0 < ss.a < 1e30:
            st = new_state(rel_tol, n_pix_global, ss.a)
    while not st.done and n_full < max_iter:
        s5, _ = local_sums(st.a, 1)
        update(st, all_reduce(s5))
        n_full += 1
    if stats is not None:
        stats.update(tau_passes=n_full, sub_passes=n_sub_passes, n_sub=n_sub_local)
    return st.a, st.f_at_a, n_full
