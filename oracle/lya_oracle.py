"""ctypes wrapper of oracle/lya_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It shares nothing with paper_1105_4747_b200/ (no imports either way);
it takes plain numpy arrays and the same free parameters the paper names
(T0, gamma, z, cosmology, <F>).

Argument marshalling only: every arithmetic step of the method is in lya_oracle.c.  The
axis handling below is pure indexing (numpy moveaxis/reshape): a sightline along axis a of
a C-order [nz][ny][nx] grid becomes one contiguous row.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lya_oracle.c")
_LIB = os.path.join(_HERE, "liblya_oracle.so")


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math) + OpenMP -> oracle/liblya_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c99", "-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp",
               "-shared", "-fPIC", "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("n_pix", C.c_int32), ("box_mpch", C.c_double), ("z", C.c_double),
                ("omega_m", C.c_double), ("h", C.c_double), ("omega_b_h2", C.c_double),
                ("gamma_m12", C.c_double), ("y_he", C.c_double), ("T0", C.c_double),
                ("gamma", C.c_double), ("delta_pivot", C.c_double)]


class _Scalars(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("Ez", "Hz", "dR_cm", "dv_kms", "V_kms", "b0_kms", "nbarH", "nbarHI", "K",
                 "tau0", "tauGP")]


@dataclass
class Params:
    """The paper's free parameters for one sightline direction."""
    n_pix: int
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
        """`w`: any object with the attribute names of paper_1105_4747_b200.workloads.Workload."""
        return cls(n_pix=w.n, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma,
                   omega_m=w.omega_m, h=w.h, omega_b_h2=w.omega_b_h2, gamma_m12=w.gamma_m12,
                   y_he=w.y_he, delta_pivot=w.delta_pivot)

    def _c(self) -> _Params:
        return _Params(self.n_pix, self.box_mpch, self.z, self.omega_m, self.h, self.omega_b_h2,
                       self.gamma_m12, self.y_he, self.T0, self.gamma, self.delta_pivot)


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, fp = C.POINTER(C.c_double), C.POINTER(C.c_float)
        L.orc_threads.restype = C.c_int
        L.orc_scalars_from_params.argtypes = [C.POINTER(_Params), C.POINTER(_Scalars)]
        L.orc_gas_from_density.argtypes = [C.POINTER(_Params), fp, C.c_size_t, dp, dp, dp]
        L.orc_tau_sightlines.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_size_t,
                                         dp, dp, fp, dp, C.c_int]
        L.orc_mean_flux.argtypes = [dp, C.c_size_t, C.c_double]
        L.orc_mean_flux.restype = C.c_double
        L.orc_normalize_mean_flux.argtypes = [dp, C.c_size_t, C.c_double, dp, dp,
                                              C.POINTER(C.c_int)]
        L.orc_flux.argtypes = [dp, C.c_size_t, C.c_double, dp]
        _lib = L
    return _lib


def threads() -> int:
    return int(lib().orc_threads())


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def scalars(p: Params) -> dict:
    s = _Scalars()
    cp = p._c()
    if lib().orc_scalars_from_params(C.byref(cp), C.byref(s)):
        raise ValueError("orc_scalars_from_params: bad parameters")
    return {k: getattr(s, k) for k, _ in _Scalars._fields_}


def gas_from_density(p: Params, delta: np.ndarray):
    """S1: fp32 delta (any shape) -> (T [K], n_HI [cm^-3], b [km/s]) as float64 arrays."""
    d = np.ascontiguousarray(delta, dtype=np.float32)
    T = np.empty(d.shape, np.float64)
    n = np.empty(d.shape, np.float64)
    b = np.empty(d.shape, np.float64)
    cp = p._c()
    if lib().orc_gas_from_density(C.byref(cp), _f(d), d.size, _d(T), _d(n), _d(b)):
        raise ValueError("orc_gas_from_density failed")
    return T, n, b


def tau_rows(p: Params, n_hi, b_kms, v_pec, mode: int = 0) -> np.ndarray:
    """S2+S3 on sightlines stored as rows: arrays [..., n_pix] -> tau float64, same shape."""
    s = scalars(p)
    n = np.ascontiguousarray(n_hi, dtype=np.float64)
    b = np.ascontiguousarray(b_kms, dtype=np.float64)
    v = np.ascontiguousarray(v_pec, dtype=np.float32)
    assert n.shape == b.shape == v.shape and n.shape[-1] == p.n_pix
    tau = np.empty(n.shape, np.float64)
    rc = lib().orc_tau_sightlines(s["K"], s["dv_kms"], p.n_pix, n.size // p.n_pix,
                                  _d(n), _d(b), _f(v), _d(tau), int(mode))
    if rc:
        raise ValueError("orc_tau_sightlines failed")
    return tau


def to_rows(a: np.ndarray, axis: int) -> np.ndarray:
    """[nz][ny][nx] grid -> sightlines along `axis` (0=x, 1=y, 2=z) as the last dimension."""
    return np.ascontiguousarray(np.moveaxis(a, 2 - axis, -1))


def from_rows(r: np.ndarray, axis: int) -> np.ndarray:
    return np.ascontiguousarray(np.moveaxis(r, -1, 2 - axis))


def tau_grid(p: Params, axis: int, n_hi, b_kms, v_pec, mode: int = 0) -> np.ndarray:
    """S2+S3 on a [nz][ny][nx] grid with sightlines along `axis`; returns tau in grid layout."""
    t = tau_rows(p, to_rows(np.asarray(n_hi), axis), to_rows(np.asarray(b_kms), axis),
                 to_rows(np.asarray(v_pec), axis), mode)
    return from_rows(t, axis)


def mean_flux(tau: np.ndarray, A: float) -> float:
    t = np.ascontiguousarray(tau, dtype=np.float64).reshape(-1)
    return float(lib().orc_mean_flux(_d(t), t.size, float(A)))


def normalize_mean_flux(tau: np.ndarray, f_target: float):
    """S4: returns (A, <F> achieved, iterations)."""
    t = np.ascontiguousarray(tau, dtype=np.float64).reshape(-1)
    A, f, it = C.c_double(), C.c_double(), C.c_int()
    rc = lib().orc_normalize_mean_flux(_d(t), t.size, float(f_target), C.byref(A), C.byref(f),
                                       C.byref(it))
    if rc == 3:
        raise ArithmeticError("no root: f_target below the zero-tau fraction")
    if rc:
        raise ValueError("orc_normalize_mean_flux: bad arguments")
    return A.value, f.value, it.value


def flux(tau: np.ndarray, A: float) -> np.ndarray:
    t = np.ascontiguousarray(tau, dtype=np.float64)
    F = np.empty(t.shape, np.float64)
    if lib().orc_flux(_d(t.reshape(-1)), t.size, float(A), _d(F.reshape(-1))):
        raise ValueError("orc_flux failed")
    return F


def run_path(p: Params, axis: int, delta, v_pec, f_target: float, mode: int = 0) -> dict:
    """S1 -> S5 in the paper's order on one grid; everything float64."""
    _, n, b = gas_from_density(p, delta)
    tau = tau_grid(p, axis, n, b, v_pec, mode)
    A, f, it = normalize_mean_flux(tau, f_target)
    return {"n_hi": n, "b": b, "tau": tau, "A": A, "f_achieved": f, "iters": it,
            "flux": flux(tau, A)}
