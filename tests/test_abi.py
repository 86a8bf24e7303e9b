"""C-ABI library (include/lya.h): loads, exports every declared symbol, host-only entry points behave.
CPU only (-m "not gpu"): no compute call is made here."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest
import torch

from paper_1105_4747_b200 import lya
from paper_1105_4747_b200.workloads import WORKLOADS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lya.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lya_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    L = lya.lib()
    names = declared_symbols()
    assert len(names) >= 16
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/lya.h but not exported"
    assert set(names) == set(lya.EXPORTS)
    assert L.lya_version() == 100
    assert L.lya_status_string(3) == b"no root"


def test_scalars_match_independent_formulas():
    # retyped here from the paper's definitions (Eq.4, Eq.6 text PAPER.md:88-90), cgs
    KB, MP, MH = 1.380649e-16, 1.67262192369e-24, 1.6735575e-24
    MPC, CL, RHOC = 3.0856775814913673e24, 2.99792458e10, 1.87834e-29
    for cfg, w in WORKLOADS.items():
        s = lya.scalars(lya.Params.from_workload(w), 0)
        Ez = math.sqrt(w.omega_m * (1 + w.z) ** 3 + 1 - w.omega_m)
        dR = w.box_mpch / (w.n * w.h * (1 + w.z)) * MPC
        nH = (1 - w.y_he) * w.omega_b_h2 * RHOC * (1 + w.z) ** 3 / MH
        nHI = 7.24e-6 * nH * (w.T0 / 1e4) ** -0.7 * (w.omega_b_h2 / 0.024) / w.gamma_m12 * ((1 + w.z) / 4) ** 3
        K = CL * 4.48e-18 * dR / math.sqrt(math.pi)
        b0 = math.sqrt(2 * KB * w.T0 / MP) / 1e5
        exp = {"Ez": Ez, "Hz": 100 * w.h * Ez, "dR_cm": dR, "dv_kms": 100 * Ez * w.box_mpch / (w.n * (1 + w.z)),
               "V_kms": 100 * Ez * w.box_mpch / (1 + w.z), "b0_kms": b0, "nbarH": nH, "nbarHI": nHI, "K": K,
               "tau0": K * nHI / (b0 * 1e5), "tauGP": CL * 4.48e-18 * nHI / (100 * w.h * Ez * 1e5 / MPC)}
        assert s["n_pix"] == w.n
        for k, v in exp.items():
            assert abs(s[k] / v - 1) < 1e-13, (cfg, k)


def test_scalars_agree_with_oracle(oracle):
    # two independent implementations (library host code, oracle C) of the same definitions
    for w in WORKLOADS.values():
        a = lya.scalars(lya.Params.from_workload(w), 0)
        b = oracle.scalars(oracle.Params.from_workload(w))
        for k, v in b.items():
            assert abs(a[k] / v - 1) < 1e-13, k


def test_scalars_axis_and_bad_arguments():
    p = lya.Params(nx=32, ny=48, nz=64, box_mpch=10.0, z=2.0, T0=1e4, gamma=1.4)
    assert [lya.scalars(p, ax)["n_pix"] for ax in (0, 1, 2)] == [32, 48, 64]
    L = lya.lib()
    s, cp = lya.CScalars(), p.c()
    assert L.lya_scalars_from_params(C.byref(cp), 3, C.byref(s)) == lya.EINVAL
    assert L.lya_scalars_from_params(None, 0, C.byref(s)) == lya.EINVAL
    for field, bad in (("T0", 0.0), ("box_mpch", -1.0), ("h", 0.0), ("gamma_m12", 0.0), ("nx", 0)):
        q = lya.Params(nx=32, ny=48, nz=64, box_mpch=10.0, z=2.0, T0=1e4, gamma=1.4)
        setattr(q, field, bad)
        cq = q.c()
        assert L.lya_scalars_from_params(C.byref(cq), 0, C.byref(s)) == lya.EINVAL, field


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_device_means_failure_not_fallback():
    h = C.c_void_p()
    assert lya.lib().lya_create(C.byref(h), 0, None) == lya.ECUDA
    assert not h.value
    with pytest.raises(lya.LyaError):
        lya.Context()
    # null context: every compute entry point refuses
    L = lya.lib()
    assert L.lya_flux(None, None, 0, 1.0, None) == lya.EINVAL
    assert L.lya_tau_sightlines(None, None, 0, 1, None, None, None, None) == lya.EINVAL
    assert L.lya_gas_from_density(None, None, None, 0, None, None) == lya.EINVAL
    assert L.lya_normalize_mean_flux(None, None, 0, 0.5, 1e-7, 10, None, None, None) == lya.EINVAL
    assert L.lya_forest_host(None, None, 0, 0, None, None, 0.5, 1e-7, 10, None, None, None, None, None) == lya.EINVAL
    assert L.lya_launch_count(None) == 0 and L.lya_sm_count(None) == 0


def _drive_root(tau, f_target, rel_tol=1e-12, max_iter=200):
    """Host-side root iteration fed with numpy sums (stand-in for lya_flux_partial_sums on the CPU box)."""
    L, st = lya.lib(), lya.CRootState()
    assert L.lya_root_init(C.byref(st), f_target, rel_tol, float(tau.size)) == lya.OK
    while not st.done and st.iters < max_iter:
        e = np.exp(-st.a * tau)
        rc = L.lya_root_update(C.byref(st), float(e.sum()), float((tau * e).sum()))
        if rc != lya.OK:
            return rc, st
    return lya.OK, st


def test_root_iteration_closed_forms():
    # P9's closed forms, applied to the library's host-side iteration
    rc, st = _drive_root(np.full(1000, 0.7), 0.8)
    assert rc == lya.OK and st.done and abs(st.a / (-math.log(0.8) / 0.7) - 1) < 1e-11
    assert abs(st.f_at_a - 0.8) < 1e-11
    tau = np.concatenate([np.full(500, 0.4), np.full(500, 0.8)])
    x = (-1 + math.sqrt(1 + 8 * 0.72)) / 2
    rc, st = _drive_root(tau, 0.72)
    assert rc == lya.OK and abs(st.a / (-math.log(x) / 0.4) - 1) < 1e-11
    assert st.iters <= 12                      # Newton, not 45 bisections


def test_root_iteration_matches_oracle(oracle):
    rng = np.random.default_rng(5)
    tau = np.exp(rng.normal(-0.5, 1.5, 20000))
    tau[::7] = 0.0
    A, f, _ = oracle.normalize_mean_flux(tau, 0.8)
    rc, st = _drive_root(tau, 0.8)
    assert rc == lya.OK and abs(st.a / A - 1) < 1e-10 and abs(st.f_at_a - 0.8) < 1e-10


def test_root_iteration_no_root_and_bad_arguments():
    L, st = lya.lib(), lya.CRootState()
    rc, st = _drive_root(np.zeros(100), 0.8)
    assert rc == lya.ENOROOT and st.done
    tau = np.concatenate([np.zeros(90), np.ones(10)])     # f(inf) = 0.9 > 0.8: no root
    rc, st = _drive_root(tau, 0.8, max_iter=400)
    assert rc == lya.ENOROOT
    for ft in (0.0, 1.0, -0.1, float("nan")):
        assert L.lya_root_init(C.byref(st), ft, 1e-7, 10.0) == lya.EINVAL
    assert L.lya_root_init(C.byref(st), 0.5, 0.0, 10.0) == lya.EINVAL
    assert L.lya_root_init(None, 0.5, 1e-7, 10.0) == lya.EINVAL


def test_params_struct_layout_matches_header():
    # nx,ny,nz (3 x int32) + padding to 8, then 10 doubles
    assert C.sizeof(lya.CParams) == 16 + 10 * 8
    assert C.sizeof(lya.CScalars) == 8 + 11 * 8
    assert C.sizeof(lya.CRootState) == 7 * 8 + 4 * 4


def test_root_iteration_with_moments_closed_forms_and_oracle(oracle):
    """lya_root_update_moments (quartic cumulant model of ln f): exact in two passes for constant tau (ln f is
    linear), and the oracle's A on a heavy-tailed sample in at most 6 passes."""
    import ctypes as C
    L = lya.lib()

    def solve(tau, f_target, tol=1e-12):
        st = lya.CRootState()
        assert L.lya_root_init(C.byref(st), f_target, tol, float(tau.size)) == lya.OK
        while not st.done:
            e = np.exp(-st.a * tau)
            s5 = (C.c_double * 5)(*[float((tau ** k * e).sum()) for k in range(5)])
            assert L.lya_root_update_moments(C.byref(st), s5) == lya.OK
            assert st.iters < 30
        return st.a, st.f_at_a, st.iters

    A, f, it = solve(np.full(1000, 0.7), 0.8)
    assert A == pytest.approx(-np.log(0.8) / 0.7, rel=1e-13) and f == pytest.approx(0.8, rel=1e-13) and it <= 2
    tau1 = 0.4
    tau = np.concatenate([np.full(500, tau1), np.full(500, 2 * tau1)])          # x^2 + x = 2 F, x = exp(-A tau1)
    A, f, it = solve(tau, 0.6)
    x = (-1 + np.sqrt(1 + 8 * 0.6)) / 2
    assert A == pytest.approx(-np.log(x) / tau1, rel=1e-11) and it <= 6
    rng = np.random.default_rng(3)
    tau = rng.lognormal(-1.0, 1.5, 300_000)
    for ft in (0.9, 0.78, 0.3):
        A, f, it = solve(tau, ft, tol=1e-10)
        A_ref, _, _ = oracle.normalize_mean_flux(tau, ft)
        assert A == pytest.approx(A_ref, rel=1e-9) and abs(f - ft) < 1e-9 and it <= 6
    st = lya.CRootState()                                                           # all tau == 0: no root
    L.lya_root_init(C.byref(st), 0.8, 1e-9, 10.0)
    assert L.lya_root_update_moments(C.byref(st), (C.c_double * 5)(10.0, 0.0, 0.0, 0.0, 0.0)) == lya.ENOROOT
