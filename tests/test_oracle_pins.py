"""Pins P1-P11 of SURVEY.md section 8(c): the oracle checked against what the paper and the
mathematics fix -- closed forms, exact identities, invariants, brute force -- never
against itself or against the CUDA path.  CPU only (-m "not gpu").

Every expected value here is derived in the test from CODATA constants / textbook
formulas typed in independently of oracle/lya_oracle.c, or read from
tests/golden/paper_values.txt (values the paper prints, with citations).
"""
import math
import os

import numpy as np
import pytest

from paper_1105_4747_b200.workloads import WORKLOADS

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                out[k] = float(v)
    return out


# independent retyping of the physical constants (cgs, CODATA 2018)
KB, MP, MH = 1.380649e-16, 1.67262192369e-24, 1.6735575e-24
MPC, CLIGHT, RHOC100 = 3.0856775814913673e24, 2.99792458e10, 1.87834e-29


def P(oracle, cfg=1, n=None, **kw):
    w = WORKLOADS[cfg]
    p = oracle.Params.from_workload(w)
    if n is not None:                      # same physical cell size on a shorter sightline
        p.box_mpch = w.box_mpch * n / w.n
        p.n_pix = n
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def theta(r, phase=0.0):
    """Poisson-summation aliasing factor 1 + 2 sum_m exp(-(pi m r)^2) cos(2 pi m phase)."""
    s, m = 1.0, 1
    while True:
        t = 2.0 * math.exp(-(math.pi * m * r) ** 2)
        if t < 1e-19:
            return s
        s += t * math.cos(2.0 * math.pi * m * phase)
        m += 1


# ---------------------------------------------------------------- P10 / unit chain
def test_p10_tau_eff_convention():
    g = golden()
    assert abs(-math.log(g["mean_flux_z3"]) - g["tau_eff_z3"]) < 5e-4


def test_sigma_alpha_is_the_textbook_cross_section():
    # sigma = pi e^2 f lambda / (m_e c^2): fixes Eq.6's prefactor convention
    e, me, f, lam = 4.80320471e-10, 9.1093837015e-28, 0.4164, 1215.67e-8
    sig = math.pi * e * e * f * lam / (me * CLIGHT ** 2)
    assert abs(sig / golden()["sigma_alpha_cm2"] - 1.0) < 1e-3


def test_scalars_unit_chain(oracle):
    g = golden()
    for cfg, w in WORKLOADS.items():
        p = P(oracle, cfg)
        s = oracle.scalars(p)
        Ez = math.sqrt(w.omega_m * (1 + w.z) ** 3 + 1 - w.omega_m)
        dv = 100.0 * Ez * w.box_mpch / (w.n * (1 + w.z))                    # km/s, h cancels
        assert abs(s["dv_kms"] / dv - 1) < 1e-14
        assert abs(s["b0_kms"] / (math.sqrt(2 * KB * w.T0 / MP) / 1e5) - 1) < 1e-14
        nH = (1 - w.y_he) * w.omega_b_h2 * RHOC100 * (1 + w.z) ** 3 / MH
        nHI = g["nhi_coefficient"] * nH * (w.T0 / 1e4) ** g["alpha_A_slope"] * ((1 + w.z) / 4) ** 3
        assert abs(s["nbarHI"] / nHI - 1) < 1e-13
        K = CLIGHT * g["sigma_alpha_cm2"] * (w.box_mpch / (w.n * w.h * (1 + w.z)) * MPC) / math.sqrt(math.pi)
        assert abs(s["K"] / K - 1) < 1e-14
        # textbook Gunn-Peterson optical depth c sigma n_HI / H(z), H in s^-1
        Hs = 100.0 * w.h * Ez * 1e5 / MPC
        assert abs(s["tauGP"] / (CLIGHT * g["sigma_alpha_cm2"] * nHI / Hs) - 1) < 1e-13
        assert abs(s["tau0"] * math.sqrt(math.pi) * s["b0_kms"] / s["dv_kms"] / s["tauGP"] - 1) < 1e-13
    # b(1e4 K) with m_p (reading C6); SURVEY 8.0 table values for cfg 1
    s1 = oracle.scalars(P(oracle, 1))
    assert abs(s1["b0_kms"] - 12.848657) < 2e-6
    assert abs(s1["dv_kms"] - 32.8815) < 1e-4 and abs(s1["tauGP"] - 0.68440) < 1e-5
    # PAPER.md:128 1 Gpc / 4096 = 244 kpc
    assert abs(1e6 / 4096 - g["box_1gpc_cell_kpc"]) < 0.5


# ---------------------------------------------------------------- P1 gas
def test_p1_gas_closed_values(oracle):
    g = golden()
    for cfg in (1, 2, 3):
        p = P(oracle, cfg)
        s = oracle.scalars(p)
        gm1 = p.gamma - 1.0
        d = np.array([0.0, 9.0, 99.0, -0.5, 9.0000001, 3.0], np.float32)
        T, n, b = oracle.gas_from_density(p, d)
        assert abs(T[0] / p.T0 - 1) < 1e-14 and abs(n[0] / s["nbarHI"] - 1) < 1e-13
        assert abs(b[0] / s["b0_kms"] - 1) < 1e-14
        piv = g["pivot_1_plus_delta"]
        # at the pivot and above it: T frozen at T0 * 10^(gamma-1)
        for k in (1, 2):
            assert abs(T[k] / (p.T0 * piv ** gm1) - 1) < 1e-13
            assert abs(b[k] / (s["b0_kms"] * piv ** (0.5 * gm1)) - 1) < 1e-13
        assert abs(n[2] / (s["nbarHI"] * piv ** (-0.7 * gm1) * 1e4) - 1) < 1e-12
        assert abs(n[1] / (s["nbarHI"] * piv ** (2 - 0.7 * gm1)) - 1) < 1e-12
        # below the pivot: n_HI ~ Delta^(2 - 0.7(gamma-1))   (Eq.4 with Eq.5, north_star)
        for k, D in ((3, 0.5), (5, 4.0)):
            assert abs(n[k] / (s["nbarHI"] * D ** (2 - 0.7 * gm1)) - 1) < 1e-12
            assert abs(b[k] / (s["b0_kms"] * D ** (0.5 * gm1)) - 1) < 1e-13
        # continuity across the pivot (float32(9.0000001) rounds to 9.0 or just above)
        assert abs(T[4] / T[1] - 1) < 1e-6
    # pivot disabled: pure power law
    p = P(oracle, 1, delta_pivot=0.0)
    T, n, b = oracle.gas_from_density(p, np.array([99.0], np.float32))
    assert abs(T[0] / (p.T0 * 100 ** 0.5) - 1) < 1e-13


# ---------------------------------------------------------------- P2 uniform field
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_p2_uniform_field_is_gunn_peterson_times_theta(oracle, cfg):
    p = P(oracle, cfg, n=64)
    s = oracle.scalars(p)
    z = np.zeros((3, 64), np.float32)
    _, n, b = oracle.gas_from_density(p, z)
    tau = oracle.tau_rows(p, n, b, z)
    expect = s["tauGP"] * theta(s["b0_kms"] / s["dv_kms"])
    assert np.max(np.abs(tau / expect - 1)) < 1e-13
    # SURVEY 8.0 table column "tau_uniform(discrete)"
    table = {1: 0.99099, 2: 0.76098, 3: 0.68562, 4: 1.23529, 5: 1.54400}
    assert abs(expect - table[cfg]) < 1e-5


def test_p2_resolved_grid_gives_textbook_gunn_peterson(oracle):
    # the paper's own 512^3 / 40 Mpc/h grid at T0 = 1.7e4 K resolves b
    p = oracle.Params(n_pix=512, box_mpch=40.0, z=3.0, T0=1.7e4, gamma=1.3, omega_m=0.26, h=0.72)
    s = oracle.scalars(p)
    assert s["b0_kms"] / s["dv_kms"] > 2.0
    z = np.zeros((1, 512), np.float32)
    _, n, b = oracle.gas_from_density(p, z)
    tau = oracle.tau_rows(p, n, b, z)
    assert np.max(np.abs(tau / s["tauGP"] - 1)) < 1e-13


# ---------------------------------------------------------------- P3 column identity
@pytest.mark.parametrize("n", [8, 64, 100])
def test_p3_column_identity(oracle, n):
    rng = np.random.default_rng(3 + n)
    p = P(oracle, 1, n=n)
    s = oracle.scalars(p)
    delta = np.expm1(rng.normal(0, 1.0, (5, n)) - 0.5).astype(np.float32)
    delta[0, 1] = 40.0                                                     # above the pivot
    v = (rng.normal(0, 60.0, (5, n))).astype(np.float32)
    _, nh, b = oracle.gas_from_density(p, delta)
    tau = oracle.tau_rows(p, nh, b, v)
    dv = s["dv_kms"]
    for r in range(5):
        rhs = 0.0
        for j in range(n):
            rhs += nh[r, j] * theta(b[r, j] / dv, float(v[r, j]) / dv)
        rhs *= 1e-5 * s["K"] * math.sqrt(math.pi)
        lhs = float(np.sum(tau[r])) * dv
        assert abs(lhs / rhs - 1) < 2e-13


# ---------------------------------------------------------------- P4 / P5 equivariance
def _random_rows(oracle, p, rows, seed, sigma_v=60.0):
    rng = np.random.default_rng(seed)
    delta = np.expm1(rng.normal(0, 1.0, (rows, p.n_pix)) - 0.5).astype(np.float32)
    v = rng.normal(0, sigma_v, (rows, p.n_pix)).astype(np.float32)
    _, nh, b = oracle.gas_from_density(p, delta)
    return delta, v, nh, b


def test_p4_cyclic_shift(oracle):
    p = P(oracle, 2, n=96)
    _, v, nh, b = _random_rows(oracle, p, 4, 44)
    tau = oracle.tau_rows(p, nh, b, v)
    for s_ in (1, 17, 95):
        t2 = oracle.tau_rows(p, np.roll(nh, s_, 1), np.roll(b, s_, 1), np.roll(v, s_, 1))
        assert np.max(np.abs(t2 / np.roll(tau, s_, 1) - 1)) < 1e-13


def test_p5_velocity_offset_sign_and_period(oracle):
    p = P(oracle, 1, n=64)
    s = oracle.scalars(p)
    _, v, nh, b = _random_rows(oracle, p, 3, 55)
    v64 = v.astype(np.float64)
    tau = oracle.tau_rows(p, nh, b, v)
    # +k pixels of peculiar velocity moves the absorption to HIGHER pixel index (reading C11).
    # fp32 storage of v + k dv rounds; compare against the oracle fed the SAME rounded values.
    k = 3
    vk = (v64 + k * s["dv_kms"]).astype(np.float32)
    resid = vk.astype(np.float64) - k * s["dv_kms"]                        # what the shift really was
    t_shift = oracle.tau_rows(p, nh, b, vk)
    t_ref = np.roll(oracle.tau_rows(p, nh, b, resid.astype(np.float32)), k, 1)
    # resid is not exactly fp32-representable: allow its rounding (1e-7 rel of ~50 km/s over b ~ 13)
    assert np.max(np.abs(t_shift - t_ref)) < 2e-6 * np.max(tau)
    assert np.max(np.abs(t_shift - np.roll(tau, k, 1))) < 2e-5 * np.max(tau)
    # a shift the wrong way must NOT match
    assert np.max(np.abs(t_shift - np.roll(tau, -k, 1))) > 1e-2 * np.max(tau)
    # v -> v + V leaves tau unchanged (period V); exact test with a power-of-two period
    p2 = P(oracle, 1, n=64)
    V = s["V_kms"]
    vV = (v64 + V).astype(np.float32)
    t_per = oracle.tau_rows(p2, nh, b, vV)
    t_eq = oracle.tau_rows(p2, nh, b, (vV.astype(np.float64) - V).astype(np.float32))
    assert np.max(np.abs(t_per - t_eq)) < 1e-5 * np.max(tau)


# ---------------------------------------------------------------- P6 single source
def test_p6_single_source_profile(oracle):
    p = P(oracle, 1, n=64)
    s = oracle.scalars(p)
    delta = np.full((1, 64), 2.0 ** -20 - 1.0, np.float32)       # background 1+delta = 2^-20
    j0, vj = 20, 41.5
    delta[0, j0] = 0.0
    v = np.zeros((1, 64), np.float32)
    v[0, j0] = vj
    _, nh, b = oracle.gas_from_density(p, delta)
    tau = oracle.tau_rows(p, nh, b, v)[0]
    i = np.arange(64)
    d = (i - j0) * s["dv_kms"] - float(np.float32(vj))
    d -= s["V_kms"] * np.round(d / s["V_kms"])
    expect = s["tau0"] * np.exp(-(d / s["b0_kms"]) ** 2)
    assert np.max(np.abs(tau - expect)) < 2e-8                            # background ~ 4e-9 tau0
    assert np.argmax(tau) == j0 + 1                                       # 41.5 km/s = +1.26 px


# ---------------------------------------------------------------- P7 brute force, 8 cells
def test_p7_brute_force_image_sum_8_cells(oracle):
    rng = np.random.default_rng(7)
    # 8 cells of 160 km/s: V/2 = 640 km/s >= 6 b_max so images beyond +-3 are < 1e-300
    p = oracle.Params(n_pix=8, box_mpch=8 * 160.0 / (100.0 * math.sqrt(0.3 * 3.5 ** 3 + 0.7)) * 3.5,
                      z=2.5, T0=1.0e4, gamma=1.5)
    s = oracle.scalars(p)
    assert abs(s["dv_kms"] - 160.0) < 1e-9
    for trial in range(20):
        delta = np.expm1(rng.normal(0, 1.0, (1, 8))).astype(np.float32)
        v = rng.uniform(-2 * s["V_kms"], 2 * s["V_kms"], (1, 8)).astype(np.float32)
        _, nh, b = oracle.gas_from_density(p, delta)
        tau = oracle.tau_rows(p, nh, b, v)[0]
        brute = np.zeros(8)
        for i in range(8):
            for j in range(8):
                for m in range(-4, 5):
                    d = (i - j) * s["dv_kms"] - float(v[0, j]) + m * s["V_kms"]
                    brute[i] += s["K"] * nh[0, j] / (b[0, j] * 1e5) * math.exp(-(d / b[0, j]) ** 2)
        assert np.max(np.abs(tau - brute)) < 1e-13 * np.max(brute)


# ---------------------------------------------------------------- P8 Gamma scaling
def test_p8_gamma_scaling(oracle):
    w = WORKLOADS[1]
    rng = np.random.default_rng(8)
    delta = np.expm1(rng.normal(0, 1, (8, 8, 64)) - 0.5).astype(np.float32)
    v = rng.normal(0, 50, (8, 8, 64)).astype(np.float32)
    r1 = oracle.run_path(P(oracle, 1), 0, delta, v, w.f_target)
    r2 = oracle.run_path(P(oracle, 1, gamma_m12=2.0), 0, delta, v, w.f_target)
    assert np.max(np.abs(r2["tau"] * 2 / r1["tau"] - 1)) < 1e-13
    assert abs(r2["A"] / (2 * r1["A"]) - 1) < 1e-11
    assert np.max(np.abs(r2["flux"] - r1["flux"])) < 1e-11


# ---------------------------------------------------------------- P9 closed forms for A
def test_p9_normalisation_closed_forms(oracle):
    A, f, _ = oracle.normalize_mean_flux(np.full(1000, 0.37), 0.72)
    assert abs(A / (-math.log(0.72) / 0.37) - 1) < 1e-12 and abs(f - 0.72) < 1e-12
    t1, Ft = 0.8, 0.6
    tau = np.concatenate([np.full(500, t1), np.full(500, 2 * t1)])
    x = (-1 + math.sqrt(1 + 8 * Ft)) / 2
    A, f, _ = oracle.normalize_mean_flux(tau, Ft)
    assert abs(A / (-math.log(x) / t1) - 1) < 1e-12
    # A > 1 branch (bracket doubling) and strict monotonicity of f(A)
    A, _, _ = oracle.normalize_mean_flux(np.full(10, 0.01), 0.5)
    assert abs(A / (math.log(2) / 0.01) - 1) < 1e-12
    rng = np.random.default_rng(9)
    t = rng.lognormal(0, 1, 5000)
    fs = [oracle.mean_flux(t, a) for a in (0.0, 0.1, 0.5, 1.0, 3.0)]
    assert fs[0] == 1.0 and all(a > b_ for a, b_ in zip(fs, fs[1:]))
    assert abs(oracle.mean_flux(t, 0.7) - float(np.mean(np.exp(-0.7 * t)))) < 1e-14
    with pytest.raises(ArithmeticError):
        oracle.normalize_mean_flux(np.array([0.0, 0.0, 1.0]), 0.5)         # f >= 2/3 always
    with pytest.raises(ValueError):
        oracle.normalize_mean_flux(np.ones(4), 1.0)
    F = oracle.flux(np.array([0.0, 1.0, 2.0]), 0.5)
    assert np.allclose(F, [1.0, math.exp(-0.5), math.exp(-1.0)], rtol=1e-15)


# ---------------------------------------------------------------- P11 skip-zero == plain
def test_p11_skip_zero_is_bit_identical(oracle):
    for cfg, n in ((1, 64), (2, 256), (5, 128)):
        p = P(oracle, cfg, n=n)
        _, v, nh, b = _random_rows(oracle, p, 6, 110 + cfg, sigma_v=WORKLOADS[cfg].sigma_v)
        a = oracle.tau_rows(p, nh, b, v, mode=0)
        c = oracle.tau_rows(p, nh, b, v, mode=1)
        assert np.array_equal(a, c)


# ---------------------------------------------------------------- axis handling (pure indexing)
def test_axis_views_match_explicit_rows(oracle):
    rng = np.random.default_rng(12)
    n = 16
    p = P(oracle, 3, n=n)
    delta = np.expm1(rng.normal(0, 1, (n, n, n)) - 0.5).astype(np.float32)
    v = rng.normal(0, 100, (n, n, n)).astype(np.float32)
    _, nh, b = oracle.gas_from_density(p, delta)
    ty = oracle.tau_grid(p, 1, nh, b, v)
    tz = oracle.tau_grid(p, 2, nh, b, v)
    iz, ix, iy = 3, 5, 7
    row = oracle.tau_rows(p, nh[iz, :, ix][None], b[iz, :, ix][None], v[iz, :, ix][None])[0]
    assert np.array_equal(ty[iz, :, ix], row)
    row = oracle.tau_rows(p, nh[:, iy, ix][None], b[:, iy, ix][None], v[:, iy, ix][None])[0]
    assert np.array_equal(tz[:, iy, ix], row)
