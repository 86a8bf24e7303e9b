"""GPU parity at BASELINE.json's full sizes (configs 3, 4, 5), in the launch configuration bench.py times.

What the oracle covers at each size (BASELINE.md section 4 has the same table):
  cfg 3 (512^3, three axes)  EVERY sightline of every axis pass (skip-zero mode, bit-identical to plain mode by pin
                             P11): tau, F, signed mean tau error, and A against the oracle's own A.
  cfg 4 (1024^3)             every sightline of a 64-plane z-slab (65,536 rows = 6.9e10 pairs): tau, F, bias, and the
                             A of THAT slab against the oracle's own; plus 2048 seeded rows from the whole grid.  The A
                             of the whole grid is a REDUCTION CHECK ONLY (the oracle's bisection over the GPU's tau):
                             1.1e12 pairs take the oracle ~5 min on 16 cores, so the whole-grid oracle A runs only with
                             LYA_FULL_ORACLE=1 (measured once: profiles/r2_full_oracle_cfg4.md).
  cfg 5 (2048^3, slabs)      every sightline of an 8-plane slab (16,384 rows = 6.9e10 pairs) incl. that slab's A; 2048
                             seeded rows of other slabs.  The whole grid's A needs 1.8e13 oracle pairs: not run.
Tolerances: BASELINE.json north_star; the signed mean relative tau error is held to 1e-6.
"""
import os

import numpy as np
import pytest
import torch

from paper_1105_4747_b200 import inputs, lya
from paper_1105_4747_b200.workloads import WORKLOADS

pytestmark = pytest.mark.gpu

TAU_REL, TAU_ABS, F_ABS, A_REL, TAU_BIAS = 2e-4, 1e-7, 1e-5, 1e-5, 1e-6


@pytest.fixture(scope="module")
def ctx():
    c = lya.Context(0)
    yield c
    c.close()
    torch.cuda.empty_cache()


def check_rows(oracle, w, d_rows, v_rows, tau_rows, F_rows, A, what):
    """tau and F of some sightlines (rows) against the oracle; returns the oracle's tau."""
    po = oracle.Params.from_workload(w)
    _, n_ref, b_ref = oracle.gas_from_density(po, d_rows)
    ref = oracle.tau_rows(po, n_ref, b_ref, v_rows, mode=1)
    g = tau_rows.astype(np.float64)
    big = ref > 1e-3
    err = g[big] / ref[big] - 1.0
    rel = np.abs(err).max()
    ab = np.abs(g[~big] - ref[~big]).max() if (~big).any() else 0.0
    assert rel <= TAU_REL and ab <= TAU_ABS, f"{what}: tau rel {rel:.2e} abs {ab:.2e}"
    assert abs(err.mean()) <= TAU_BIAS, f"{what}: signed mean relative tau error {err.mean():.2e}"
    dF = np.abs(F_rows - oracle.flux(ref, A)).max()
    assert dF <= F_ABS, f"{what}: F abs {dF:.2e}"
    return ref


def sightline_rows(t, axis, idx_a, idx_b):
    """Rows of a [nz][ny][nx] device tensor along `axis` at the index pairs of the two other axes."""
    if axis == 0:
        return t[idx_a, idx_b, :].cpu().numpy()                 # (iz, iy)
    if axis == 1:
        return t[idx_a, :, idx_b].cpu().numpy()                 # (iz, ix)
    return t[:, idx_a, idx_b].T.contiguous().cpu().numpy()      # (iy, ix)


def test_cfg3_three_axes_every_sightline(ctx, oracle):
    w = WORKLOADS[3]
    f = inputs.make_fields(w, device="cuda")
    delta = f["delta"]
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, delta)
    d_np = delta.cpu().numpy()
    for ax in w.axes:
        v = f["v_pec"][ax]
        tau = ctx.tau_sightlines(p, ax, n_hi, b, v)
        A, fa, it, _ = ctx.normalize_mean_flux(tau, w.f_target)
        F = ctx.flux(tau, A)
        v_np = v.cpu().numpy()
        ref = check_rows(oracle, w, oracle.to_rows(d_np, ax), oracle.to_rows(v_np, ax),
                         oracle.to_rows(tau.cpu().numpy(), ax), oracle.to_rows(F.cpu().numpy(), ax), A, f"cfg3 axis {ax}")
        A_ref, _, _ = oracle.normalize_mean_flux(ref, w.f_target)          # the oracle's A over the oracle's tau
        assert abs(A / A_ref - 1.0) < A_REL, (ax, A, A_ref)
        s, _ = ctx.flux_partial_sums(tau, [A])
        assert abs(s[0] / tau.numel() - w.f_target) < 1e-6 and it <= 12
        del tau, F, ref


def test_cfg4_full_size(ctx, oracle):
    w = WORKLOADS[4]
    n = w.n
    f = inputs.make_fields(w, device="cuda")
    delta, v = f["delta"], f["v_pec"][0]
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, 0, n_hi, b, v)
    del n_hi, b
    A, fa, it, _ = ctx.normalize_mean_flux(tau, w.f_target)
    F = ctx.flux(tau, A)
    # (i) 2048 seeded rows of the whole grid
    rng = np.random.default_rng(w.seed)
    ia = torch.from_numpy(rng.integers(0, n, 2048)).cuda()
    ib = torch.from_numpy(rng.integers(0, n, 2048)).cuda()
    check_rows(oracle, w, sightline_rows(delta, 0, ia, ib), sightline_rows(v, 0, ia, ib),
               sightline_rows(tau, 0, ia, ib), sightline_rows(F, 0, ia, ib), A, "cfg4 rows")
    # (ii) every sightline of planes 480..543: tau, F, bias, and that slab's A against the oracle's own
    z0, z1 = 480, 544
    A_s, _, it_s, _ = ctx.normalize_mean_flux(tau[z0:z1], w.f_target)
    F_s = ctx.flux(tau[z0:z1], A_s)
    ref = check_rows(oracle, w, delta[z0:z1].cpu().numpy(), v[z0:z1].cpu().numpy(), tau[z0:z1].cpu().numpy(),
                     F_s.cpu().numpy(), A_s, "cfg4 slab")
    A_ref, _, _ = oracle.normalize_mean_flux(ref, w.f_target)
    assert abs(A_s / A_ref - 1.0) < A_REL, (A_s, A_ref)
    del ref, F_s
    # (iii) the whole grid's A: reduction check only (oracle bisection in double over the GPU's tau) ...
    A_red, _, _ = oracle.normalize_mean_flux(tau.cpu().numpy().astype(np.float64).ravel(), w.f_target)
    assert abs(A / A_red - 1.0) < A_REL and it <= 12
    s, _ = ctx.flux_partial_sums(tau, [A])
    assert abs(s[0] / tau.numel() - w.f_target) < 1e-6
    # ... unless asked for the real thing: the oracle's tau on all 1,048,576 sightlines, 64 planes at a time
    if os.environ.get("LYA_FULL_ORACLE") == "1":
        tau_ref = np.empty((n, n, n), dtype=np.float64)
        po = oracle.Params.from_workload(w)
        worst, bias_sum, bias_n = 0.0, 0.0, 0
        for c0 in range(0, n, 64):
            _, n_ref, b_ref = oracle.gas_from_density(po, delta[c0:c0 + 64].cpu().numpy())
            tau_ref[c0:c0 + 64] = oracle.tau_rows(po, n_ref, b_ref, v[c0:c0 + 64].cpu().numpy(), mode=1)
            g, r = tau[c0:c0 + 64].cpu().numpy().astype(np.float64), tau_ref[c0:c0 + 64]
            big = r > 1e-3
            err = g[big] / r[big] - 1.0
            worst = max(worst, float(np.abs(err).max()))
            bias_sum, bias_n = bias_sum + float(err.sum()), bias_n + int(big.sum())
            assert np.abs(g[~big] - r[~big]).max() <= TAU_ABS
        A_full, _, _ = oracle.normalize_mean_flux(tau_ref.ravel(), w.f_target)
        print(f"cfg4 full oracle: tau max rel {worst:.3e} signed mean {bias_sum / bias_n:.3e} "
              f"A gpu {A:.12f} oracle {A_full:.12f} rel {A / A_full - 1:.3e}")
        assert worst <= TAU_REL and abs(bias_sum / bias_n) <= TAU_BIAS and abs(A / A_full - 1.0) < A_REL


def test_cfg5_slabs_of_complete_rows(ctx, oracle):
    """Config 5 is processed in z-slabs of complete x-rows (64 planes per launch in bench.py).  One seeded 64-plane
    slab from the middle of the 2048^3 grid on the GPU in that launch shape; the oracle covers every sightline of 8
    of its planes (incl. the A of those 8 planes) and 2048 seeded rows of the others."""
    w = WORKLOADS[5]
    n, z0, nzl = w.n, 992, 64
    f = inputs.make_fields(w, device="cuda", z0=z0, z1=z0 + nzl)
    delta, v = f["delta"], f["v_pec"][0]
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, 0, n_hi, b, v, nz_local=nzl)
    A, fa, it, _ = ctx.normalize_mean_flux(tau, w.f_target)      # this slab's own A (the grid's needs all slabs)
    F = ctx.flux(tau, A)
    rng = np.random.default_rng(w.seed)
    ia = torch.from_numpy(rng.integers(0, nzl, 2048)).cuda()
    ib = torch.from_numpy(rng.integers(0, n, 2048)).cuda()
    check_rows(oracle, w, sightline_rows(delta, 0, ia, ib), sightline_rows(v, 0, ia, ib),
               sightline_rows(tau, 0, ia, ib), sightline_rows(F, 0, ia, ib), A, "cfg5 rows")
    s0, s1 = 28, 36
    A_s, _, _, _ = ctx.normalize_mean_flux(tau[s0:s1], w.f_target)
    F_s = ctx.flux(tau[s0:s1], A_s)
    ref = check_rows(oracle, w, delta[s0:s1].cpu().numpy(), v[s0:s1].cpu().numpy(), tau[s0:s1].cpu().numpy(),
                     F_s.cpu().numpy(), A_s, "cfg5 planes")
    A_ref, _, _ = oracle.normalize_mean_flux(ref, w.f_target)
    assert abs(A_s / A_ref - 1.0) < A_REL, (A_s, A_ref)
    A_red, _, _ = oracle.normalize_mean_flux(tau.cpu().numpy().astype(np.float64).ravel(), w.f_target)
    assert abs(A / A_red - 1.0) < A_REL


@pytest.mark.parametrize("n,rows,windowed", [(4096, 96, False), (4096, 96, True), (8192, 24, False), (12000, 10, False)])
def test_long_sightlines(ctx, oracle, n, rows, windowed):
    """The paper's own sightline length (4096 pixels of ~244 kpc) and beyond: groups of 8-16 warps
    share a row whose staged cells fill most of an SM's shared memory."""
    w = WORKLOADS[5]
    rng = np.random.default_rng(n)
    delta = torch.from_numpy(np.expm1(rng.normal(0, 1.3, (1, rows, n)) - 0.845).astype(np.float32)).cuda()
    v = torch.from_numpy(rng.normal(0, 150.0, (1, rows, n)).astype(np.float32)).cuda()
    p = lya.Params(nx=n, ny=rows, nz=1, box_mpch=w.box_mpch * n / w.n, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    if windowed:
        tau = ctx.tau_sightlines_opt(p, 0, v, n_hi=n_hi, b_kms=b, windowed=True)
        assert torch.equal(tau, ctx.tau_sightlines(p, 0, n_hi, b, v))
    else:
        tau = ctx.tau_sightlines(p, 0, n_hi, b, v)
    torch.cuda.synchronize()
    po = oracle.Params(n_pix=n, box_mpch=p.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    sel = [0, rows // 2, rows - 1]
    _, n_ref, b_ref = oracle.gas_from_density(po, delta[0, sel].cpu().numpy())
    ref = oracle.tau_rows(po, n_ref, b_ref, v[0, sel].cpu().numpy(), mode=1)
    g = tau[0, sel].cpu().numpy().astype(np.float64)
    big = ref > 1e-3
    assert np.abs(g[big] / ref[big] - 1).max() <= TAU_REL and np.abs(g[~big] - ref[~big]).max() <= TAU_ABS
