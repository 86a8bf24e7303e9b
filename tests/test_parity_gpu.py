"""GPU parity: the CUDA path (through the C ABI, paper_1105_4747_b200.lya) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
tau: relative 2e-4 where tau > 1e-3, absolute 1e-7 otherwise; F: absolute 1e-5; A: relative 1e-5.
"""
import numpy as np
import pytest
import torch

from paper_1105_4747_b200 import inputs, lya
from paper_1105_4747_b200.workloads import WORKLOADS, scaled

pytestmark = pytest.mark.gpu

TAU_REL, TAU_ABS, F_ABS, A_REL = 2e-4, 1e-7, 1e-5, 1e-5
TAU_BIAS = 1e-6        # |signed mean relative tau error|: A moves one for one with a BIAS in tau, so the
                       # mean error is held 200 x tighter than the per-pixel bar


@pytest.fixture(scope="module")
def ctx():
    c = lya.Context(0)
    yield c
    c.close()


def assert_tau_close(tau_gpu, tau_ref, what=""):
    g = np.asarray(tau_gpu, dtype=np.float64)
    r = np.asarray(tau_ref, dtype=np.float64)
    assert g.shape == r.shape
    big = r > 1e-3
    rel = np.abs(g[big] / r[big] - 1.0).max() if big.any() else 0.0
    ab = np.abs(g[~big] - r[~big]).max() if (~big).any() else 0.0
    assert np.isfinite(g).all(), what
    assert rel <= TAU_REL, f"{what}: tau max rel err {rel:.3e}"
    assert ab <= TAU_ABS, f"{what}: tau max abs err (tau<=1e-3) {ab:.3e}"
    if big.sum() >= 4096:                                 # enough pixels for the mean to be a statement about bias
        bias = float((g[big] / r[big] - 1.0).mean())
        assert abs(bias) <= TAU_BIAS, f"{what}: signed mean relative tau error {bias:.3e}"
    return rel, ab


def gpu_fields(w, device="cuda", **kw):
    f = inputs.make_fields(w, device=device, **kw)
    return f["delta"], f["v_pec"]


def run_gpu(ctx, w, delta, v, axis=0):
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, axis, n_hi, b, v)
    A, f, it, _ = ctx.normalize_mean_flux(tau, w.f_target)
    F = ctx.flux(tau, A)
    torch.cuda.synchronize()
    return n_hi, b, tau, A, f, it, F


# ------------------------------------------------------------------ S1
def test_gas_parity_and_pivot_edges(ctx, oracle):
    w = WORKLOADS[1]
    delta, _ = gpu_fields(w)
    edge = torch.tensor([-0.999, -0.5, 0.0, 1.0, 8.9999, 9.0, 9.0001, 99.0, 999.0, 1e-8 - 1.0 + 1.0],
                        dtype=torch.float32, device="cuda")
    d = torch.cat([delta.reshape(-1), edge])            # also makes the length ragged (not % 4)
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, d)
    _, n_ref, b_ref = oracle.gas_from_density(oracle.Params.from_workload(w), d.cpu().numpy())
    assert np.abs(n_hi.cpu().numpy() / n_ref - 1).max() < 2e-6
    assert np.abs(b.cpu().numpy() / b_ref - 1).max() < 1e-6
    # pivot off
    w2 = scaled(w, 64)
    p.delta_pivot = 0.0
    po = oracle.Params.from_workload(w2)
    po.delta_pivot = 0.0
    n_hi, b = ctx.gas_from_density(p, d)
    _, n_ref, b_ref = oracle.gas_from_density(po, d.cpu().numpy())
    assert np.abs(n_hi.cpu().numpy() / n_ref - 1).max() < 2e-6
    assert np.abs(b.cpu().numpy() / b_ref - 1).max() < 1e-6
    # unaligned views take the scalar path
    n2, b2 = torch.empty(d.numel() + 1, device="cuda"), torch.empty(d.numel() + 1, device="cuda")
    ctx.gas_from_density(p, d[1:], n2[2:], b2[2:])
    assert torch.equal(n2[2:], n_hi[1:]) and torch.equal(b2[2:], b[1:])


# ------------------------------------------------------------------ whole path, configs 1 and 2
def test_full_path_cfg1_every_pixel(ctx, oracle):
    w = WORKLOADS[1]
    delta, v = gpu_fields(w)
    n_hi, b, tau, A, f, it, F = run_gpu(ctx, w, delta, v[0])
    ref = oracle.run_path(oracle.Params.from_workload(w), 0, delta.cpu().numpy(), v[0].cpu().numpy(), w.f_target)
    assert_tau_close(tau.cpu().numpy(), ref["tau"], "cfg1")
    assert abs(A / ref["A"] - 1) < A_REL
    assert it <= 15
    assert abs(oracle.mean_flux(ref["tau"], A) - w.f_target) < 2e-6      # the oracle's mean flux at the GPU's A
    assert np.abs(F.cpu().numpy() - ref["flux"]).max() < F_ABS


def test_full_path_cfg2_every_pixel(ctx, oracle):
    """256^3 in bench.py's launch configuration against the oracle on EVERY sightline (4.3e9 pairs, skip-zero mode,
    bit-identical to plain mode by pin P11): tau and F on every pixel, the signed mean tau error, and A against the
    oracle's own A over the oracle's own tau -- not a bisection over the GPU's tau."""
    w = WORKLOADS[2]
    delta, v = gpu_fields(w)
    n_hi, b, tau, A, f, it, F = run_gpu(ctx, w, delta, v[0])
    ref = oracle.run_path(oracle.Params.from_workload(w), 0, delta.cpu().numpy(), v[0].cpu().numpy(), w.f_target, mode=1)
    assert_tau_close(tau.cpu().numpy(), ref["tau"], "cfg2")
    assert abs(A / ref["A"] - 1) < A_REL, (A, ref["A"])
    assert np.abs(F.cpu().numpy() - ref["flux"]).max() < F_ABS
    # f_achieved is the cumulant model's value at A (lya.h); the MEASURED mean flux at the returned A, through the
    # library's own reduction and through the oracle's, must hit the target
    s, _ = ctx.flux_partial_sums(tau, [A])
    assert abs(s[0] / tau.numel() - w.f_target) < 1e-6 and abs(f - s[0] / tau.numel()) < 1e-7
    assert abs(oracle.mean_flux(ref["tau"], A) - w.f_target) < 2e-6


def test_forest_host_cfg2_against_the_oracle(ctx, oracle):
    """lya_forest_host (S1 fused into S3, z-slab streaming from pinned host memory) on the whole of config 2 against
    the ORACLE: tau_h, flux_h and A, not against the stepwise GPU path."""
    w = WORKLOADS[2]
    f = inputs.make_fields(w, device="cuda")
    dh, vh = f["delta"].cpu().pin_memory(), f["v_pec"][0].cpu().pin_memory()
    del f
    tau_h, flux_h = torch.empty_like(dh).pin_memory(), torch.empty_like(dh).pin_memory()
    A, fa, it = ctx.forest_host(lya.Params.from_workload(w), 0, dh, vh, w.f_target, tau_h=tau_h, flux_h=flux_h)
    ref = oracle.run_path(oracle.Params.from_workload(w), 0, dh.numpy(), vh.numpy(), w.f_target, mode=1)
    assert_tau_close(tau_h.numpy(), ref["tau"], "forest_host cfg2")
    assert abs(A / ref["A"] - 1) < A_REL
    assert np.abs(flux_h.numpy() - ref["flux"]).max() < F_ABS


@pytest.mark.parametrize("sigma_g,f_target", [(2.0, 0.5), (2.5, 0.9)])
def test_normalisation_on_heavy_tailed_tau_against_the_full_oracle(ctx, oracle, sigma_g, f_target):
    """A on a 128^3 grid whose tau distribution is far heavier-tailed than the configs' (sigma_g 2-2.5: the
    cumulant model of root_iter.h is least accurate there), against the oracle's A over the oracle's own tau."""
    import dataclasses
    w = dataclasses.replace(scaled(WORKLOADS[4], 128), sigma_g=sigma_g, f_target=f_target)
    delta, v = gpu_fields(w)
    _, _, tau, A, f, it, F = run_gpu(ctx, w, delta, v[0])
    ref = oracle.run_path(oracle.Params.from_workload(w), 0, delta.cpu().numpy(), v[0].cpu().numpy(), f_target, mode=1)
    assert_tau_close(tau.cpu().numpy(), ref["tau"], "heavy tail")
    assert abs(A / ref["A"] - 1) < A_REL, (A, ref["A"], it)
    s, _ = ctx.flux_partial_sums(tau, [A])
    assert abs(s[0] / tau.numel() - f_target) < 1e-6
    assert np.abs(F.cpu().numpy() - ref["flux"]).max() < F_ABS


# ------------------------------------------------------------------ S3 shapes: ragged, tiny, strided, slabs
@pytest.mark.parametrize("n", [1, 2, 8, 13, 31, 32, 33, 64, 100, 128, 200, 257, 258, 384, 1001, 1002])
def test_tau_ragged_lengths_x_axis(ctx, oracle, n):
    w = scaled(WORKLOADS[2], n)
    rng = np.random.default_rng(n)
    ny, nz = 5, 3
    delta = torch.from_numpy(np.expm1(rng.normal(0, 1.0, (nz, ny, n)) - 0.5).astype(np.float32)).cuda()
    v = torch.from_numpy(rng.normal(0, 80.0, (nz, ny, n)).astype(np.float32)).cuda()
    p = lya.Params(nx=n, ny=ny, nz=nz, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, 0, n_hi, b, v)
    po = oracle.Params.from_workload(w)
    _, n_ref, b_ref = oracle.gas_from_density(po, delta.cpu().numpy())
    ref = oracle.tau_rows(po, n_ref, b_ref, v.cpu().numpy())
    assert_tau_close(tau.cpu().numpy(), ref, f"n={n}")


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_tau_all_axes_noncubic(ctx, oracle, axis):
    nx, ny, nz = 44, 136, 72                               # ragged in x (not % 8), different per axis
    n = (nx, ny, nz)[axis]
    w = scaled(WORKLOADS[3], n)
    rng = np.random.default_rng(10 + axis)
    delta = torch.from_numpy(np.expm1(rng.normal(0, 1.2, (nz, ny, nx)) - 0.72).astype(np.float32)).cuda()
    v = torch.from_numpy(rng.normal(0, 100.0, (nz, ny, nx)).astype(np.float32)).cuda()
    p = lya.Params(nx=nx, ny=ny, nz=nz, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, axis, n_hi, b, v)
    po = oracle.Params.from_workload(w)
    _, n_ref, b_ref = oracle.gas_from_density(po, delta.cpu().numpy())
    ref = oracle.tau_grid(po, axis, n_ref, b_ref, v.cpu().numpy())
    assert_tau_close(tau.cpu().numpy(), ref, f"axis={axis}")


def test_tau_z_slabs_equal_whole_grid(ctx):
    w = scaled(WORKLOADS[2], 128)
    delta, v = gpu_fields(w)
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, delta)
    for axis in (0, 1):
        whole = ctx.tau_sightlines(p, axis, n_hi, b, v[0])
        parts = torch.empty_like(whole)
        for z0, z1 in ((0, 40), (40, 41), (41, 128)):
            ctx.tau_sightlines(p, axis, n_hi[z0:z1], b[z0:z1], v[0][z0:z1], tau=parts[z0:z1], nz_local=z1 - z0)
        assert torch.equal(whole, parts)
    with pytest.raises(lya.LyaError):
        ctx.tau_sightlines(p, 2, n_hi[:64], b[:64], v[0][:64], nz_local=64)


def test_tau_large_velocities_take_the_general_path(ctx, oracle):
    """|v_pec| up to 2 V (multi-wrap) and a sightline whose displacements break the fast-path condition."""
    n = 256
    w = scaled(WORKLOADS[2], n)
    po = oracle.Params.from_workload(w)
    V = oracle.scalars(po)["V_kms"]
    rng = np.random.default_rng(77)
    delta = torch.from_numpy(np.expm1(rng.normal(0, 1.0, (1, 16, n)) - 0.5).astype(np.float32)).cuda()
    v = torch.from_numpy(rng.uniform(-2 * V, 2 * V, (1, 16, n)).astype(np.float32)).cuda()
    p = lya.Params(nx=n, ny=16, nz=1, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, 0, n_hi, b, v)
    _, n_ref, b_ref = oracle.gas_from_density(po, delta.cpu().numpy())
    ref = oracle.tau_rows(po, n_ref, b_ref, v.cpu().numpy())
    # fp32 v_pec of order V carries ~V 6e-8 / dv pixels of input rounding, shared by both sides
    assert_tau_close(tau.cpu().numpy(), ref, "large v")


def test_tau_unaligned_rows_use_plain_loads(ctx):
    w = scaled(WORKLOADS[2], 128)
    delta, v = gpu_fields(w)
    p = lya.Params(nx=128, ny=128, nz=4, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta[:4].contiguous())
    vv = v[0][:4].contiguous()
    ref = ctx.tau_sightlines(p, 0, n_hi, b, vv)
    pad = lambda t: torch.cat([torch.zeros(1, device="cuda"), t.reshape(-1)])[1:].reshape(t.shape)
    got = ctx.tau_sightlines(p, 0, pad(n_hi), pad(b), pad(vv))
    assert torch.equal(ref, got)


# ------------------------------------------------------------------ invariants run on the GPU library (T2)
def test_gpu_invariants_shift_and_velocity_offset(ctx, oracle):
    w = scaled(WORKLOADS[2], 256)
    delta, v = gpu_fields(w)
    delta, vx = delta[:8].contiguous(), v[0][:8].contiguous()
    p = lya.Params(nx=256, ny=256, nz=8, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    dv = lya.scalars(p, 0)["dv_kms"]
    n_hi, b = ctx.gas_from_density(p, delta)
    tau = ctx.tau_sightlines(p, 0, n_hi, b, vx)
    s = 37                                                            # P4: cyclic shift
    tau_s = ctx.tau_sightlines(p, 0, n_hi.roll(s, 2).contiguous(), b.roll(s, 2).contiguous(),
                               vx.roll(s, 2).contiguous())
    # a pixel's rounding depends on where it sits in its lane's group of R pixels (x_ref is up to 2 cells away:
    # dx <= ulp(|x| + 2w)/2 ~ 2e-6, i.e. ~ln2 * 2 x dx <= 5e-6 relative per term), so two
    # evaluations of the same sum at shifted positions may differ by twice that
    assert torch.allclose(tau_s, tau.roll(s, 2), rtol=1e-5, atol=1e-9)
    k = 5                                                             # P5: +k dv moves tau by +k pixels
    tau_k = ctx.tau_sightlines(p, 0, n_hi, b, (vx.double() + k * dv).float())
    assert torch.allclose(tau_k, tau.roll(k, 2), rtol=3e-5, atol=1e-8)


# ------------------------------------------------------------------ S4 / S5
def test_normalize_closed_forms_and_errors(ctx):
    n = 1_000_003                                                     # ragged, > one grid-stride
    tau = torch.full((n,), 0.7, device="cuda")
    A, f, it, _ = ctx.normalize_mean_flux(tau, 0.8)
    assert abs(A / (-np.log(0.8) / 0.7) - 1) < 1e-6 and abs(f - 0.8) < 1e-6
    tau[: n // 2] = 0.35
    x = None
    # half tau1, half 2 tau1 (+1 odd pixel at 2 tau1): solve the exact mixture by bisection in numpy
    t = tau.double().cpu().numpy()
    lo, hi = 0.0, 10.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if np.exp(-mid * t).mean() > 0.72 else (lo, mid)
    A, f, it, _ = ctx.normalize_mean_flux(tau, 0.72)
    assert abs(A / lo - 1) < 1e-6 and it <= 12
    # unaligned view
    A2, _, _, _ = ctx.normalize_mean_flux(tau[1:], 0.72)
    assert abs(A2 / A - 1) < 1e-5
    with pytest.raises(lya.LyaError) as e:
        ctx.normalize_mean_flux(torch.zeros(4096, device="cuda"), 0.8)
    assert e.value.status == lya.ENOROOT
    with pytest.raises(lya.LyaError) as e:
        ctx.normalize_mean_flux(tau, 1.0)
    assert e.value.status == lya.EINVAL
    # partial sums (the slab / multi-GPU building block) against numpy
    s, d = ctx.flux_partial_sums(tau, [0.0, 0.5, 2.0])
    for a, si, di in zip([0.0, 0.5, 2.0], s, d):
        e_ = np.exp(-a * t)
        assert abs(si / e_.sum() - 1) < 1e-6 and abs(di / (t * e_).sum() - 1) < 1e-6


def test_nested_normalisation_subsample_then_full(ctx, oracle):
    """S4's nested iteration forced on a small, heavy-tailed, ragged tau: the subsample (every 4th 4 KiB chunk of the
    aligned body) only supplies the starting point, so A must equal the oracle's root of the mean over ALL pixels, and
    the plain iteration's A, to the iteration's tolerance; tau is then streamed once or twice instead of 4-5 times.  The
    subsample sums themselves are checked against a float64 numpy sum over the chunks of the definition in lya.h."""
    rng = np.random.default_rng(92)
    n = 3_000_017
    t = np.exp(rng.normal(-0.4, 2.3, n)).astype(np.float32)               # max ~ 1e5 x median
    t[rng.integers(0, n, 50)] = 0.0
    tau = torch.from_numpy(t).cuda()
    A_ref, _, _ = oracle.normalize_mean_flux(t.astype(np.float64), 0.8)
    try:
        for view, off in ((tau, 0), (tau[3:], 3)):                        # aligned and unaligned (head scalars)
            ctx.set_normalize_subsample(0, 0)
            A0, _, it0, _ = ctx.normalize_mean_flux(view, 0.8)
            st0 = ctx.last_normalize_stats()
            assert st0 == dict(tau_passes=it0, sub_passes=0, row_pass=0, n_sub=0)
            ctx.set_normalize_subsample(4, 0)
            A1, f1, it1, _ = ctx.normalize_mean_flux(view, 0.8)
            st1 = ctx.last_normalize_stats()
            assert abs(A1 / A0 - 1) < 2e-7 and st1["sub_passes"] >= 2 and it1 == st1["tau_passes"] <= 2 < it0
            if off == 0:
                assert abs(A1 / A_ref - 1) < 1e-6
            s, _ = ctx.flux_partial_sums(view, [A1])
            assert abs(s[0] / view.numel() - 0.8) < 1e-6
            # the subsample: float4 body after the head, chunks of 256 float4, every 4th
            tv = t[off:].astype(np.float64)
            head = (-(tau.data_ptr() + 4 * off) % 16) // 4
            body = tv[head: head + ((tv.size - head) // 4) * 4]
            chunks = [body[c: c + 1024] for c in range(0, body.size, 4096)]
            sub = np.concatenate(chunks)
            assert st1["n_sub"] == sub.size
            sums, npx = ctx.flux_moment_sums_sub(view, 0.37, 4)
            assert npx == sub.size
            e = np.exp(-0.37 * sub)
            for k in range(5):
                assert abs(sums[k] / (sub ** k * e).sum() - 1) < 2e-6
            full, npx1 = ctx.flux_moment_sums_sub(view, 0.37, 1)
            assert npx1 == view.numel() and full == ctx.flux_moment_sums(view, 0.37)
        # the sharded loop nests the same way and lands on the same root
        ctx.set_normalize_subsample(0, 0)
        stats = {}
        A2, _, it2 = lya.normalize_mean_flux_sharded(ctx, tau, 0.8, n, sub_every=4, sub_min_pix=0, stats=stats)
        assert abs(A2 / A_ref - 1) < 1e-6 and stats["sub_passes"] >= 2 and it2 <= 2
        # a subsample of zeros (every chunk it holds is empty) must not derail the full iteration
        z = tau.clone()
        zb = z[(-z.data_ptr() % 16) // 4:]
        for c in range(0, zb.numel(), 4096):
            zb[c: c + 1024] = 0.0
        ctx.set_normalize_subsample(4, 0)
        A3, _, _, _ = ctx.normalize_mean_flux(z, 0.8)
        A3_ref, _, _ = oracle.normalize_mean_flux(z.cpu().numpy().astype(np.float64), 0.8)
        assert abs(A3 / A3_ref - 1) < 1e-6
    finally:
        ctx.set_normalize_subsample(32, 1 << 24)


def test_flux_in_place_and_ragged(ctx, oracle):
    rng = np.random.default_rng(3)
    t = np.exp(rng.normal(-0.5, 1.5, 100_003)).astype(np.float32)
    tau = torch.from_numpy(t).cuda()
    F = ctx.flux(tau, 1.37)
    ref = oracle.flux(t.astype(np.float64), 1.37)
    assert np.abs(F.cpu().numpy() - ref).max() < 2e-7
    t2 = tau.clone()
    ctx.flux(t2, 1.37, out=t2)
    assert torch.equal(t2, F)
    F3 = ctx.flux(tau[3:], 1.37)
    assert torch.equal(F3, F[3:])


def test_forest_host_matches_stepwise_path(ctx, oracle):
    """lya_forest_host = slab-streamed fused S1+S3 with per-sightline moments, S4 started from them, S5: bit-equal to
    the same steps called one by one on the whole grid, for every slab size."""
    w = scaled(WORKLOADS[2], 128)
    delta, v = gpu_fields(w)
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, delta)
    rowm = torch.empty((128 * 128, 5), dtype=torch.float64, device="cuda")
    tau = ctx.tau_sightlines_opt(p, 0, v[0], n_hi=n_hi, b_kms=b, row_moments=rowm)
    A, f, it, _ = ctx.normalize_mean_flux(tau, w.f_target, row_moments=rowm)
    F = ctx.flux(tau, A)
    dh, vh = delta.cpu().pin_memory(), v[0].cpu().pin_memory()
    tau_h = torch.empty_like(dh).pin_memory()
    flux_h = torch.empty_like(dh).pin_memory()
    for slab in (0, 1, 50, 128):
        A2, f2, it2 = ctx.forest_host(p, 0, dh, vh, w.f_target, slab_nz=slab, tau_h=tau_h, flux_h=flux_h)
        assert torch.equal(tau_h, tau.cpu()) and A2 == A and it2 == it
        assert torch.equal(flux_h, F.cpu())
    # the three-step form with the caller owning S4 (what a rank of a sharded run does)
    A3, f3, it3 = lya.forest_host_sharded(ctx, p, 0, dh, vh, w.f_target, tau.numel(), tau_h=tau_h, flux_h=flux_h)
    assert torch.equal(tau_h, tau.cpu()) and abs(A3 / A - 1) < 1e-9 and it3 == it
    # A3 differs from A in the last digits (host-side sum of per-call partials instead of the cooperative kernel's
    # order), so ex2.approx's argument does too: F may move by a couple of fp32 ulps (6e-8 each below 1)
    assert np.abs(flux_h.numpy() - F.cpu().numpy()).max() < 5e-7
    with pytest.raises(lya.LyaError):                                  # no resident tau any more
        ctx._check(lya.lib().lya_forest_host_finish(ctx._h, A, None))


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_row_moments_of_the_tau_epilogue(ctx, axis):
    """lya_tau_sightlines_opt(row_moments=...) leaves sum_i tau_i^k, k = 0..4, per sightline (fp32 within a tile of
    128 pixels, double above): against a float64 numpy sum of the tau it wrote, for all three axes, the windowed and
    fused variants, a ragged row length, and z-slabs; S4 started from them reaches the plain call's A."""
    nx, ny, nz = (300, 24, 20) if axis == 0 else (40, 264, 136)
    n = (nx, ny, nz)[axis]
    w = scaled(WORKLOADS[3], n)
    rng = np.random.default_rng(20 + axis)
    delta = torch.from_numpy(np.expm1(rng.normal(0, 1.2, (nz, ny, nx)) - 0.72).astype(np.float32)).cuda()
    v = torch.from_numpy(rng.normal(0, 100.0, (nz, ny, nx)).astype(np.float32)).cuda()
    p = lya.Params(nx=nx, ny=ny, nz=nz, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    n_sl = delta.numel() // n
    for kw in (dict(n_hi=n_hi, b_kms=b), dict(n_hi=n_hi, b_kms=b, windowed=True), dict(delta=delta)):
        rowm = torch.full((n_sl, 5), -1.0, dtype=torch.float64, device="cuda")
        tau = ctx.tau_sightlines_opt(p, axis, v, row_moments=rowm, **kw)
        t = np.moveaxis(tau.double().cpu().numpy(), 2 - axis, -1).reshape(n_sl, n)     # sightline index: lya.h
        ref = np.stack([(t ** k).sum(axis=1) for k in range(5)], axis=1)
        assert np.allclose(rowm.cpu().numpy(), ref, rtol=2e-6, atol=0), np.abs(rowm.cpu().numpy() / ref - 1).max()
        assert np.allclose(ctx.row_moment_sums(rowm), ref.sum(axis=0), rtol=1e-7)
        A0, _, it0, _ = ctx.normalize_mean_flux(tau, 0.8)
        A1, _, it1, _ = ctx.normalize_mean_flux(tau, 0.8, row_moments=rowm)
        assert abs(A1 / A0 - 1) < 2e-7 and it1 <= it0 + 1
    if axis < 2:                                                      # z-slabs write their own sightlines' moments
        rowm2 = torch.empty_like(rowm)
        per_plane = n_sl // nz
        for z0, z1 in ((0, 7), (7, 8), (8, nz)):
            ctx.tau_sightlines_opt(p, axis, v[z0:z1], delta=delta[z0:z1], nz_local=z1 - z0,
                                   row_moments=rowm2[z0 * per_plane:z1 * per_plane])
        assert torch.equal(rowm2, rowm)


def test_sharded_normalisation_on_one_gpu(ctx):
    """The slab / multi-rank S4 route (partial sums + host root update) agrees with the device-side loop."""
    w = scaled(WORKLOADS[2], 128)
    delta, v = gpu_fields(w)
    _, _, tau, A, f, it, _ = run_gpu(ctx, w, delta, v[0])
    A2, f2, it2 = lya.normalize_mean_flux_sharded(ctx, tau, w.f_target, tau.numel())
    assert abs(A2 / A - 1) < 1e-9 and abs(f2 - f) < 1e-9


# ------------------------------------------------------------------ windowed / fused tau
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_tau_windowed_and_fused_are_bit_identical_to_the_full_sum(ctx, oracle, axis):
    """LYA_TAU_WINDOWED leaves out only terms that are exactly 0 in fp32; LYA_TAU_FROM_DENSITY applies S1 with
    lya_gas_from_density's arithmetic while staging: both must reproduce the two-call full sum bit for bit
    (whose parity with the oracle the tests above establish), and the window must really shrink the work."""
    w = scaled(WORKLOADS[4], 512) if axis == 0 else scaled(WORKLOADS[3], 192)
    n = w.n
    nz = 6 if axis == 0 else n
    f = inputs.make_fields(w, device="cuda", z0=0, z1=nz, axes=(axis,))
    delta, v = f["delta"], f["v_pec"][axis]
    p = lya.Params(nx=n, ny=n, nz=nz, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    if axis == 2:
        p.nz = n
    n_hi, b = ctx.gas_from_density(p, delta)
    full = ctx.tau_sightlines(p, axis, n_hi, b, v)
    win, pairs_w = ctx.tau_sightlines_opt(p, axis, v, n_hi=n_hi, b_kms=b, windowed=True, count_pairs=True)
    fus, pairs_f = ctx.tau_sightlines_opt(p, axis, v, delta=delta, count_pairs=True)
    both = ctx.tau_sightlines_opt(p, axis, v, delta=delta, windowed=True)
    assert torch.equal(win, full) and torch.equal(fus, full) and torch.equal(both, full)
    assert pairs_f == delta.numel() * n                      # full sum: N pairs per pixel
    # a tile walks 128 + 2 * reach sources instead of N: a third of them at N = 512, most of them at N = 192
    assert pairs_w < (0.5 if axis == 0 else 0.95) * pairs_f, (pairs_w, pairs_f)
    if axis == 0:                                            # and against the oracle on a few rows
        po = oracle.Params.from_workload(w)
        _, n_ref, b_ref = oracle.gas_from_density(po, delta[0, :8].cpu().numpy())
        ref = oracle.tau_rows(po, n_ref, b_ref, v[0, :8].cpu().numpy())
        assert_tau_close(both[0, :8].cpu().numpy(), ref, "windowed+fused")


def test_tau_windowed_falls_back_when_the_reach_does_not_fit(ctx):
    """Huge velocities / tiny rows: the window would exceed the row, the full (or general) loop must run."""
    w = scaled(WORKLOADS[1], 64)
    f = inputs.make_fields(w, device="cuda", z0=0, z1=4)
    delta, v = f["delta"], (f["v_pec"][0] * 40.0).contiguous()          # |v| of order V
    p = lya.Params(nx=64, ny=64, nz=4, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    full = ctx.tau_sightlines(p, 0, n_hi, b, v)
    win, pairs = ctx.tau_sightlines_opt(p, 0, v, n_hi=n_hi, b_kms=b, windowed=True, count_pairs=True)
    assert torch.equal(win, full) and pairs == delta.numel() * 64
    with pytest.raises(lya.LyaError):
        lya.lib().lya_tau_sightlines_opt  # noqa: B018  (symbol exists)
        ctx._check(lya.lib().lya_tau_sightlines_opt(ctx._h, lya.C.byref(p.c()), 0, 4, 8, n_hi.data_ptr(),
                                                    b.data_ptr(), v.data_ptr(), full.data_ptr(), None, None))


# ------------------------------------------------------------------ empty inputs and size limits
def test_empty_inputs_and_size_limits(ctx):
    p = lya.Params(nx=64, ny=4, nz=1, box_mpch=20.0, z=2.5, T0=1e4, gamma=1.5)
    empty = torch.empty((0,), device="cuda")
    n_hi, b = ctx.gas_from_density(p, empty)                        # zero cells: nothing launched, no error
    assert n_hi.numel() == 0 and b.numel() == 0
    assert ctx.flux(empty, 0.5).numel() == 0
    s, d = ctx.flux_partial_sums(empty, [0.3, 0.6])
    assert s == [0.0, 0.0] and d == [0.0, 0.0]
    assert ctx.flux_moment_sums(empty, 0.3) == [0.0] * 5
    counts, pdf = ctx.flux_pdf(empty)
    assert counts.sum() == 0 and not pdf.any()
    with pytest.raises(lya.LyaError) as e:
        ctx.normalize_mean_flux(empty, 0.8)                         # the mean of nothing is undefined
    assert e.value.status == lya.EINVAL
    assert ctx.observe_rows(torch.empty((0, 64), device="cuda"), 5.0, 10.0).shape == (0, 64)
    # a sightline whose staged cells (16 B each) exceed one SM's shared memory is refused, not mis-computed
    n = 20000
    big = lya.Params(nx=n, ny=1, nz=1, box_mpch=2000.0, z=2.5, T0=1e4, gamma=1.5)
    x = torch.ones((1, 1, n), device="cuda")
    for axis_p, arr in ((big, x),):
        with pytest.raises(lya.LyaError) as e:
            ctx.tau_sightlines(axis_p, 0, arr, arr, arr)
        assert e.value.status == lya.EINVAL and "shared memory" in str(e.value)
    # the longest row that does fit (14 000 pixels: 224 KB of cells) still runs and gives the uniform-field value
    n = 14000
    ok = lya.Params(nx=n, ny=2, nz=1, box_mpch=1500.0, z=2.5, T0=1e4, gamma=1.5)
    n_hi, b = ctx.gas_from_density(ok, torch.zeros((1, 2, n), device="cuda"))
    tau = ctx.tau_sightlines(ok, 0, n_hi, b, torch.zeros((1, 2, n), device="cuda"))
    torch.cuda.synchronize()
    assert torch.allclose(tau, tau[0, 0, 0].expand_as(tau), rtol=1e-6) and tau[0, 0, 0].item() > 0


def test_nan_in_one_sightline_stays_in_that_sightline(ctx):
    """The per-cell content is not scanned (lya.h): a NaN density or velocity poisons its own sightline only."""
    w = scaled(WORKLOADS[2], 256)
    f = inputs.make_fields(w, device="cuda", z0=0, z1=2)
    delta, v = f["delta"].clone(), f["v_pec"][0].clone()
    p = lya.Params(nx=256, ny=256, nz=2, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    n_hi, b = ctx.gas_from_density(p, delta)
    good = ctx.tau_sightlines(p, 0, n_hi, b, v)
    delta[0, 7, 100] = float("nan")
    v[1, 200, 3] = float("nan")
    n_hi, b = ctx.gas_from_density(p, delta)
    for kw in (dict(), dict(windowed=True)):
        tau = ctx.tau_sightlines_opt(p, 0, v, n_hi=n_hi, b_kms=b, **kw)
        bad = torch.isnan(tau).any(dim=2)
        assert bad[0, 7] and bad[1, 200] and int(bad.sum()) == 2
        assert torch.equal(tau[~bad], good[~bad])
