"""GPU parity of the instrument model, flux PDF and 1D flux power against
oracle/lya_obs_oracle.c, through the C ABI.  Tolerances: observed flux 1e-5 absolute (the north_star's bar for
F); PDF counts bit-exact against the oracle's double-precision decision at the real edges (reading O4); power 1e-4 relative plus 1e-9 of
the largest mode (fp32 FFT of dF)."""
import numpy as np
import pytest
import torch

from paper_1105_4747_b200 import inputs, lya
from paper_1105_4747_b200.workloads import WORKLOADS

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = lya.Context(0)
    yield c
    c.close()


@pytest.fixture(scope="module")
def obs():
    from oracle import lya_obs_oracle
    lya_obs_oracle.build()
    return lya_obs_oracle


@pytest.fixture(scope="module")
def flux_rows(ctx):
    """F of the first 4 planes of config 2 (1024 rows of 256 pixels) through the library's own S1-S5."""
    w = WORKLOADS[2]
    f = inputs.make_fields(w, device="cuda", z0=0, z1=4)
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, f["delta"])
    tau = ctx.tau_sightlines(p, 0, n_hi, b, f["v_pec"][0], nz_local=4)
    A, _, _, _ = ctx.normalize_mean_flux(tau, w.f_target)
    F = ctx.flux(tau, A).reshape(-1, w.n)
    return F, lya.scalars(p, 0)["dv_kms"], w


# the paper's three instruments + pure cases
@pytest.mark.parametrize("fwhm,dlam,snr", [(7.0, 0.05, 50.0), (170.0, 1.0, 3.8), (224.0, 1.0375, 5.0),
                                           (120.0, 0.0, 0.0), (0.0, 1.0375, 0.0), (0.0, 0.0, 5.0)])
def test_observe_rows_parity(ctx, obs, flux_rows, fwhm, dlam, snr):
    F, dv, w = flux_rows
    bin_kms = lya.bin_kms_from_angstrom(w.z, dlam) if dlam > 0 else 0.0
    assert bin_kms == pytest.approx(obs.bin_kms_from_angstrom(w.z, dlam), rel=1e-12)
    nb = obs.n_bins(w.n, dv, bin_kms)
    g = torch.Generator(device="cuda").manual_seed(7)
    noise = torch.randn((F.shape[0], nb), device="cuda", generator=g) if snr > 0 else None
    out = ctx.observe_rows(F, dv, fwhm, bin_kms, snr, noise)
    torch.cuda.synchronize()
    rows = slice(0, 192)
    ref = obs.observe_rows(F[rows].cpu().numpy(), dv, fwhm, bin_kms, snr,
                           None if noise is None else noise[rows].cpu().numpy())
    assert out.shape == (F.shape[0], nb) and ref.shape[1] == nb
    err = np.abs(out[rows].cpu().numpy() - ref).max()
    assert err < 1e-5, f"observed flux max abs err {err:.2e}"


# (512, 30.0) and (1024, 53.5): 25 and 41 tap slots, the packed-FP32 (FFMA2) convolution up to its last
# instantiation; (1000, 55.0) is the first size past it (scalar FFMA)
@pytest.mark.parametrize("n,fwhm", [(5, 3.0), (13, 40.0), (100, 9.0), (257, 300.0), (512, 30.0), (1024, 53.5), (1000, 55.0), (2048, 100.0), (3000, 30.0), (4096, 224.0)])
def test_observe_rows_ragged_and_wide_kernels(ctx, obs, n, fwhm):
    """Ragged row lengths, a Gaussian as wide as the row (every nearest image contributes), bins that do not
    divide the row."""
    rng = np.random.default_rng(n)
    F = torch.from_numpy(rng.uniform(0, 1, (7, n)).astype(np.float32)).cuda()
    dv, bin_kms = 6.5, 17.3 if n > 5 else 0.0
    out = ctx.observe_rows(F, dv, fwhm, bin_kms)
    ref = obs.observe_rows(F.cpu().numpy(), dv, fwhm, bin_kms, 0.0)
    assert out.shape == ref.shape
    assert np.abs(out.cpu().numpy() - ref).max() < 1e-5


def test_observe_rows_errors(ctx):
    F = torch.rand((4, 64), device="cuda")
    with pytest.raises(lya.LyaError):
        ctx.observe_rows(F, 5.0, 10.0, 1000.0)                     # bin wider than the row
    with pytest.raises(lya.LyaError):
        ctx.observe_rows(F, 5.0, 10.0, 0.0, snr=5.0)               # noise requested, no draws given
    with pytest.raises(lya.LyaError):
        ctx.observe_rows(F, 5.0, 10.0, 0.0, out=F)                 # aliasing


def test_flux_pdf_bit_exact(ctx, obs, flux_rows):
    F, dv, w = flux_rows
    g = torch.Generator(device="cuda").manual_seed(11)
    noisy = (F + 0.2 * torch.randn(F.shape, device="cuda", generator=g)).contiguous()    # spills over both ends
    for arr in (F, noisy, noisy.reshape(-1)[3:100_002]):            # the last one: unaligned base, ragged length
        arr = arr.contiguous() if arr.dim() == 2 else arr
        counts, pdf = ctx.flux_pdf(arr)
        c_ref, p_ref = obs.flux_pdf(arr.cpu().numpy())
        assert np.array_equal(counts, c_ref)
        assert np.allclose(pdf, p_ref, rtol=1e-14)
        assert counts.sum() == arr.numel()
    counts, _ = ctx.flux_pdf(noisy, n_bins=100, f_lo=-0.5, width=0.02)
    assert np.array_equal(counts, obs.flux_pdf(noisy.cpu().numpy(), 100, -0.5, 0.02)[0])


def test_flux_pdf_edge_decisions_match_the_real_number_bins(ctx, obs):
    """PAPER.md:156 (reading O4): fluxes AT every interior edge's nearest fp32 and one ulp either side, the dyadic
    edges, out-of-range values, infinities and NaN -- the kernel's counts must equal the oracle's double-precision
    decision against the real edges, both for lya_flux_pdf and for the fused S5 + PDF pass."""
    vals = []
    for b in range(1, 21):
        e = np.float32((2 * b - 1) / 40.0)
        vals += [np.nextafter(e, np.float32(-9)), e, np.nextafter(e, np.float32(9))]
    vals += [np.float32(x) for x in (-0.025, -0.0250001, 1.025, 1.0250001, -3.0, 7.0, 0.0, 1.0, 0.125, 0.375, 0.625, 0.875)]
    vals += [np.float32("inf"), np.float32("-inf"), np.float32("nan")]
    base = np.array(vals, dtype=np.float32)
    F = torch.from_numpy(np.tile(base, 997)[:-1].copy()).cuda()           # ragged length, every thread sees edges
    counts, _ = ctx.flux_pdf(F)
    assert np.array_equal(counts, obs.flux_pdf(F.cpu().numpy())[0])
    one_each = [ctx.flux_pdf(torch.from_numpy(np.array([v], dtype=np.float32)).cuda())[0] for v in base]
    for v, c in zip(base, one_each):
        assert np.array_equal(c, obs.flux_pdf(np.array([v], dtype=np.float32))[0]), float(v)
    # the fused pass bins the F it writes: tau = -ln F / A reproduces fluxes close to the edges; whatever F
    # comes out, its counts must equal the oracle's on that same F
    tau = (-torch.log(F[torch.isfinite(F) & (F > 0)]) / 0.7).contiguous()
    F2, c2, _ = ctx.flux_with_pdf(tau, 0.7)
    assert np.array_equal(c2, obs.flux_pdf(F2.cpu().numpy())[0])
    # other bin layouts, including one whose edges are all fp32-representable
    g = torch.Generator(device="cuda").manual_seed(5)
    R = (torch.rand(300_001, device="cuda", generator=g) * 2.4 - 0.7).contiguous()
    R[:4096] = torch.arange(4096, device="cuda") / 64.0 - 8.0              # multiples of 1/64: on the edges below
    for nb, lo, w in ((100, -0.5, 0.02), (64, -0.5, 0.03125), (7, 0.1, 0.13), (256, -1.0, 0.01)):
        assert np.array_equal(ctx.flux_pdf(R, nb, lo, w)[0], obs.flux_pdf(R.cpu().numpy(), nb, lo, w)[0]), (nb, lo, w)


@pytest.mark.parametrize("n_rows", [1, 2, 333])
def test_flux_power_parity(ctx, obs, flux_rows, n_rows):
    F, dv, w = flux_rows
    Fr = F[:n_rows].contiguous()
    fbar = float(Fr.double().mean())
    P = ctx.flux_power_rows(Fr, dv, fbar)
    ref = obs.flux_power(Fr.cpu().numpy(), dv, fbar)
    assert P.shape == ref.shape == (w.n // 2 + 1,)
    assert np.all(np.abs(P - ref) <= 1e-4 * ref + 1e-9 * ref.max()), np.abs(P / ref - 1).max()


@pytest.mark.parametrize("n", [8, 64, 2048, 8192])
def test_flux_power_lengths_and_errors(ctx, obs, n):
    rng = np.random.default_rng(n)
    F = torch.from_numpy(rng.uniform(0.05, 1, (5, n)).astype(np.float32)).cuda()
    P = ctx.flux_power_rows(F, 2.0, 0.5)
    ref = obs.flux_power(F.cpu().numpy(), 2.0, 0.5)
    assert np.all(np.abs(P - ref) <= 1e-4 * ref + 1e-9 * ref.max())
    with pytest.raises(lya.LyaError):
        ctx.flux_power_rows(F[:, : n - 1].contiguous(), 2.0, 0.5)   # not a power of two


@pytest.mark.parametrize("n", [256, 512, 1024, 2048, 4096])
@pytest.mark.parametrize("n_rows", [1, 7, 22])
def test_flux_power_kernels_of_the_config_row_lengths(ctx, obs, n, n_rows):
    """Every compile-time plan (256 ... 4096) and both warp-per-transform kernels (1024: one warp per row pair; 2048: a
    team of two warps per pair) against the oracle's direct DFT: odd row counts (a last pair with no second row), fewer
    pairs than warps, and a 4-byte-aligned view (the kernels without cp.async staging)."""
    rng = np.random.default_rng(1000 * n + n_rows)
    host = rng.uniform(0.0, 1.0, (n_rows, n)).astype(np.float32)
    host[0] = 0.8                                                    # a constant row: only the k = 0 mode
    ref = obs.flux_power(host, 3.5, 0.6)
    buf = torch.empty(n_rows * n + 4, device="cuda")
    for off in (0, 1):                                               # 16-byte aligned, then 4-byte aligned only
        F = buf[off: off + n_rows * n].view(n_rows, n)
        F.copy_(torch.from_numpy(host))
        assert (F.data_ptr() % 16 == 0) == (off == 0)
        P = ctx.flux_power_rows(F, 3.5, 0.6)
        assert np.all(np.abs(P - ref) <= 1e-4 * ref + 1e-9 * ref.max()), (off, np.abs(P / ref - 1).max())


@pytest.mark.parametrize("n", [1024, 2048])
def test_flux_power_at_full_size_by_tiling(ctx, obs, n):
    """Configs 4 and 5 at the size bench.py times (2^30 pixels: about 295 row pairs per warp, so the fp32 accumulators'
    flush every 256 pairs is taken): the mean over rows of a block of rows repeated many times is the block's own, which
    the oracle can compute."""
    block, reps = 32, (1 << 30) // (32 * n)
    rng = np.random.default_rng(n)
    host = np.exp(-rng.lognormal(-1.0, 1.5, (block, n))).astype(np.float32)      # F = exp(-tau), heavy-tailed tau
    fbar = float(host.astype(np.float64).mean())
    ref = obs.flux_power(host, 51.5, fbar)
    F = torch.from_numpy(host).cuda().repeat(reps, 1)
    assert F.shape == (block * reps, n)
    P = ctx.flux_power_rows(F, 51.5, fbar)
    assert np.all(np.abs(P - ref) <= 1e-4 * ref + 1e-9 * ref.max()), np.abs(P / ref - 1).max()
    assert np.allclose(P, ctx.flux_power_rows(F, 51.5, fbar), rtol=1e-12)          # atomics: order-dependent only in the last bits


def test_flux_with_pdf_equals_the_two_calls(ctx, flux_rows):
    """S5 and the PDF fused in one pass: F and the counts are bit-identical to lya_flux + lya_flux_pdf."""
    w = WORKLOADS[2]
    f = inputs.make_fields(w, device="cuda", z0=0, z1=4)
    p = lya.Params.from_workload(w)
    n_hi, b = ctx.gas_from_density(p, f["delta"])
    tau = ctx.tau_sightlines(p, 0, n_hi, b, f["v_pec"][0], nz_local=4)
    for t in (tau, tau.reshape(-1)[5:200_003]):                       # aligned, and unaligned + ragged
        t = t.contiguous() if t.dim() == 3 else t
        F = ctx.flux(t, 0.7)
        c_ref, p_ref = ctx.flux_pdf(F)
        F2, counts, pdf = ctx.flux_with_pdf(t, 0.7)
        assert torch.equal(F2, F) and np.array_equal(counts, c_ref) and np.allclose(pdf, p_ref, rtol=1e-14)
    F3, counts, _ = ctx.flux_with_pdf(tau, 0.7, out=tau.clone(), n_bins=40, f_lo=0.0, width=0.025)
    assert counts.sum() == tau.numel()
