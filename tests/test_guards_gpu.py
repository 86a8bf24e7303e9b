"""Out-of-bounds and race checks written by hand (compute-sanitizer is closed on this pool: profiles/r2_sanitizer.md).

memcheck stand-in: every array a kernel writes is an interior view of a larger buffer whose guard bands hold a
sentinel bit pattern; after the call the guards must be bit-for-bit intact and the interior fully written.  Every
array a kernel reads is embedded in NaN guards, and the result must be bit-identical to a run on separately
allocated inputs -- a read past either end that reaches the arithmetic shows up as a different (NaN) output.
Offsets are odd on purpose (4-byte aligned only) to take the scalar edge paths too.

racecheck stand-in: the kernels that synchronise by hand (named barriers and the atomic row scheduler of
tau_x_kernel with G = 1, 2, 4, 8 warps per group; the CTA-wide staging of tau_strided_kernel; the grid barrier and
ping-pong partials of normalize_kernel; the shared-memory histograms and FFT exchanges) must give bit-identical
results run after run, with the schedule perturbed by a competing kernel on another stream.
"""
import numpy as np
import pytest
import torch

from paper_1105_4747_b200 import lya
from paper_1105_4747_b200.workloads import WORKLOADS, scaled

pytestmark = pytest.mark.gpu

SENT = 0x7FC0DEAD          # a quiet-NaN payload as int32
GUARD = 1031               # floats on either side: odd, so the arrays are 4-byte aligned only (scalar edge paths);
GUARD16 = 1032             # a multiple of 4 keeps torch's 16-byte alignment (vector paths)


@pytest.fixture(scope="module")
def ctx():
    c = lya.Context(0)
    yield c
    c.close()


class Guarded:
    """An n-float output window inside a sentinel-filled buffer."""

    def __init__(self, n, dtype=torch.float32, lead=GUARD):
        self.n, self.lead = n, lead
        words = 1 if dtype == torch.float32 else 2
        self.raw = torch.full(((n + 2 * lead + 8) * words,), SENT, dtype=torch.int32, device="cuda")
        self.view = self.raw.view(dtype)[lead: lead + n]

    def check(self, what, must_be_written=True):
        r = self.raw.view(self.view.dtype)
        ints = lambda t: t.view(torch.int32)
        assert bool((ints(r[: self.lead]) == SENT).all()), f"{what}: wrote before the array"
        assert bool((ints(r[self.lead + self.n:]) == SENT).all()), f"{what}: wrote past the array"
        if must_be_written and self.n:
            iv = ints(self.view.contiguous())
            if self.view.dtype == torch.float32:
                assert not bool((iv == SENT).any()), f"{what}: left elements unwritten"
            else:
                assert not bool(((iv[0::2] == SENT) & (iv[1::2] == SENT)).any()), f"{what}: left elements unwritten"


def embedded(t, lead=GUARD):
    """A copy of t with NaN guards on both sides."""
    buf = torch.full((t.numel() + 2 * lead,), float("nan"), dtype=t.dtype, device="cuda")
    buf[lead: lead + t.numel()] = t.reshape(-1)
    return buf[lead: lead + t.numel()].view(t.shape)


def fields(shape, seed, sigma_v=100.0):
    rng = np.random.default_rng(seed)
    delta = torch.from_numpy(np.expm1(rng.normal(0, 1.2, shape) - 0.72).astype(np.float32)).cuda()
    v = torch.from_numpy(rng.normal(0, sigma_v, shape).astype(np.float32)).cuda()
    return delta, v


@pytest.mark.parametrize("lead", [GUARD, GUARD16])
@pytest.mark.parametrize("n", [1, 5, 1027, 300_001])
def test_gas_and_flux_stay_inside_their_arrays(ctx, n, lead):
    p = lya.Params.from_workload(WORKLOADS[1])
    delta, _ = fields((n,), n)
    ref_n, ref_b = ctx.gas_from_density(p, delta)
    G = lambda m: Guarded(m, lead=lead)
    emb = lambda t: embedded(t, lead)
    g_n, g_b = G(n), G(n)
    ctx.gas_from_density(p, emb(delta), g_n.view, g_b.view)
    g_n.check("gas n_hi"); g_b.check("gas b")
    assert torch.equal(g_n.view, ref_n) and torch.equal(g_b.view, ref_b)
    tau = delta.abs()
    ref_f = ctx.flux(tau, 0.9)
    g_f = G(n)
    ctx.flux(emb(tau), 0.9, out=g_f.view)
    g_f.check("flux")
    assert torch.equal(g_f.view, ref_f)
    g_f2 = G(n)
    F, counts, _ = ctx.flux_with_pdf(emb(tau), 0.9, out=g_f2.view)
    g_f2.check("flux_with_pdf")
    assert torch.equal(g_f2.view, ref_f) and int(counts.sum()) == n


@pytest.mark.parametrize("axis,shape", [(0, (3, 5, 333)), (0, (2, 9, 1024)), (0, (1, 7, 2052)), (0, (1, 3, 4100)),
                                        (1, (5, 136, 43)), (2, (72, 6, 43))])
@pytest.mark.parametrize("variant", ["plain", "windowed", "fused", "windowed_fused"])
@pytest.mark.parametrize("lead", [GUARD, GUARD16])
def test_tau_stays_inside_its_arrays(ctx, axis, shape, variant, lead):
    emb = lambda t: embedded(t, lead)
    nz, ny, nx = shape
    n = (nx, ny, nz)[axis]
    w = scaled(WORKLOADS[3], max(n, 64))
    p = lya.Params(nx=nx, ny=ny, nz=nz, box_mpch=w.box_mpch * n / max(n, 64), z=w.z, T0=w.T0, gamma=w.gamma)
    delta, v = fields(shape, 7 * n + axis)
    n_hi, b = ctx.gas_from_density(p, delta)
    kw = dict(windowed="windowed" in variant)
    kw.update(dict(delta=delta) if "fused" in variant else dict(n_hi=n_hi, b_kms=b))
    n_sl = delta.numel() // n
    ref_m = torch.empty((n_sl, 5), dtype=torch.float64, device="cuda")
    ref = ctx.tau_sightlines_opt(p, axis, v, row_moments=ref_m, **kw)
    g_t, g_m = Guarded(delta.numel(), lead=lead), Guarded(5 * n_sl, torch.float64, lead=GUARD + 1)
    kw2 = dict(windowed=kw["windowed"])
    kw2.update(dict(delta=emb(delta)) if "fused" in variant else dict(n_hi=emb(n_hi), b_kms=emb(b)))
    ctx.tau_sightlines_opt(p, axis, emb(v), tau=g_t.view.view(shape), row_moments=g_m.view.view(n_sl, 5), **kw2)
    g_t.check(f"tau {variant} axis {axis}"); g_m.check(f"row moments {variant} axis {axis}")
    assert torch.equal(g_t.view.view(shape), ref) and torch.equal(g_m.view.view(n_sl, 5), ref_m)
    assert bool(torch.isfinite(ref).all())


@pytest.mark.parametrize("n,fwhm,dlam", [(256, 7.0, 0.05), (1024, 224.0, 1.0375), (1000, 170.0, 1.0), (3001, 30.0, 0.3)])
def test_observe_rows_stays_inside_its_arrays(ctx, n, fwhm, dlam):
    rows = 37
    rng = np.random.default_rng(n)
    flux = torch.from_numpy(rng.uniform(0, 1, (rows, n)).astype(np.float32)).cuda()
    dv = 41.0
    bin_kms = lya.bin_kms_from_angstrom(2.5, dlam)
    nb = lya.lib().lya_instrument_bins(n, dv, lya.C.byref(lya.CInstrument(fwhm, bin_kms, 5.0)))
    noise = torch.from_numpy(rng.normal(0, 1, (rows, nb)).astype(np.float32)).cuda()
    ref = ctx.observe_rows(flux, dv, fwhm, bin_kms, 5.0, noise)
    for lead in (GUARD, GUARD16):          # unaligned rows (general kernel) and 16-byte aligned rows (lean kernel)
        g = Guarded(rows * nb, lead=lead)
        ctx.observe_rows(embedded(flux, lead), dv, fwhm, bin_kms, 5.0, embedded(noise, lead), g.view.view(rows, nb))
        g.check("observe_rows")
        assert torch.allclose(g.view.view(rows, nb), ref, rtol=0, atol=2e-6)


def test_forest_host_stays_inside_the_host_buffers(ctx):
    w = scaled(WORKLOADS[2], 48)
    p = lya.Params.from_workload(w)
    delta, v = fields((48, 48, 48), 48)
    n = delta.numel()
    lead = 777
    def host_guarded():
        raw = torch.full((n + 2 * lead,), SENT, dtype=torch.int32).pin_memory()
        return raw, raw.view(torch.float32)[lead: lead + n].view(48, 48, 48)
    raw_t, tau_h = host_guarded()
    raw_f, flux_h = host_guarded()
    dh = torch.full((n + 2 * lead,), float("nan")).pin_memory()
    vh = torch.full((n + 2 * lead,), float("nan")).pin_memory()
    dh[lead: lead + n] = delta.cpu().reshape(-1)
    vh[lead: lead + n] = v.cpu().reshape(-1)
    for slab in (0, 5, 48):
        A, f, it = ctx.forest_host(p, 0, dh[lead: lead + n].view(48, 48, 48), vh[lead: lead + n].view(48, 48, 48),
                                   w.f_target, slab_nz=slab, tau_h=tau_h, flux_h=flux_h)
        for raw, what in ((raw_t, "tau_h"), (raw_f, "flux_h")):
            assert bool((raw[:lead] == SENT).all()) and bool((raw[lead + n:] == SENT).all()), what
            assert not bool((raw[lead: lead + n] == SENT).any()), what
        assert bool(torch.isfinite(tau_h).all()) and bool(torch.isfinite(flux_h).all()) and 0 < A < 1e3


def _busy(stream, x):
    with torch.cuda.stream(stream):
        for _ in range(8):
            x.mul_(1.0000001)


@pytest.mark.parametrize("n,rows", [(512, 4099), (1024, 2051), (2048, 1033), (4096, 517), (8192, 130)])
def test_tau_x_is_reproducible_under_a_perturbed_schedule(ctx, n, rows):
    """G = 1, 2, 4, 8, 16 warps per group share a staged row through named barriers; rows come from an atomic counter.
    A race in either shows as run-to-run differences once another kernel competes for the SMs."""
    w = scaled(WORKLOADS[4], n)
    p = lya.Params(nx=n, ny=rows, nz=1, box_mpch=w.box_mpch, z=w.z, T0=w.T0, gamma=w.gamma)
    delta, v = fields((1, rows, n), n)
    n_hi, b = ctx.gas_from_density(p, delta)
    side = torch.cuda.Stream()
    x = torch.ones(1 << 24, device="cuda")
    for kw in (dict(n_hi=n_hi, b_kms=b), dict(n_hi=n_hi, b_kms=b, windowed=True), dict(delta=delta)):
        m0 = torch.empty((rows, 5), dtype=torch.float64, device="cuda")
        t0 = ctx.tau_sightlines_opt(p, 0, v, row_moments=m0, **kw)
        for rep in range(3):
            _busy(side, x)
            m1 = torch.empty_like(m0)
            t1 = ctx.tau_sightlines_opt(p, 0, v, row_moments=m1, **kw)
            torch.cuda.synchronize()
            assert torch.equal(t1, t0) and torch.equal(m1, m0), (kw.keys(), rep)


def test_reductions_are_reproducible_under_a_perturbed_schedule(ctx):
    rng = np.random.default_rng(5)
    n = 20_000_003
    tau = torch.from_numpy(np.exp(rng.normal(-0.5, 1.6, n)).astype(np.float32)).cuda()
    side = torch.cuda.Stream()
    x = torch.ones(1 << 24, device="cuda")
    ctx.set_normalize_subsample(8, 0)
    try:
        first = None
        for rep in range(4):
            _busy(side, x)
            A, f, it, _ = ctx.normalize_mean_flux(tau, 0.8)
            s5 = ctx.flux_moment_sums(tau, A)
            F, counts, _ = ctx.flux_with_pdf(tau, A)
            rows = F[: 4096 * 1024].view(4096, 1024)
            P = ctx.flux_power_rows(rows, 41.0, 0.8)
            got = (A, f, it, tuple(s5), tuple(counts.tolist()))
            if first is None:
                first, P0 = got, P
            assert got == first
            # the power accumulator is summed with double atomics across CTAs: order-dependent in the last bits only
            assert np.allclose(P, P0, rtol=1e-12, atol=0)
    finally:
        ctx.set_normalize_subsample(32, 1 << 24)
