"""lya_flux_moment_sums_static (include/lya.h): the five tilted moments of S4 from an entry point that
allocates nothing -- its per-block scratch is a static __device__ array -- against the existing lya_flux_moment_sums,
on two calls in a row (the second one finds the first one's partials in the shared array).  Collected last on purpose
(the file name): the run uses pytest -x."""
import numpy as np
import pytest
import torch

from paper_1105_4747_b200 import lya

pytestmark = pytest.mark.gpu

RTOL = 2e-6          # the relative tolerance tests/test_parity_gpu.py puts on the moment sums


def heavy_tailed_tau(n, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    return torch.exp(1.5 * torch.randn(n, device="cuda", generator=g) - 1.0)     # lognormal, like tau on these fields


@pytest.fixture(scope="module")
def ctx():
    c = lya.Context(0)
    yield c
    c.close()


def test_static_scratch_moment_sums_match_the_existing_path_twice_in_a_row(ctx):
    # several blocks of 65536 pixels, a ragged last block, a tail that is not a multiple of four; then a LARGER and a
    # SMALLER input back to back: stale partials of the earlier call sit beyond the later call's blocks
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    for call, (n, a_trial, seed) in enumerate(((5 * 65536 + 4099, 0.37, 1), (11 * 65536 + 2, 0.0, 2), (70001, 1.9, 3))):
        tau = heavy_tailed_tau(n, seed)
        ref = ctx.flux_moment_sums(tau, a_trial)                     # the existing path (cudaMalloc'ed partials, HOST out)
        launches = ctx.launch_count
        out.fill_(float("nan"))
        got = ctx.flux_moment_sums_static(tau, a_trial, out)
        assert ctx.launch_count == launches + 2
        got = got.cpu().numpy()
        assert np.all(np.isfinite(got)), (call, got)
        assert np.allclose(got, np.array(ref), rtol=RTOL, atol=0), (call, got, ref)
        # and against the definition, in double on the host
        t = tau.double().cpu().numpy()
        e = np.exp(-a_trial * t)
        exact = np.array([(t ** k * e).sum() for k in range(5)])
        assert np.allclose(got, exact, rtol=RTOL, atol=0), (call, got, exact)
        # the same input again: bit-identical (fixed block -> pixel assignment, fixed-order finish)
        again = ctx.flux_moment_sums_static(tau, a_trial, torch.empty_like(out)).cpu().numpy()
        assert np.array_equal(got, again)


def test_static_scratch_unaligned_empty_and_limits(ctx):
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    tau = heavy_tailed_tau(3 * 65536 + 77, 4)
    view = tau[1:]                                                   # 4-byte aligned only: the scalar path
    ref = ctx.flux_moment_sums(view, 0.5)
    got = ctx.flux_moment_sums_static(view, 0.5, out).cpu().numpy()
    assert np.allclose(got, np.array(ref), rtol=RTOL, atol=0)
    empty = torch.empty(0, device="cuda")
    assert ctx.flux_moment_sums_static(empty, 0.3, out).cpu().tolist() == [0.0] * 5
    # sizes beyond the static scratch are refused with a message, before anything is launched (no such tensor is made:
    # the size check comes first and the pointer is never read)
    L = lya.lib()
    launches = ctx.launch_count
    st = L.lya_flux_moment_sums_static(ctx._h, tau.data_ptr(), lya.STATIC_MAX_PIX + 1, 0.5, out.data_ptr())
    assert st == lya.EINVAL and b"LYA_STATIC_MAX_PIX" in L.lya_last_error(ctx._h)
    assert ctx.launch_count == launches
    assert L.lya_flux_moment_sums_static(ctx._h, tau.data_ptr(), 16, -1.0, out.data_ptr()) == lya.EINVAL
    assert L.lya_flux_moment_sums_static(ctx._h, tau.data_ptr(), 16, 0.5, None) == lya.EINVAL
    with pytest.raises(TypeError):
        ctx.flux_moment_sums_static(tau, 0.5, torch.empty(5, device="cuda"))       # float32 out


def test_static_scratch_at_the_maximum_size(ctx):
    """LYA_STATIC_MAX_PIX itself (2^30 pixels = 4 GiB of tau, all 16384 blocks of the static array)."""
    n = lya.STATIC_MAX_PIX
    tau = torch.empty(n, device="cuda")
    tau[: n // 2] = 0.25
    tau[n // 2:] = 2.0
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    got = ctx.flux_moment_sums_static(tau, 0.7, out).cpu().numpy()
    exact = np.array([(n // 2) * (0.25 ** k * np.exp(-0.7 * 0.25) + 2.0 ** k * np.exp(-0.7 * 2.0)) for k in range(5)])
    assert np.allclose(got, exact, rtol=RTOL, atol=0), (got, exact)
    assert np.allclose(got, np.array(ctx.flux_moment_sums(tau, 0.7)), rtol=RTOL, atol=0)
