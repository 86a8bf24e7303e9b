"""Pins of oracle/lya_obs_oracle.c (instrument model, flux PDF, 1D flux power; PAPER.md:124,130,156,166,
172-176) against closed forms, invariants, special cases and a library FFT -- none re-types its formulas."""
import math

import numpy as np
import pytest


@pytest.fixture(scope="module")
def obs():
    from oracle import lya_obs_oracle
    lya_obs_oracle.build()
    return lya_obs_oracle


# ---------------------------------------------------------------- convolution
def test_constant_stays_constant(obs):
    F = np.full((3, 50), 0.37)
    assert np.allclose(obs.convolve_rows(F, 7.0, 40.0), 0.37, rtol=1e-14)


def test_spike_becomes_the_normalised_gaussian_and_wraps(obs):
    n, dv, fwhm, j = 64, 5.0, 23.548200450309494, 3          # sigma = 10 km/s exactly
    F = np.zeros((1, n))
    F[0, j] = 2.5
    out = obs.convolve_rows(F, dv, fwhm)[0]
    d = (np.arange(n) - j) * dv
    d = (d + n * dv / 2) % (n * dv) - n * dv / 2               # nearest image, by hand
    g = np.exp(-0.5 * (d / 10.0) ** 2)
    assert np.allclose(out, 2.5 * g / g.sum(), rtol=1e-12, atol=1e-300)
    assert out[(j - 4) % n] == pytest.approx(out[j + 4], rel=1e-12)      # symmetric across the wrap
    assert out[j + 2] / out[j] == pytest.approx(math.exp(-0.5), rel=1e-12)  # one sigma = 2 pixels away


def test_convolution_conserves_the_sum_and_fwhm_zero_copies(obs):
    rng = np.random.default_rng(1)
    F = rng.uniform(0, 1, (4, 37))
    out = obs.convolve_rows(F, 3.0, 11.0)
    assert np.allclose(out.sum(axis=1), F.sum(axis=1), rtol=1e-13)
    assert np.array_equal(obs.convolve_rows(F, 3.0, 0.0), F)
    # linear and shift-equivariant
    assert np.allclose(obs.convolve_rows(np.roll(F, 5, axis=1), 3.0, 11.0), np.roll(out, 5, axis=1), rtol=1e-13)


def test_fwhm_is_a_full_width_at_half_maximum(obs):
    n, dv = 401, 0.5
    F = np.zeros((1, n))
    F[0, 200] = 1.0
    out = obs.convolve_rows(F, dv, 20.0)[0]                    # half maximum 10 km/s = 20 pixels from the peak
    assert out[220] / out[200] == pytest.approx(0.5, rel=1e-12)


# ---------------------------------------------------------------- rebinning
def test_rebin_identity_pair_mean_and_bin_count(obs):
    rng = np.random.default_rng(2)
    F = rng.uniform(0, 1, (2, 12))
    assert np.allclose(obs.rebin_rows(F, 4.0, 4.0), F, rtol=1e-14)
    assert np.allclose(obs.rebin_rows(F, 4.0, 8.0), 0.5 * (F[:, 0::2] + F[:, 1::2]), rtol=1e-14)
    assert obs.n_bins(12, 4.0, 8.0) == 6 and obs.n_bins(12, 4.0, 9.0) == 5 and obs.n_bins(12, 4.0, 0.0) == 12
    assert np.array_equal(obs.rebin_rows(F, 4.0, 0.0), F)


def test_rebin_fractional_overlap_by_hand_and_oversampling(obs):
    F = np.array([[1.0, 3.0, 5.0, 7.0]])                       # dv = 2: pixels [0,2) [2,4) [4,6) [6,8)
    out = obs.rebin_rows(F, 2.0, 3.0)                          # bins [0,3) [3,6): floor(8/3) = 2 bins
    assert out.shape == (1, 2)
    assert out[0, 0] == pytest.approx((2 * 1.0 + 1 * 3.0) / 3.0, rel=1e-14)
    assert out[0, 1] == pytest.approx((1 * 3.0 + 2 * 5.0) / 3.0, rel=1e-14)
    fine = obs.rebin_rows(F, 2.0, 0.5)                         # bins smaller than pixels: piecewise constant
    assert np.allclose(fine[0], np.repeat(F[0], 4), rtol=1e-14)


def test_rebin_conserves_the_integral_when_bins_tile_the_box(obs):
    rng = np.random.default_rng(3)
    F = rng.uniform(0, 1, (3, 30))
    out = obs.rebin_rows(F, 2.0, 7.5)                          # V = 60 = 8 bins of 7.5
    assert out.shape[1] == 8
    assert np.allclose(out.sum(axis=1) * 7.5, F.sum(axis=1) * 2.0, rtol=1e-13)


def test_bin_width_from_angstrom_matches_the_papers_pair(obs):
    # "FWHM of ~3.63 A (~224 km/s)" for spectra at z ~ 3
    assert obs.bin_kms_from_angstrom(3.0, 3.63) == pytest.approx(224.0, rel=0.01)


# ---------------------------------------------------------------- noise
def test_noise_is_unit_draws_over_snr(obs):
    Fb = np.array([0.2, 0.9, 1.0])
    un = np.array([1.0, -2.0, 0.5], dtype=np.float32)
    assert np.allclose(obs.add_noise(Fb, 5.0, un), [0.4, 0.5, 1.1], rtol=1e-14)
    assert np.array_equal(obs.add_noise(Fb, 0.0, un), Fb)


# ---------------------------------------------------------------- flux PDF
def test_pdf_bins_of_the_paper(obs):
    # first bin -0.025 <= F < 0.025, 21 bins of 0.05
    F = np.array([0.0, 0.024, 0.026, 0.5, 0.974, 0.976, 1.0, 1.3, -0.4], dtype=np.float32)
    counts, pdf = obs.flux_pdf(F)
    expect = np.zeros(21, dtype=np.uint64)
    expect[0] = 3            # 0.0, 0.024, and -0.4 clamped (reading O4)
    expect[1] = 1            # 0.026
    expect[10] = 1           # 0.5 (bin centre)
    expect[19] = 1           # 0.974
    expect[20] = 3           # 0.976, 1.0, and 1.3 clamped
    assert np.array_equal(counts, expect)
    assert pdf.sum() * 0.05 == pytest.approx(1.0, rel=1e-14)
    assert counts.sum() == F.size


def test_pdf_of_uniform_fluxes_is_flat(obs):
    F = ((np.arange(200000) + 0.5) / 200000).astype(np.float32)       # uniform on (0,1)
    counts, pdf = obs.flux_pdf(F)
    assert np.allclose(pdf[1:20], 1.0, rtol=2e-3)                       # full-width bins
    assert pdf[0] == pytest.approx(0.5, rel=5e-3) and pdf[20] == pytest.approx(0.5, rel=5e-3)   # half bins


def _exact_bin(f32, n_bins=21, lo=(-1, 40), width=(1, 20)):
    """Bin of one fp32 flux by EXACT rational arithmetic against the paper's real edges (2b-1)/40."""
    from fractions import Fraction
    f = float(f32)
    if f != f:
        return 0
    if f in (float("inf"), float("-inf")):
        return n_bins - 1 if f > 0 else 0
    x, b = Fraction(f), 0
    while b + 1 < n_bins and x >= Fraction(*lo) + (b + 1) * Fraction(*width):
        b += 1
    return b


def test_pdf_edges_are_the_papers_real_edges(obs):
    """bins of width 0.05 starting at -0.025, i.e. real edges (2b-1)/40.  The oracle's edges (built
    from the doubles nearest -0.025 and 0.05) must sit within 2^-52 of them -- six orders of magnitude closer
    than any fp32 flux that is not the edge itself can come (>= 2^-32 away from a non-dyadic edge here) -- and the
    four edges an fp32 flux CAN equal, the dyadic 0.125, 0.375, 0.625, 0.875, must be exact."""
    from fractions import Fraction
    for b in range(0, 22):
        e = obs.flux_pdf_edge(b)
        exact = Fraction(2 * b - 1, 40)
        assert abs(Fraction(e) - exact) <= Fraction(1, 2 ** 52)
        f32 = Fraction(float(np.float32(float(exact))))                 # nearest fp32 to the real edge
        assert f32 == exact or abs(f32 - exact) >= Fraction(1, 2 ** 32)
    assert [obs.flux_pdf_edge(b) for b in (3, 8, 13, 18)] == [0.125, 0.375, 0.625, 0.875]


def test_pdf_decisions_at_every_edge_and_its_fp32_neighbours(obs):
    """Fluxes AT each of the 20 interior edges' nearest fp32 and one ulp either side, judged by exact rational
    comparison with the real edges (lower edge inclusive: "-0.025 <= F < 0.025"), plus values
    outside the range, infinities and NaN.  A bin decision taken in fp32 arithmetic fails this pin."""
    vals = []
    for b in range(1, 21):
        e = np.float32((2 * b - 1) / 40.0)
        vals += [np.nextafter(e, np.float32(-9)), e, np.nextafter(e, np.float32(9))]
    vals += [np.float32(x) for x in (-0.025, -0.0250001, 1.025, 1.0250001, -3.0, 7.0, 0.0, 1.0)]
    vals += [np.float32("inf"), np.float32("-inf"), np.float32("nan")]
    F = np.array(vals, dtype=np.float32)
    expect = np.zeros(21, dtype=np.uint64)
    for f in F:
        expect[_exact_bin(f)] += 1
    counts, pdf = obs.flux_pdf(F)
    assert np.array_equal(counts, expect)
    # each value on its own too (a compensating pair of errors cannot hide)
    for f in F:
        c, _ = obs.flux_pdf(np.array([f], dtype=np.float32))
        assert c[_exact_bin(f)] == 1, float(f)
    # the dyadic edges are inclusive lower edges
    for b, e in ((3, 0.125), (8, 0.375), (13, 0.625), (18, 0.875)):
        assert obs.flux_pdf(np.array([e], dtype=np.float32))[0][b] == 1
        assert obs.flux_pdf(np.array([np.nextafter(np.float32(e), np.float32(0))]))[0][b - 1] == 1


def test_pdf_general_bins_against_exact_rationals(obs):
    """Other (n_bins, f_lo, width): random fp32 fluxes, exact rational bins of the given doubles' real values --
    the oracle's fma-rounded edge can differ from the real one only for an F that equals the rounded edge."""
    from fractions import Fraction
    rng = np.random.default_rng(156)
    F = rng.uniform(-0.7, 1.7, 4000).astype(np.float32)
    for nb, lo, w in ((100, -0.5, 0.02), (40, 0.0, 0.025), (7, 0.1, 0.13)):
        expect = np.zeros(nb, dtype=np.uint64)
        for f in F:
            x, b = Fraction(float(f)), 0
            while b + 1 < nb and x >= Fraction(lo) + (b + 1) * Fraction(w):
                b += 1
            expect[b] += 1
        assert np.array_equal(obs.flux_pdf(F, nb, lo, w)[0], expect)


# ---------------------------------------------------------------- 1D power
def test_power_of_one_cosine_mode(obs):
    n, dv, m0, eps, fbar = 64, 3.0, 5, 0.2, 0.7
    i = np.arange(n)
    F = fbar * (1.0 + eps * np.cos(2 * np.pi * m0 * i / n + 0.3))
    P = obs.flux_power(F[None, :], dv, fbar)
    expect = np.zeros(n // 2 + 1)
    expect[m0] = (n * dv) * eps ** 2 / 4.0                     # |X|^2 = (eps N / 2)^2, times V / N^2
    assert np.allclose(P, expect, atol=1e-12)


def test_power_parseval_and_library_fft(obs):
    rng = np.random.default_rng(4)
    n, dv = 48, 2.5
    F = rng.uniform(0.1, 1.0, (5, n))
    fbar = F.mean()
    P = obs.flux_power(F, dv, fbar)
    d = F / fbar - 1.0
    X = np.fft.rfft(d, axis=1)
    assert np.allclose(P, (np.abs(X) ** 2).mean(axis=0) * dv / n, rtol=1e-11, atol=1e-14)
    # Parseval: sum over ALL N modes of |X|^2 = N sum d^2; modes 1..N/2-1 appear twice
    wts = np.full(n // 2 + 1, 2.0)
    wts[0] = wts[-1] = 1.0
    assert (P * wts).sum() == pytest.approx((d ** 2).sum(axis=1).mean() * dv, rel=1e-12)


def test_power_odd_length_and_mean_mode(obs):
    rng = np.random.default_rng(5)
    F = rng.uniform(0.1, 1.0, (2, 15))
    P = obs.flux_power(F, 1.0, 0.5)
    X = np.fft.rfft(F / 0.5 - 1.0, axis=1)
    assert P.shape == (8,)
    assert np.allclose(P, (np.abs(X) ** 2).mean(axis=0) / 15, rtol=1e-11)
