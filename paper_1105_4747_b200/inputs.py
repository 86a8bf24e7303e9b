"""Seeded synthetic input fields (delta, v_pec) for the workloads of `workloads.py`.

This module is the ONLY code shared by the CUDA path's tests/bench and the oracle's
tests.  It holds none of the method's arithmetic (no Eq.4/5/6 of PAPER.md): it draws
counter-based white noise, smooths it, and applies the lognormal map that
BASELINE.json's configs prescribe for the *inputs*:

    g      = Gaussian field: Philox4x32-10 white noise, Gaussian-smoothed at R cells,
             rescaled to rms sigma_g by the ANALYTIC factor 1/(sum w^2)^(3/2)
    delta  = exp(g - sigma_g^2/2) - 1                      (stored fp32)
    v_pec  = sigma_v * (independent smoothed unit field)   (stored fp32, km/s)

These stand in for the paper's rank-ordered, hydro-calibrated delta_b and
its linear-theory velocity field (Eq.3), which need inputs not in the
container.

Determinism: noise for plane iz of field `fid` depends only on (seed, fid, iz, cell), so
any z-slab can be generated on its own (needed for the 2048^3 slab path), on the CPU or
on the GPU (torch ops only; the integer part is bit-identical on both, the Box-Muller
transcendental may differ in the last ulp between devices - every test hands the SAME
arrays to both sides, so that does not matter).
"""
from __future__ import annotations

import math

import torch

from .workloads import Workload

FIELD_G, FIELD_VX, FIELD_VY, FIELD_VZ = 0, 1, 2, 3
_HALO = 8                                   # smoothing kernel half-width [cells] (k = -8..8)

_M0, _M1 = 0xD2511F53, 0xCD9E8D57           # Philox4x32 multipliers
_W0, _W1 = 0x9E3779B9, 0xBB67AE85           # Philox4x32 Weyl key increments
_MASK = 0xFFFFFFFF


def _mulhilo(a: int, b: torch.Tensor):
    """32x32 -> (hi, lo) with operands held in int64 (the wrapped product keeps all 64 bits)."""
    p = b * a
    return (p >> 32) & _MASK, p & _MASK


def philox4x32(c0, c1, c2, c3, k0: int, k1: int):
    """Philox4x32-10 (Salmon et al. 2011). Counters: int64 tensors holding uint32 values."""
    for _ in range(10):
        hi0, lo0 = _mulhilo(_M0, c0)
        hi1, lo1 = _mulhilo(_M1, c2)
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & _MASK, lo1, (hi0 ^ c3 ^ k1) & _MASK, lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def white_noise_planes(seed: int, fid: int, izs, n: int, device) -> torch.Tensor:
    """N(0,1) white noise for the z-planes `izs` (a sequence of plane indices), float64 [len(izs), n, n], all planes
    in one batch of elementwise launches.  Key = (seed, fid), counter = (cell/4, iz): plane iz depends on nothing
    but (seed, fid, iz)."""
    m = (n * n + 3) // 4
    idx = torch.arange(m, dtype=torch.int64, device=device).unsqueeze(0)                      # [1, m]
    zz = (torch.as_tensor(list(izs), dtype=torch.int64, device=device) & _MASK).unsqueeze(1)  # [P, 1]
    c0, c1 = (idx & _MASK).expand(zz.shape[0], m), (idx >> 32).expand(zz.shape[0], m)
    r = philox4x32(c0, c1, zz.expand(-1, m), torch.zeros_like(c0),
                   seed & _MASK, ((seed >> 32) ^ (fid * 0x9E3779B1)) & _MASK)
    u = [(x.to(torch.float64) + 0.5) * (1.0 / 4294967296.0) for x in r]
    del r
    # Box-Muller on (u0,u1) and (u2,u3): four normals per counter
    r01 = torch.sqrt(-2.0 * torch.log(u[0]))
    r23 = torch.sqrt(-2.0 * torch.log(u[2]))
    t01 = (2.0 * math.pi) * u[1]
    t23 = (2.0 * math.pi) * u[3]
    del u
    g = torch.stack([r01 * torch.cos(t01), r01 * torch.sin(t01),
                     r23 * torch.cos(t23), r23 * torch.sin(t23)], dim=2).reshape(zz.shape[0], -1)
    return g[:, : n * n].reshape(zz.shape[0], n, n)


def white_noise_plane(seed: int, fid: int, iz: int, n: int, device) -> torch.Tensor:
    """One plane of white_noise_planes: float64 [n, n]."""
    return white_noise_planes(seed, fid, [iz], n, device)[0]


def smoothing_weights(r_cells: float) -> torch.Tensor:
    k = torch.arange(-_HALO, _HALO + 1, dtype=torch.float64)
    w = torch.exp(-0.5 * (k / r_cells) ** 2)
    return w / w.sum()


def _smooth_periodic(x: torch.Tensor, w: torch.Tensor, dim: int) -> torch.Tensor:
    out = torch.zeros_like(x)
    for t in range(2 * _HALO + 1):
        out += float(w[t]) * torch.roll(x, shifts=t - _HALO, dims=dim)
    return out


def unit_gaussian_field(seed: int, fid: int, n: int, r_cells: float, device="cpu",
                        z0: int = 0, z1: int | None = None, chunk: int = 32) -> torch.Tensor:
    """Smoothed periodic Gaussian field of (analytic) unit variance, planes z0..z1-1, float64."""
    z1 = n if z1 is None else z1
    w = smoothing_weights(r_cells)
    norm = 1.0 / float((w * w).sum()) ** 1.5
    out = torch.empty((z1 - z0, n, n), dtype=torch.float64, device=device)
    for c0 in range(z0, z1, chunk):
        c1 = min(c0 + chunk, z1)
        stack = white_noise_planes(seed, fid, [iz % n for iz in range(c0 - _HALO, c1 + _HALO)], n, device)
        stack = _smooth_periodic(_smooth_periodic(stack, w, 2), w, 1)  # along x, then y: [c1-c0+2H, n, n]
        acc = torch.zeros((c1 - c0, n, n), dtype=torch.float64, device=device)
        for t in range(2 * _HALO + 1):
            # out[z] = sum_t w[t] * x[z - (t - H)]  (same convention as torch.roll above)
            acc += float(w[t]) * stack[2 * _HALO - t: 2 * _HALO - t + (c1 - c0)]
        out[c0 - z0: c1 - z0] = acc * norm
    return out


def make_fields(w: Workload, device="cpu", z0: int = 0, z1: int | None = None,
                axes=None) -> dict:
    """delta [nz,n,n] fp32 and v_pec per requested axis (dict axis -> fp32 [nz,n,n], km/s)."""
    axes = tuple(w.axes) if axes is None else tuple(axes)
    g = unit_gaussian_field(w.seed, FIELD_G, w.n, w.smooth_r, device, z0, z1) * w.sigma_g
    delta = torch.expm1(g - 0.5 * w.sigma_g ** 2).to(torch.float32)
    del g
    v = {}
    for ax in axes:
        u = unit_gaussian_field(w.seed, FIELD_VX + ax, w.n, w.smooth_r, device, z0, z1)
        v[ax] = (u * w.sigma_v).to(torch.float32)
    return {"delta": delta.contiguous(), "v_pec": v}
