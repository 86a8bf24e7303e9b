"""N > 1 path on CPU (gloo, world_size 2): the sharded normalisation of DESIGN.md "Multi-GPU".

Each rank owns half of the pixels; per pass the ranks all-reduce (sum exp(-A tau), sum tau exp(-A tau)) -- two
doubles -- and apply the library's host-side scalar update lya_root_update, so every rank must end with the
same A, equal to the oracle's bisection over ALL pixels.  The per-rank partial sums, which the product takes
from the CUDA kernel behind lya_flux_partial_sums, are stood in for here by numpy (test-only) because this
container has no GPU; everything else (init, all-reduce, update, stopping rule) is the product's code.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, f_target: float, out_path: str, moments: bool = False):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1105_4747_b200 import lya
    rng = np.random.default_rng(4747)                          # same stream on both ranks, split below
    tau_all = rng.lognormal(mean=-1.0, sigma=1.2, size=200_003).astype(np.float32)
    lo, hi = (0, 120_000) if rank == 0 else (120_000, tau_all.size)   # uneven shards on purpose
    tau = tau_all[lo:hi].astype(np.float64)

    def partial_sums(a):
        e = np.exp(-a * tau)
        if moments:                                            # the five tilted moments of lya_flux_moment_sums
            return [float((tau ** k * e).sum()) for k in range(5)]
        return [float(e.sum())], [float((tau * e).sum())]

    A, f, iters = lya.normalize_mean_flux_sharded(None, None, f_target, tau_all.size, rel_tol=1e-10,
                                                  partial_sums=partial_sums)
    got = torch.tensor([A, f, float(iters)], dtype=torch.float64)
    gathered = [torch.zeros_like(got) for _ in range(world)]
    dist.all_gather(gathered, got)
    if rank == 0:
        np.save(out_path, np.stack([g.numpy() for g in gathered]))
    dist.destroy_process_group()


@pytest.mark.parametrize("f_target,moments", [(0.80, False), (0.35, False), (0.80, True), (0.35, True)])
def test_sharded_normalisation_two_ranks_gloo(tmp_path, oracle, f_target, moments):
    out = str(tmp_path / "res.npy")
    mp.spawn(_worker, args=(2, _free_port(), f_target, out, moments), nprocs=2, join=True)
    res = np.load(out)
    assert np.array_equal(res[0], res[1]), "ranks disagree on (A, <F>, passes)"
    A, f, iters = res[0]
    rng = np.random.default_rng(4747)
    tau_all = rng.lognormal(mean=-1.0, sigma=1.2, size=200_003).astype(np.float32).astype(np.float64)
    A_ref, f_ref, _ = oracle.normalize_mean_flux(tau_all, f_target)
    assert abs(A / A_ref - 1.0) < 1e-8
    assert abs(f - f_target) < 1e-9 and iters <= (6 if moments else 20)


def _nested_worker(rank: int, world: int, port: int, f_target: float, out_path: str):
    """The nested iteration of normalize_mean_flux_sharded (A = 0 pass, subsample passes, then passes over all of
    tau) with numpy standing in for lya_flux_moment_sums_sub: every `every`-th chunk of 1024 pixels of the local tau."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1105_4747_b200 import lya
    rng = np.random.default_rng(4748)
    tau_all = rng.lognormal(mean=-0.6, sigma=2.2, size=400_000).astype(np.float32)     # heavy tail: max ~ 1e4 x median
    lo, hi = (0, 150_000) if rank == 0 else (150_000, tau_all.size)
    tau = tau_all[lo:hi].astype(np.float64)
    calls = []

    def kernel_sums(a, every):
        t = tau if every <= 1 else np.concatenate([tau[c: c + 1024] for c in range(0, tau.size, 1024 * every)])
        e = np.exp(-a * t)
        calls.append(every)
        return [float((t ** k * e).sum()) for k in range(5)], int(t.size)

    stats = {}
    A, f, passes = lya.normalize_mean_flux_sharded(None, None, f_target, tau_all.size, rel_tol=1e-9, kernel_sums=kernel_sums,
                                                   sub_every=8, sub_min_pix=0, stats=stats)
    got = torch.tensor([A, f, float(passes), float(stats["sub_passes"]), float(sum(1 for c in calls if c <= 1))], dtype=torch.float64)
    gathered = [torch.zeros_like(got) for _ in range(world)]
    dist.all_gather(gathered, got)
    if rank == 0:
        np.save(out_path, np.stack([g.numpy() for g in gathered]))
    dist.destroy_process_group()


@pytest.mark.parametrize("f_target", [0.80, 0.35])
def test_sharded_nested_iteration_two_ranks_gloo(tmp_path, oracle, f_target):
    out = str(tmp_path / "res.npy")
    mp.spawn(_nested_worker, args=(2, _free_port(), f_target, out), nprocs=2, join=True)
    res = np.load(out)
    assert np.array_equal(res[0], res[1]), "ranks disagree"
    A, f, passes, sub_passes, full_calls = res[0]
    rng = np.random.default_rng(4748)
    tau_all = rng.lognormal(mean=-0.6, sigma=2.2, size=400_000).astype(np.float32).astype(np.float64)
    A_ref, _, _ = oracle.normalize_mean_flux(tau_all, f_target)
    assert abs(A / A_ref - 1.0) < 1e-8 and abs(f - f_target) < 1e-9
    # the subsample did the climbing: the A = 0 pass plus at most two passes over all of tau
    assert sub_passes >= 2 and passes == full_calls <= 3


def test_sharded_weak_scaling_slabs_are_independent_problems():
    """bench.py's N > 1 layout: rank r generates ITS slab from (seed + 100 r): no rank needs another's cells."""
    from paper_1105_4747_b200 import inputs
    from paper_1105_4747_b200.workloads import WORKLOADS, Workload, scaled
    w = scaled(WORKLOADS[1], 32)
    w1 = Workload(**{**w.as_dict(), "axes": tuple(w.axes), "cfg": w.cfg + 100})
    a = inputs.make_fields(w, device="cpu", z0=0, z1=4)["delta"]
    b = inputs.make_fields(w1, device="cpu", z0=0, z1=4)["delta"]
    assert a.shape == b.shape == (4, 32, 32) and not torch.equal(a, b)
