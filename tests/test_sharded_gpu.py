"""N > 1 path with the KERNELS in the loop, on one GPU.

Two processes share cuda:0 (gloo for the exchange, so no rank's kernel ever waits for another rank's kernel: the
all-reduce is a host-side sum of five doubles).  Each rank owns a z-slab of complete x-rows of ONE seeded grid --
uneven on purpose -- and runs the product path of a sharded run:

    lya_gas_from_density -> lya_tau_sightlines_opt(row_moments) on its slab
    per pass: lya_row_moment_sums (A = 0) / lya_flux_moment_sums -> all-reduce -> lya_root_update_moments
    lya_flux with the global A

and, second, the same from HOST buffers (lya_forest_host_begin / _moment_sums / _finish: bench.py's N > 1 e2e leg).
Both ranks must end with the same A, equal to the single-process A of the whole grid to 1e-9 and to the oracle's own
A (oracle tau over ALL pixels) to the north_star's 1e-5; F of each slab against the oracle's F.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1105_4747_b200 import inputs
from paper_1105_4747_b200.workloads import WORKLOADS, scaled

pytestmark = pytest.mark.gpu

N = 96
SPLIT = 40            # rank 0: planes [0, 40), rank 1: planes [40, 96)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1105_4747_b200 import lya
    torch.cuda.set_device(0)
    w = scaled(WORKLOADS[2], N)
    z0, z1 = (0, SPLIT) if rank == 0 else (SPLIT, N)
    f = inputs.make_fields(w, device="cpu", z0=z0, z1=z1)          # the generator is slab-local by construction
    dh, vh = f["delta"].contiguous(), f["v_pec"][0].contiguous()
    delta, v = dh.cuda(), vh.cuda()
    p = lya.Params.from_workload(w)
    ctx = lya.Context(0)
    nzl = z1 - z0

    # (1) device-resident shard
    n_hi, b = ctx.gas_from_density(p, delta)
    rowm = torch.empty((nzl * N, 5), dtype=torch.float64, device="cuda")
    tau = ctx.tau_sightlines_opt(p, 0, v, n_hi=n_hi, b_kms=b, nz_local=nzl, row_moments=rowm)
    A, fa, it = lya.normalize_mean_flux_sharded(ctx, tau, w.f_target, N ** 3, rel_tol=1e-9, row_moments=rowm)
    F = ctx.flux(tau, A)
    # (2) the same shard from host buffers (global A again)
    dp, vp = dh.pin_memory(), vh.pin_memory()
    tau_h, flux_h = torch.empty_like(dp).pin_memory(), torch.empty_like(dp).pin_memory()
    p_loc = lya.Params(**{**p.__dict__, "nz": nzl})               # lya_forest_host_begin takes the LOCAL grid
    A2, fa2, it2 = lya.forest_host_sharded(ctx, p_loc, 0, dp, vp, w.f_target, N ** 3, rel_tol=1e-9, slab_nz=16,
                                           tau_h=tau_h, flux_h=flux_h)
    torch.cuda.synchronize()
    assert torch.equal(tau_h, tau.cpu())
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), A=A, A2=A2, it=it, it2=it2, F=F.cpu().numpy(),
             F2=flux_h.numpy(), launches=ctx.launch_count)
    ctx.close()
    dist.destroy_process_group()


def test_two_ranks_share_one_global_A_through_the_kernels(tmp_path, oracle):
    from paper_1105_4747_b200 import lya
    mp.spawn(_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (np.load(tmp_path / f"rank{r}.npz") for r in (0, 1))
    assert float(r0["A"]) == float(r1["A"]) and float(r0["A2"]) == float(r1["A2"]), "ranks disagree on A"
    assert int(r0["launches"]) > 0 and int(r1["launches"]) > 0
    A = float(r0["A"])

    # single process, whole grid, device-side loop
    w = scaled(WORKLOADS[2], N)
    f = inputs.make_fields(w, device="cpu")
    p = lya.Params.from_workload(w)
    ctx = lya.Context(0)
    n_hi, b = ctx.gas_from_density(p, f["delta"].cuda())
    tau = ctx.tau_sightlines(p, 0, n_hi, b, f["v_pec"][0].cuda())
    A1, _, _, _ = ctx.normalize_mean_flux(tau, w.f_target, rel_tol=1e-9)
    ctx.close()
    assert abs(A / A1 - 1.0) < 1e-9 and abs(float(r0["A2"]) / A1 - 1.0) < 1e-9

    # the oracle over all pixels (its own tau), then F per slab
    ref = oracle.run_path(oracle.Params.from_workload(w), 0, f["delta"].numpy(), f["v_pec"][0].numpy(), w.f_target)
    assert abs(A / ref["A"] - 1.0) < 1e-5
    F_all = np.concatenate([r0["F"], r1["F"]], axis=0)
    F2_all = np.concatenate([r0["F2"], r1["F2"]], axis=0)
    assert np.abs(F_all - ref["flux"]).max() < 1e-5 and np.abs(F2_all - ref["flux"]).max() < 1e-5
