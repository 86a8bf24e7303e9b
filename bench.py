#!/usr/bin/env python
"""bench.py -- one JSON line for the Lya-forest hot path (S1 gas, S2+S3 tau, S4 normalisation, S5 flux).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg C] [--impl ours|reference]

A step is one pass of the whole hot path over one synthetic grid.  Default workload: the LARGEST single-GPU
configuration of BASELINE.json that this box can hold -- configs[4] (2048^3, 4.19M sightlines x 2048 px, processed
in 64-plane z-slabs with delta, v_pec and tau resident: 96 GiB of HBM, and 96 GiB of pinned host memory for the
e2e leg), else configs[3] (1024^3); `--cfg` picks any of the five.  `value` = tau pixel-pair evaluations per second
over the whole step, inputs resident in HBM; `e2e` = the same through lya_forest_host with pinned HOST buffers (H2D
of delta and v_pec, D2H of F inside the timed region).  N > 1 (torchrun): every rank owns its own seeded grid of
complete x-rows (weak scaling: slabs of one N-times-taller grid); the only exchange is S4's all-reduce of five
doubles per pass, in the resident leg and in the e2e leg alike (one GLOBAL A).
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from paper_1105_4747_b200 import inputs
from paper_1105_4747_b200.workloads import WORKLOADS, Workload

METRIC = "tau_pixel_pair_evals_per_s"
UNIT = "pair-evals/s"
SM_COUNT_B200, MUFU_PER_CLK_SM = 148, 16          # MUFU.EX2 results / clk / SM
# The tau pair loop sends one exponential in eight to the FMA pipe (rows of >= 128 pixels), so the
# MUFU pipe -- still the binding one for that instruction mix -- bounds it at 16 / (1 - 1/8) pairs per clock and SM.
TAU_FMA_EXP_FRACTION = 1.0 / 8.0
# dram__bytes_read.sum + dram__bytes_write.sum of ONE tau-kernel launch in this bench's launch shape, copied from the
# committed `ncu --set full` captures named beside each figure (NOT measured in this run: a number printed under a
# profiler is never a bench value, so the capture is a separate command).  Algorithmic traffic is 16 B per cell.
TAU_TRAFFIC = {
    2: (201.476864e6 + 35.543552e6, "profiles/r1_ncu_full_final.md"),
    3: (1.611410e9 + 0.504592e9, "profiles/r1_ncu_full_final.md"),
    4: (12.910775e9 + 4.285084e9, "profiles/r2_ncu_full_s1s5.md (addendum: the shipped kernel)"),
    5: (3.228292e9 + 1.036349e9, "profiles/r2_ncu_full_s1s5.md (addendum: the shipped kernel)"),   # one 64-plane slab = one launch
}


def default_cfg() -> int:
    """Largest single-GPU config this box holds: 5 needs ~105 GiB of HBM and, for the e2e leg, 96 GiB of pinned host
    memory; otherwise 4.  Both arms (ours / reference) call this, so they name the same workload."""
    try:
        import psutil
        world = int(os.environ.get("WORLD_SIZE", "1"))
        host_ok = psutil.virtual_memory().available >= (100 * world + 30) * 2 ** 30
    except Exception:
        host_ok = False
    gpu_ok = False
    if torch.cuda.is_available():
        free, total = torch.cuda.mem_get_info(int(os.environ.get("LOCAL_RANK", "0")))
        gpu_ok = free >= 120 * 2 ** 30
    return 5 if (host_ok and gpu_ok) else 4


def peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    REASONS = {0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x8: "hw_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake"}

    def __init__(self, local_rank: int):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.phase_samples, self.phase_reasons, self.phase = [], set(), False   # whole measurement phase (see summary)
        self._stop_evt, self.active, self.h = threading.Event(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = local_rank
            if vis:
                tok = vis.split(",")[local_rank].strip()
                idx = int(tok) if tok.isdigit() else local_rank
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def run(self):
        while self.h is not None and not self._stop_evt.is_set():
            try:
                before = self.active                    # an NVML query can take longer than a short timed region:
                mhz = float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                bits = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                why = {v for k, v in self.REASONS.items() if bits & k}
                if before or self.active:               # a query that overlaps the region counts
                    self.samples.append(mhz)
                    self.reasons |= why
                if self.phase:
                    self.phase_samples.append(mhz)
                    self.phase_reasons |= why
            except Exception:
                pass
            time.sleep(0.001)

    def stop(self):
        self._stop_evt.set()

    def summary(self, fallback_max: float) -> dict:
        # Samples of the timed region itself when it is long enough to hold a few NVML queries; otherwise those of
        # the whole measurement phase (timed region + the tau-variant and next-row kernel timings right after it, GPU
        # under load throughout).
        if len(self.samples) >= 3 or not self.phase_samples:
            smp, why, window = self.samples, self.reasons, "timed region"
        else:
            smp, why, window = self.phase_samples, self.reasons | self.phase_reasons, \
                "timed region + the kernel timings right after it (the timed region is shorter than three NVML queries)"
        return {"sm_mhz": statistics.median(smp) if smp else None,
                "sm_max_mhz": self.max_mhz or fallback_max, "reasons": sorted(why),
                "samples": len(smp), "window": window}


# ------------------------------------------------------------------------------------------ ours
def bench_ours(args) -> dict:
    import torch.distributed as dist
    from paper_1105_4747_b200 import lya

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # LYA_BENCH_BACKEND=gloo with LYA_BENCH_ONE_DEVICE=1 exists for ONE purpose: tests/test_bench_contract.py runs the
    # N > 1 code path (per-rank slabs, global A, barriers, max over ranks) with two ranks on a one-GPU box.  Its numbers
    # are not measurements (the ranks time-slice one GPU) and the line says so in config.parallelism.
    backend = os.environ.get("LYA_BENCH_BACKEND", "nccl")
    if os.environ.get("LYA_BENCH_ONE_DEVICE") == "1":
        local = 0
    if world > 1:
        if backend == "nccl":
            os.environ.setdefault("NCCL_DEBUG", "INFO")        # communicator lines stay on: the driver counts ranks
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    torch.cuda.set_device(local)
    if args.cfg is None:
        args.cfg = default_cfg()
        if world > 1:                                          # every rank must run the same workload
            c = torch.tensor([args.cfg], device="cuda")
            dist.all_reduce(c, op=dist.ReduceOp.MIN)
            args.cfg = int(c.item())
    w: Workload = WORKLOADS[args.cfg]
    n = w.n
    pk = peaks()

    # inputs: rank r owns planes of its own seeded slab (weak scaling: independent slabs of one N*n-plane grid;
    # complete x-rows, so S1-S3 and S5 need no exchange).  Config 5 (32 GiB per field) is generated and
    # processed in z-slabs: delta, v_pec and tau stay resident (96 GiB), n_HI / b exist for one slab at a time
    # and F overwrites tau.
    wl = w if world == 1 else Workload(**{**w.as_dict(), "axes": tuple(w.axes), "cfg": w.cfg + 100 * rank})
    slab_nz = 64 if w.cfg == 5 else n
    if w.cfg == 5:
        delta = torch.empty((n, n, n), dtype=torch.float32, device="cuda")
        vels = [torch.empty_like(delta)]
        for z0 in range(0, n, 32):
            f = inputs.make_fields(wl, device="cuda", z0=z0, z1=z0 + 32)
            delta[z0:z0 + 32] = f["delta"]
            vels[0][z0:z0 + 32] = f["v_pec"][w.axes[0]]
            del f
    else:
        fields = inputs.make_fields(wl, device="cuda")
        delta = fields["delta"]
        vels = [fields["v_pec"][ax] for ax in w.axes]
    p = lya.Params.from_workload(w)
    ctx = lya.Context(local)
    n_hi, b = (torch.empty((slab_nz, n, n), dtype=torch.float32, device="cuda") for _ in range(2))
    tau = torch.empty_like(delta)
    # per-sightline plain moments of tau, written by the tau kernels' epilogue: S4's first pass reads these 40 B per
    # sightline instead of tau (lya_tau_sightlines_opt row_moments / lya_normalize_mean_flux_rows)
    rowm = torch.empty((n * n, 5), dtype=torch.float64, device="cuda")
    flux = tau if w.cfg == 5 else torch.empty_like(delta)
    n_cells = delta.numel()
    n_slabs = n // slab_nz
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2

    ev = lambda: torch.cuda.Event(enable_timing=True)
    results = {}

    def step(timers=None):
        """S1 once, then S2-S5 per sightline axis (config 3 has three; the others one).  With slabs (config 5)
        S1 and S3 alternate per slab; the per-kernel event pairs of gas and tau bracket the FIRST slab's launch."""
        t = {"gas": [], "tau": [], "normalize": [], "flux": []} if timers is not None else None

        def timed(name, fn):
            if t is None:
                return fn()
            e0, e1 = ev(), ev()
            e0.record()
            r = fn()
            e1.record()
            t[name].append((e0, e1))
            return r

        for k, ax in enumerate(w.axes):
            for sl in range(n_slabs):
                z0, z1 = sl * slab_nz, (sl + 1) * slab_nz
                run = timed if sl == 0 else (lambda name, fn: fn())
                if k == 0 or n_slabs > 1:
                    run("gas", lambda: ctx.gas_from_density(p, delta[z0:z1], n_hi, b))
                # sightline index of the moments: axis 0 iz n + iy, axis 1 iz n + ix (slabs are whole planes); axis 2
                # needs the whole grid (one slab)
                run("tau", lambda: ctx.tau_sightlines_opt(p, ax, vels[k][z0:z1], n_hi=n_hi, b_kms=b, tau=tau[z0:z1],
                                                          row_moments=rowm[z0 * n:z1 * n]))
            if world == 1:
                A, f, it, _ = timed("normalize", lambda: ctx.normalize_mean_flux(tau, w.f_target, rel_tol=1e-7,
                                                                                 max_iter=60, row_moments=rowm))
                nst = ctx.last_normalize_stats()
            else:
                nst = {"row_pass": 1}
                A, f, it = timed("normalize", lambda: lya.normalize_mean_flux_sharded(
                    ctx, tau, w.f_target, n_cells * world, rel_tol=1e-7, row_moments=rowm, stats=nst))
            timed("flux", lambda: ctx.flux(tau, A, flux))
            results.update(A=A, f=f, passes=it, norm=nst)
        if timers is not None:
            timers.append(t)

    # the oracle's sample for the cpu_baseline leg: the first >= 65536 sightlines (whole planes), copied now
    nz_cpu = min(n, max(1, 65536 // n))
    cpu_rows = (delta[:nz_cpu].reshape(-1, n).cpu().numpy(), vels[0][:nz_cpu].reshape(-1, n).cpu().numpy())

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = ctx.launch_count
    timers, step_ev = [], []
    sampler.active = sampler.phase = True
    wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.zero_()                                   # L2 flush, outside the event-timed span
        s, e = ev(), ev()
        s.record()
        step(timers)
        e.record()
        step_ev.append((s, e))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    wall = time.perf_counter() - wall0
    sampler.active = False
    launches = ctx.launch_count - launches0

    step_ms = [s.elapsed_time(e) for s, e in step_ev]
    total_ms = sum(step_ms)
    if world > 1:
        tt = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    ms_per_step = total_ms / args.steps
    n_ax = len(w.axes)
    pairs_per_step = float(n) ** 4 * n_ax * world
    pix_per_step = float(n) ** 3 * n_ax * world

    # per-launch means (rank 0): gas and tau launches cover one slab (= the whole grid unless config 5)
    k_ms = {}
    for name in ("gas", "tau", "normalize", "flux"):
        spans = [e0.elapsed_time(e1) for t in timers for e0, e1 in t[name]]
        k_ms[name] = sum(spans) / len(spans)
    slab_cells = slab_nz * n * n

    # ---- the work-efficient tau variants on the same inputs (not part of `value`:
    # they evaluate fewer pairs, so they are reported as sightline pixels/s; outputs are bit-identical)
    tau_variants = None
    if not args.no_next:
        tau_variants = {}
        z1 = slab_nz
        ctx.gas_from_density(p, delta[:z1], n_hi, b)
        full = ctx.tau_sightlines(p, w.axes[0], n_hi, b, vels[0][:z1]).clone()      # the full sum of this slab
        for name, kw in (("fused_gas", dict(delta=delta[:z1])),
                         ("windowed", dict(n_hi=n_hi, b_kms=b, windowed=True)),
                         ("windowed_fused_gas", dict(delta=delta[:z1], windowed=True))):
            if "n_hi" in kw:
                ctx.gas_from_density(p, delta[:z1], n_hi, b)
            _, pairs_ev = ctx.tau_sightlines_opt(p, w.axes[0], vels[0][:z1], tau=tau[:z1], count_pairs=True, **kw)
            same = bool(torch.equal(tau[:z1], full))                                # measured, every pixel of the slab
            spans = []
            for _ in range(4):
                flush.zero_()
                e0, e1 = ev(), ev()
                e0.record()
                ctx.tau_sightlines_opt(p, w.axes[0], vels[0][:z1], tau=tau[:z1], **kw)
                e1.record()
                torch.cuda.synchronize()
                spans.append(e0.elapsed_time(e1))
            ms = sum(spans[1:]) / 3
            tau_variants[name] = {"ms": ms, "sightline_pixels_per_s": slab_nz * n * n / (ms * 1e-3),
                                  "pairs_evaluated": pairs_ev, "pairs_fraction_of_full": pairs_ev / (float(slab_nz) * n ** 3),
                                  "pair_evals_per_s": pairs_ev / (ms * 1e-3),
                                  "bit_identical_to_full_sum": same}
        del full

    # ---- the rows after F, timed per kernel on this workload's F; not part of `value`
    next_rows = None
    if not args.no_next and (n & (n - 1)) == 0:
        dv = lya.scalars(p, 0)["dv_kms"]
        # config 5 keeps F in tau's storage and the variants above overwrote its first slab: rebuild tau and F of the
        # first 256 planes (1.07e9 pixels, as many as the whole of config 4) and time the rows after F on those
        nr_z = n if w.cfg != 5 else 256
        if w.cfg == 5:
            for z0 in range(0, nr_z, slab_nz):
                ctx.gas_from_density(p, delta[z0:z0 + slab_nz], n_hi, b)
                ctx.tau_sightlines(p, w.axes[0], n_hi, b, vels[0][z0:z0 + slab_nz], tau[z0:z0 + slab_nz])
            tau_nr = tau[:nr_z]
            flux_nr = ctx.flux(tau_nr, results["A"])
        else:
            tau_nr, flux_nr = tau, flux
        nr_cells = flux_nr.numel()
        Frows = flux_nr.reshape(-1, n)
        bin_kms = lya.bin_kms_from_angstrom(w.z, 1.0375)                   # BOSS-like instrument
        nb = lya.lib().lya_instrument_bins(n, dv, lya.C.byref(lya.CInstrument(224.0, bin_kms, 5.0)))
        noise = torch.randn((Frows.shape[0], nb), device="cuda")
        obs_out = torch.empty_like(noise)

        def timed_ms(fn, reps=5):
            spans = []
            for _ in range(reps + 1):
                flush.zero_()
                e0, e1 = ev(), ev()
                e0.record()
                fn()
                e1.record()
                torch.cuda.synchronize()
                spans.append(e0.elapsed_time(e1))
            return sum(spans[1:]) / reps

        t_obs = timed_ms(lambda: ctx.observe_rows(Frows, dv, 224.0, bin_kms, 5.0, noise, obs_out))
        t_pdf = timed_ms(lambda: ctx.flux_pdf(flux_nr))
        t_pow = timed_ms(lambda: ctx.flux_power_rows(Frows, dv, results["f"]))
        t_fpdf = timed_ms(lambda: ctx.flux_with_pdf(tau_nr, results["A"], out=flux_nr))
        b_obs = 4 * nr_cells + 8 * obs_out.numel()
        row = lambda ms, nbytes, **kw: {"ms": ms, "bytes": int(nbytes), "gbs": nbytes / ms / 1e6,
                                        "frac_hbm": nbytes / ms / 1e6 / pk["hbm_gbs"], **kw}
        next_rows = {
            "on": f"{Frows.shape[0]} rows of {n} pixels" + (" (the first 256 planes)" if w.cfg == 5 else ""),
            "observe_rows": row(t_obs, b_obs, instrument="FWHM 224 km/s, 1.0375 A bins, S/N 5 (PAPER.md:130)", bins_per_row=int(nb)),
            "flux_pdf": row(t_pdf, 4 * nr_cells),
            "flux_with_pdf": row(t_fpdf, 8 * nr_cells, note="S5 and the flux PDF in one pass (replaces flux + flux_pdf: 12 B/pixel)"),
            "flux_power_rows": row(t_pow, 4 * nr_cells, note="one warp per two-row complex FFT for rows of 256 ... 2048 pixels (two register passes, rows prefetched by cp.async.bulk), Stockham radix-16/8 per CTA otherwise: bound by issue slots, FMA pipe and shared memory together, not by HBM")}
        del noise, obs_out
        if w.cfg == 5:
            del flux_nr, Frows, tau_nr
        # delta_b and v_x from a DM field (here: the workload's delta) -- one R2C, one k-space
        # kernel for both outputs, two C2R; the FFTs are cuFFT's
        if w.cfg <= 3 or args.fields:
            try:
                t_fld = timed_ms(lambda: ctx.fields_from_dm(delta, w.box_mpch, w.h, w.z, w.omega_m, 6.5,
                                                            want=("delta_b", "v_x")), reps=3)
                next_rows["fields_from_dm"] = {"outputs": "delta_b, v_x", "ms": t_fld,
                                               "kspace_kernel_bytes": int(3 * 8 * (n // 2 + 1) * n * n),
                                               "note": "3 cuFFT transforms + 1 k-space kernel (8 B in + 2 x 8 B out per mode)"}
            except lya.LyaError as exc:                   # cuFFT not installed on this box: the row is optional
                next_rows["fields_from_dm"] = {"unavailable": str(exc)}

    # ---- end to end through lya_forest_host: pinned host inputs, F read back, every step
    sampler.phase = False                               # host copies below: not "under load" for the clocks line
    e2e = None
    if not args.no_e2e:
        pinned = lambda src: torch.empty(src.shape, dtype=src.dtype, pin_memory=True).copy_(src)
        try:
            dh = pinned(delta)
            vh = [pinned(v) for v in vels]
            fh = torch.empty(dh.shape, dtype=dh.dtype, pin_memory=True)
        except RuntimeError as exc:                     # the host cannot pin 3 grids: say so instead of dying
            e2e = {"unavailable": "pinned host allocation failed: " + str(exc).splitlines()[0]}
            args.no_e2e = True
    if not args.no_e2e:
        if w.cfg == 5:                                  # lya_forest_host keeps its own tau + slab workspace
            del delta, vels, tau, flux, n_hi, b, rowm
            torch.cuda.empty_cache()
        n_pix_global = n_cells * world

        def e2e_step():
            for k, ax in enumerate(w.axes):
                if world == 1:
                    ctx.forest_host(p, ax, dh, vh[k], w.f_target, flux_h=fh)
                else:                                   # one GLOBAL A over all ranks' pixels
                    lya.forest_host_sharded(ctx, p, ax, dh, vh[k], w.f_target, n_pix_global, flux_h=fh)

        t0 = time.perf_counter()
        e2e_step()                                      # warm-up (allocates the workspace); also sizes the leg
        torch.cuda.synchronize()
        est = time.perf_counter() - t0
        if w.cfg != 5:
            e2e_step()
        # every step moves the whole grid over PCIe: at most ~40 s of them, never fewer than 2 (the count is reported)
        e2e_steps = max(2, min(args.steps, int(40.0 / max(est, 1e-3))))
        if world > 1:
            c = torch.tensor([e2e_steps], device="cuda")
            dist.all_reduce(c, op=dist.ReduceOp.MIN)
            e2e_steps = int(c.item())
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            tt = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        e2e = {"value": pairs_per_step * e2e_steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(2 * 4 * n_cells * n_ax), "d2h_bytes_per_step": int(4 * n_cells * n_ax),
               "ms_per_step": 1e3 * dt / e2e_steps, "steps": e2e_steps,
               "note": "lya_forest_host from pinned host buffers (S1 fused into S3 per axis pass), F copied back; "
                       "bytes are per rank" + ("; S4 all-reduced over ranks: one global A" if world > 1 else "")}
        del dh, vh, fh
    sampler.stop()

    clocks = sampler.summary(pk["sm_max_mhz"])
    mufu_measured = ctx.measure_mufu_peak()                                   # pure ex2 micro-kernel, this device
    torch.cuda.empty_cache()
    hbm_own = ctx.measure_hbm_peak(1 << 32)                                   # the library's own streaming copy, 4 GiB
    phi = TAU_FMA_EXP_FRACTION if n >= 128 else 0.0
    f_peak_mufu = MUFU_PER_CLK_SM * ctx.sm_count * pk["sm_max_mhz"] * 1e6     # MUFU.EX2 results/s at max SM clock
    f_peak = f_peak_mufu / (1.0 - phi)                                        # pair-evals/s the MUFU pipe allows this mix
    tau_rate = float(slab_cells) * n / (k_ms["tau"] * 1e-3)      # pairs of one launch / its duration
    hbm = pk["hbm_gbs"]
    gbs = lambda bytes_, ms: bytes_ / (ms * 1e-3) / 1e9
    passes, nst = results["passes"], results["norm"]
    # S4's bytes: passes over all of tau (the A = 0 one reads the tau kernels' 40 B per sightline instead), plus the
    # subsample passes of the nested iteration (n_sub pixels each)
    norm_bytes = 4 * n_cells * (nst["tau_passes"] - nst["row_pass"]) + 40 * n * n * nst["row_pass"] \
        + 4 * nst["n_sub"] * nst["sub_passes"]
    out = {
        "metric": METRIC, "value": pairs_per_step / (ms_per_step * 1e-3), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "grid": [n, n, n * world], "sightlines": n * n * world * n_ax,
                   "pixels_per_sightline": n, "axes": list(w.axes), "f_target": w.f_target, "slab_nz": slab_nz,
                   "l2": "256 MiB memset between steps (outside the event spans); working set %d MiB" %
                         (6 * 4 * n_cells >> 20),
                   "parallelism": ("z-slabs per rank; S4 all-reduce of 5 doubles per pass"
                                   + ("" if backend == "nccl" else f" [TEST RUN over {backend}: ranks may share a GPU, not a measurement]"))
                   if world > 1 else "1 GPU"},
        "sightline_pixels_per_s": pix_per_step / (ms_per_step * 1e-3),
        "tau_kernel_pixels_per_s": float(slab_cells) / (k_ms["tau"] * 1e-3),
        "A": results["A"], "mean_flux": results["f"], "normalize_passes": passes,
        "kernel_ms": k_ms, "wall_s_timed_region_incl_flush": wall,
        "roofline": {"bound": "alu", "kernel": "tau_kernel", "achieved": tau_rate / 1e9, "peak": f_peak / 1e9,
                     "unit": "Gpair-evals/s", "frac": tau_rate / f_peak,
                     "traffic": TAU_TRAFFIC[w.cfg][0] if w.cfg in TAU_TRAFFIC else None,
                     "traffic_src": ("ncu dram__bytes_read.sum + dram__bytes_write.sum of one launch, copied from "
                                     + TAU_TRAFFIC[w.cfg][1] + " (a separate run under ncu, not this one)")
                                    if w.cfg in TAU_TRAFFIC else None,
                     "traffic_algorithmic": 16 * slab_cells, "launch": "%d planes of %d x %d" % (slab_nz, n, n),
                     "peak_measured": mufu_measured / (1.0 - phi) / 1e9,
                     "frac_of_measured_peak": tau_rate * (1.0 - phi) / mufu_measured,
                     "peak_mufu_only": f_peak_mufu / 1e9, "frac_of_mufu_only_peak": tau_rate / f_peak_mufu,
                     "fma_pipe_exp_fraction": phi,
                     "peak_def": "16 MUFU.EX2/clk/SM x %d SMs x %.0f MHz (max SM clock, %s) / (1 - %g): %g of the "
                                 "exponentials run as a packed polynomial on the FMA pipe, the MUFU pipe stays the binding "
                                 "one (DESIGN.md section 6); peak_mufu_only is the figure without that offload" %
                                 (ctx.sm_count, pk["sm_max_mhz"], pk["src"], phi, phi),
                     "frac_at_measured_clock": (tau_rate * (1.0 - phi) / (MUFU_PER_CLK_SM * ctx.sm_count * clocks["sm_mhz"] * 1e6))
                     if clocks["sm_mhz"] else None},
        "roofline_hbm": {
            "peak_gbs": hbm, "peak_src": pk["src"] + " (MEASURED_PEAKS.json: torch copy_)" if pk["src"] == "measured" else pk["src"],
            "own_copy_gbs": hbm_own, "own_copy_def": "lya_measure_hbm_peak: 128-bit streaming copy kernel, 4 GiB of traffic, best of 5",
            "frac_def": "algorithmic bytes / event time / peak_gbs; a frac slightly above 1 means the 1:1 streaming "
                        "pattern beats the torch copy_ the driver measured -- compare with own_copy_gbs",
            "gas": {"bytes": 12 * slab_cells, "gbs": gbs(12 * slab_cells, k_ms["gas"]), "frac": gbs(12 * slab_cells, k_ms["gas"]) / hbm},
            "normalize": {"bytes": norm_bytes, "passes": nst,
                          "passes_def": "nested iteration: the A = 0 pass reads the tau kernels' per-sightline moments (40 B per "
                                        "sightline), sub_passes read the n_sub-pixel subsample, the other tau_passes all of tau "
                                        "(4 B per pixel)",
                          "gbs": gbs(norm_bytes, k_ms["normalize"]), "frac": gbs(norm_bytes, k_ms["normalize"]) / hbm},
            "flux": {"bytes": 8 * n_cells, "gbs": gbs(8 * n_cells, k_ms["flux"]), "frac": gbs(8 * n_cells, k_ms["flux"]) / hbm}},
        "clocks": clocks, "e2e": e2e, "tau_variants": tau_variants, "next_rows": next_rows, "gpu_launches": int(launches), "sm_count": ctx.sm_count,
    }
    if rank == 0 and world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(w, cpu_rows[0], cpu_rows[1], budget_s=args.cpu_seconds)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return out if rank == 0 else {}


# ------------------------------------------------------------------------------------------ oracle legs
def _oracle_sample(orc, w, d_rows, v_rows):
    """The oracle's whole path (S1..S5, plain mode: one exp per pair) on a set of sightlines."""
    po = orc.Params.from_workload(w)
    _, n_ref, b_ref = orc.gas_from_density(po, d_rows)
    tau = orc.tau_rows(po, n_ref, b_ref, v_rows, mode=0)
    A, _, _ = orc.normalize_mean_flux(tau, w.f_target)
    orc.flux(tau, A)
    return A


def _calibrated_rows(orc, w, d, v, seconds):
    n = w.n
    probe = min(64, d.shape[0])
    t0 = time.perf_counter()
    _oracle_sample(orc, w, d[:probe], v[:probe])
    rate = probe / max(time.perf_counter() - t0, 1e-4)                       # sightlines / s
    return int(max(probe, min(d.shape[0], rate * seconds)))


def cpu_baseline(w, d, vv, budget_s=12.0) -> dict:
    """d, vv: [rows, n] numpy arrays of delta and v_pec (the first planes of the bench's own fields)."""
    from oracle import lya_oracle as orc
    n = w.n
    rows = _calibrated_rows(orc, w, d, vv, budget_s)
    t0 = time.perf_counter()
    _oracle_sample(orc, w, d[:rows], vv[:rows])
    dt = time.perf_counter() - t0
    rate = rows * float(n) ** 2 / dt
    return {"value": rate, "unit": UNIT, "cores": orc.threads(), "kind": "oracle",
            "sample": f"first {rows} of {n * n} sightlines of {w.name}, whole path S1..S5 in double, "
                      f"plain mode, {dt:.1f} s",
            "cpu_model": _cpu_model(),
            "extrapolated_full_grid_s": float(n) ** 4 * len(w.axes) / rate}     # labelled as an extrapolation


def _cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def bench_reference(args) -> dict:
    if int(os.environ.get("RANK", "0")) != 0:
        return {}
    from oracle import lya_oracle as orc
    if args.cfg is None:
        args.cfg = default_cfg()
    w = WORKLOADS[args.cfg]
    n = w.n
    # the same seeded fields as our arm, only the planes the sample needs (generated on the CPU)
    nz_need = max(1, min(8, 2048 // n))
    f = inputs.make_fields(w, device="cpu", z0=0, z1=nz_need)
    d = f["delta"].reshape(-1, n).numpy()
    v = f["v_pec"][w.axes[0]].reshape(-1, n).numpy()
    rows = _calibrated_rows(orc, w, d, v, seconds=1.5)
    for _ in range(min(args.warmup, 1)):
        _oracle_sample(orc, w, d[:rows], v[:rows])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_sample(orc, w, d[:rows], v[:rows])
    dt = time.perf_counter() - t0
    val = rows * float(n) ** 2 * args.steps / dt
    sample = f"{rows} sightlines (first planes) of {w.name} per step, whole path S1..S5 in double, plain mode"
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": orc.threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=None, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json configs[cfg-1]; default: 5 if this box holds it (HBM and pinned host memory), else 4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--fields", action="store_true", help="time lya_fields_from_dm on config 4 too (17 GB of workspace)")
    ap.add_argument("--no-next", action="store_true", help="skip the per-kernel timing of the rows after F")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    args = ap.parse_args()
    out = bench_reference(args) if args.impl == "reference" else bench_ours(args)
    if out:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
