"""bench.py's one-line JSON contract (keys the driver and DESIGN.md section 8 rely on), on the small config."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                       cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    return json.loads(r.stdout.strip().splitlines()[-1])


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys():
    d = _run("--cfg", "1", "--steps", "3", "--warmup", "3", "--cpu-seconds", "1")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "clocks", "e2e", "gpu_launches"):
        assert k in d, k
    assert d["metric"] == "tau_pixel_pair_evals_per_s" and d["unit"] == "pair-evals/s" and d["dtype"] == "f32"
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and d["n_gpus"] == 1 and d["steps"] == 3
    assert d["config"]["workload"].startswith("cfg1_") and "model" not in d["config"]
    r = d["roofline"]
    assert r["bound"] == "alu" and 0 < r["frac"] < 1.05 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert 0.95 < r["peak_measured"] / r["peak"] < 1.02                  # 16 MUFU.EX2 / clk / SM, measured
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == d["unit"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 2 * 4 * 64 ** 3 and e["d2h_bytes_per_step"] == 4 * 64 ** 3
    assert e["value"] < 1.5 * d["value"]          # host copies are inside its timed region (config 1 is launch-bound: both legs within noise of each other)
    assert d["gpu_launches"] == 4 * 3                                     # gas, tau, normalise, flux per step
    assert d["value"] == pytest.approx(64.0 ** 4 / (d["ms_per_step"] * 1e-3), rel=1e-9)
    assert abs(d["mean_flux"] - 0.80) < 1e-6


@pytest.mark.gpu
def test_two_rank_bench_path_on_one_gpu():
    """The N > 1 path of bench.py (per-rank slabs of one taller grid, ONE global A through the sharded S4, barriers, max
    over ranks, rank 0 alone prints) with two gloo ranks time-slicing GPU 0: the code path, not a measurement."""
    env = dict(os.environ, LYA_BENCH_BACKEND="gloo", LYA_BENCH_ONE_DEVICE="1", MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29541", os.path.join(ROOT, "bench.py"),
                        "--gpus", "2", "--cfg", "1", "--steps", "3", "--warmup", "3"],
                       capture_output=True, text=True, cwd=ROOT, timeout=900, env=env)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                              # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["config"]["grid"] == [64, 64, 128]
    assert d["config"]["sightlines"] == 2 * 64 * 64 and "all-reduce" in d["config"]["parallelism"]
    assert d["value"] == pytest.approx(2 * 64.0 ** 4 / (d["ms_per_step"] * 1e-3), rel=1e-9)
    assert abs(d["mean_flux"] - 0.80) < 1e-6                            # the global A reaches the target over BOTH slabs
    assert d["e2e"]["value"] > 0 and "one global A" in d["e2e"]["note"]


def test_reference_arm_line():                                          # no GPU needed: the oracle on the host cores
    d = _run("--impl", "reference", "--cfg", "1", "--steps", "1", "--warmup", "0")
    assert d["impl"] == "reference" and d["metric"] == "tau_pixel_pair_evals_per_s" and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
