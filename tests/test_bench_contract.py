"""bench.py's contract that can be checked without a GPU: the reference arm (the oracle on the host cores) prints one
JSON line with the keys the driver reads, the byte accounting matches DESIGN.md section 6, and the product arm does not
fall back to anything when there is no CUDA device."""
import json
import os
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_algorithmic_bytes_per_cell():
    # fused kernel: h, g read + written, f read + written, phi, T, u
    assert bench.fused_kernel_values_per_cell("lb_d3q7") * 8 == 1056
    assert bench.fused_kernel_values_per_cell("lb_d3q15") * 8 == 1184
    assert bench.fused_kernel_values_per_cell("lb_d3q19") * 8 == 1248
    assert bench.fused_kernel_values_per_cell("lb_d3q27") * 8 == 1376
    assert bench.fused_kernel_values_per_cell("rk2") * 8 == 936
    # whole step on the Runge-Kutta paths of the benchmark fluid (kappa_H = kappa_L: stage 1 inside the fused kernel)
    assert bench.step_values_per_cell("rk2") * 8 == 936 + 8 + 56
    assert bench.step_values_per_cell("rk4") * 8 == 936 + 16 + 72 + 72 + 56
    assert bench.step_values_per_cell("lb_d3q7") * 8 == 1056
    assert bench.step_values_per_cell("lb_d3q7", 19) * 8 == 928         # D3Q19 hydrodynamic lattice: 16 values less


def test_benchmark_fluid_has_equal_conductivities():
    import workloads as W
    assert W.BENCH_FLUID["kappa_H"] == W.BENCH_FLUID["kappa_L"]     # what step_values_per_cell assumes


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1",
                          "--ref-size", "24"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference"
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in line, key
    assert line["unit"] == "MLUPS" and line["value"] > 0 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["vs_baseline"] is None


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the behaviour without a CUDA device")
def test_product_arm_fails_loudly_without_a_gpu():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--size", "16", "--steps", "1", "--warmup", "1", "--no-cpu",
                          "--no-e2e"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode != 0
    assert "MLUPS" not in out.stdout          # no number from any fallback


def test_variants_cover_baseline_configs4_and_traffic_has_provenance():
    """The default line carries short device-timed runs of the other rows of BASELINE configs[4] (>= 7 entries: D3Q15/19/27,
    RK2, RK4, AA at 400^3 fp64, fp32 at 512^3, D3Q7 at 256^3); every ncu traffic figure names its commit and command."""
    assert len(bench.VARIANTS) >= 7
    got = {(v[0], v[1], v[2]) for v in bench.VARIANTS}
    for need in ((400, "lb_d3q15", "f64"), (400, "lb_d3q19", "f64"), (400, "lb_d3q27", "f64"), (400, "rk2", "f64"),
                 (400, "rk4", "f64"), (512, "lb_d3q7", "f32"), (256, "lb_d3q7", "f64")):
        assert need in got
    assert isinstance(bench.recorded_traffic("lb_d3q7_f64_400"), int)
    table = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    for key, entry in table.items():
        if key.startswith("_"):
            continue
        assert entry["commit"] and entry["command"].startswith("ncu ") and os.path.exists(os.path.join(ROOT, entry["profile"]))
