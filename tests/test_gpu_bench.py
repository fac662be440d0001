"""bench.py's JSON line (`-m gpu`): the contract keys of the task, on a small population so that it runs in seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_has_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--particles", "512", "--steps", "2", "--warmup", "3",
                          "--no-cpu-baseline"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "e2e", "gpu_launches", "clocks"):
        assert k in line, k
    assert line["n_gpus"] == 1 and line["steps"] == 2 and line["warmup"] == 3 and line["higher_is_better"] is True
    assert "workload" in line["config"] and line["config"]["workload"].startswith("c3")
    assert line["value"] > 0 and line["gpu_launches"] > 0 and line["vs_baseline"] is None
    # value counts evaluated (particle, bin) pairs: never more than the nominal rate
    assert line["value"] <= line["nominal_particle_bin_per_s"] * (1 + 1e-12) and 0 < line["evaluated_fraction"] <= 1
    r = line["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "frac_pipe_fma", "frac_model"):
        assert k in r, k
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and 0 < r["frac"] < 1 and r["frac"] == r["frac_pipe_fma"]
    assert r["frac"] == pytest.approx(r["achieved"] / r["peak"], rel=1e-9)
    e = line["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 512 * 72 and e["d2h_bytes_per_step"] == 512 * 72
    for k in ("adaptive_segments_N100", "coherent_N1", "tensor_core_flavour", "three_channels", "streams_x_one_template"):
        assert k in line["extras"], k
    assert "ms_per_eval" in line["extras"]["three_channels"] and "ms_per_eval" in line["extras"]["coherent_N1"]
