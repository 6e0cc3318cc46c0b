"""bench.py prints ONE JSON line with the keys the driver reads (both arms)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches"}


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    """--impl reference: the oracle, as it stands, on the host cores; same metric/unit/config keys, no GPU work claimed."""
    line = _run("--impl", "reference", "--config", "0", "--steps", "2", "--warmup", "1")
    assert BASE_KEYS <= set(line) and line["impl"] == "reference"
    assert line["unit"] == "jacobian_builds/s" and line["dtype"] == "f64" and line["data"] == "synthetic"
    assert line["value"] > 0 and line["gpu_launches"] == 0 and line["vs_baseline"] is None
    assert line["config"]["workload"] == "cfg0-tiny" and "model" not in line["config"]
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", ["0", "2"])
def test_gpu_arm_line(cfg):
    line = _run("--config", cfg, "--steps", "5", "--warmup", "3", "--no-cpu-baseline")
    assert BASE_KEYS | {"roofline", "clocks"} <= set(line)
    assert line["n_gpus"] == 1 and line["steps"] == 5 and line["warmup"] >= 3 and line["higher_is_better"] is True
    assert line["value"] > 0 and abs(line["value"] - 1e3 / line["ms_per_step"]) <= 1e-6 * line["value"]
    assert line["gpu_launches"] >= 1 * 5                       # at least one kernel per step (pipelined shapes: the whole build)
    r = line["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert 30.0 < r["peak"] < 45.0 and r["kernel_ms"] > 0
    e = line["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert e["value"] < line["value"] * 1.05                   # the host-buffer path cannot beat the device-resident one
    assert set(line["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    if cfg == "2":
        s = line["newton_solve"]
        assert s["steps_per_solve"] == 8 and s["converged_solve"]["status"] == 1
        assert abs(s["converged_solve"]["alpha_MZ2"] - 0.118) < 1e-3
    else:
        assert line["with_newton_update"]["value"] > 0
