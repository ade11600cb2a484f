"""bench.py end to end on a small BASELINE config (config 1, 33.5 M cells): one JSON line with the contract's keys,
a physical roofline fraction, launches counted, an end-to-end figure through host buffers."""
import json
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent


def test_bench_line_on_config_1():
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--config", "1", "--steps", "5", "--warmup", "3",
                        "--no-cpu-baseline", "--species-steps", "2"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, "exactly one JSON line on stdout"
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "e2e"):
        assert k in d, k
    assert d["metric"] == "phase_space_cell_updates_per_sec" and d["dtype"] == "f64" and d["n_gpus"] == 1
    assert d["steps"] == 5 and d["gpu_launches"] == 10                  # two fused kernels per step
    assert abs(d["value"] - 33554432 * 5 / (d["ms_per_step"] * 5e-3)) < 1e-6 * d["value"]
    rf = d["roofline"]
    assert rf["unit"] == "GB/s" and 0.05 < rf["frac"] < 1.2 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    assert rf["frac_algorithmic_unfused"] > rf["frac"] and rf["bound"] in ("issue", "hbm")
    assert d["e2e"]["h2d_bytes_per_step"] == 33554432 * 8 and d["e2e"]["value"] < d["value"]
    assert d["two_species"]["serial"]["ms_per_step"] > 0 and d["e2e_resident"]["value"] > d["e2e"]["value"]
