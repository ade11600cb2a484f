"""Host-side arithmetic of bench.py (no GPU): the roofline object is a physical fraction, the survey's unfused
currency is kept under its own names, ncu counters are quoted only while the source hash matches."""
import json
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))


class _W:
    name = "c3_harris2d_128x64x40^3"
    n_cells = 524288000


def _timings(ms_v=2.0, ms_x=1.5, steps=10):
    nf = _W.n_cells
    return {"fused_vx_vy_vz_moments": dict(ms=ms_v * steps, launches=steps, alg_bytes=56.0 * nf, moved_bytes=16.0 * nf),
            "fused_sx_sy": dict(ms=ms_x * steps, launches=steps, alg_bytes=32.0 * nf, moved_bytes=16.0 * nf)}


def test_roofline_fraction_is_moved_bytes_over_time_over_peak(monkeypatch, tmp_path):
    import bench
    monkeypatch.setattr(bench, "COUNTERS", tmp_path / "none.json")
    r = bench.make_roofline(_timings(), 10, 3.5, 6551.7, "measured", {"sm_mhz": 1965.0}, 148, _W)
    assert r["kernel"] == "fused_vx_vy_vz_moments" and r["bound"] == "issue"
    want = 16.0 * _W.n_cells / 2.0e-3 / 1e9
    assert abs(r["achieved"] - want) < 1e-6 * want and abs(r["frac"] - want / 6551.7) < 1e-9
    assert r["frac"] < 1.0 < r["frac_algorithmic_unfused"]          # fusion shows only in the unfused currency
    assert abs(r["step"]["frac"] - 32.0 * _W.n_cells / 3.5e-3 / 1e9 / 6551.7) < 1e-9
    assert abs(r["step"]["frac_algorithmic_unfused_of_8TBps"] - 88.0 * _W.n_cells / 3.5e-3 / 8e12) < 1e-9
    assert r["traffic"] is None and "traffic_note" in r
    assert r["kernels"]["fused_sx_sy"]["bound"] == "hbm" and abs(r["share_of_step"] - 2.0 / 3.5) < 1e-12


def test_counters_are_quoted_only_for_matching_sources(monkeypatch, tmp_path):
    import bench
    cj = tmp_path / "kernel_counters.json"
    monkeypatch.setattr(bench, "COUNTERS", cj)
    k = {"fused_vx_vy_vz_moments": {"dram_bytes": 8374000000, "warp_instructions": 1221000000,
                                     "fp64_pipe_warp_instructions": 620000000, "dfma_warp_instructions": 187000000}}
    cj.write_text(json.dumps({"csrc_sha16": "0" * 16, "commit": "x", "workload": _W.name, "kernels": k}))
    r = bench.make_roofline(_timings(), 10, 3.5, 6551.7, "measured", {"sm_mhz": 1965.0}, 148, _W)
    assert r["traffic"] is None and "differ" in r["traffic_note"]
    cj.write_text(json.dumps({"csrc_sha16": bench.csrc_sha16(), "commit": "x", "workload": _W.name, "kernels": k}))
    r = bench.make_roofline(_timings(), 10, 3.5, 6551.7, "measured", {"sm_mhz": 1965.0}, 148, _W)
    assert r["traffic"] == 8374000000
    # issue roofline: one instruction per scheduler per cycle; fp64 pipe: 2 cycles per DADD / DSETP / DMUL, 3 per DFMA
    assert abs(r["issue"]["frac"] - 1221000000 / 2.0e-3 / (148 * 4 * 1.965e9)) < 1e-4
    cycles = 2.0 * (620000000 - 187000000) + 3.0 * 187000000
    assert abs(r["fp64_pipe"]["pipe_floor_ms"] - cycles / 592 / 1.965e9 * 1e3) < 1e-3
    assert abs(r["fp64_pipe"]["frac"] - r["fp64_pipe"]["pipe_floor_ms"] / 2.0) < 1e-3


def test_committed_counters_match_the_committed_sources():
    import bench
    cj = json.loads((ROOT / "profiles" / "kernel_counters.json").read_text())
    assert cj["csrc_sha16"] == bench.csrc_sha16(), "profiles/kernel_counters.json is stale: re-capture it (DESIGN.md sec. 7)"


def test_reference_arm_prints_one_json_line():
    """bench.py --impl reference: the oracle on the host cores, same metric and workload name, no GPU needed."""
    import subprocess
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "phase_space_cell_updates_per_sec" and d["value"] > 0
    assert d["config"]["workload"] == _W.name and d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
