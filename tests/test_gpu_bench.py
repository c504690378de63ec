"""bench.py prints ONE JSON line with the keys the driver's contract names (``-m gpu``; small L so it runs in
seconds -- the numbers of this run are not bench values)."""
import json
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parents[1]


def run_bench(*extra):
    cmd = [sys.executable, str(ROOT / "bench.py"), "--L", "2048", "--mcs", "20", "--steps", "2", "--warmup", "3", *extra]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_bench_line_has_the_contract_keys():
    d = run_bench()
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline"):
        assert key in d, key
    assert d["unit"] == "updates/s" and d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 3
    assert d["dtype"].startswith("u8") and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert "workload" in d["config"] and "model" not in d["config"]
    assert d["config"]["variant"] == 14                   # AUTO -> PACKED for a uint8 lattice of L = 2048
    assert d["value"] > 0 and d["e2e"]["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 2048 * 2048 and d["e2e"]["d2h_bytes_per_step"] > 2048 * 2048
    # (seed upload + init) + (seed/table upload + density + pack + order + 16 phases per MCS + unpack + finalize), per step
    assert d["gpu_launches"] == 2 * ((1 + 1) + (1 + 1 + 1 + 1 + 16 * 20 + 1 + 1))
    r = d["roofline"]                                     # the phases run on the packed working copy: ALU-bound
    assert r["bound"] == "alu" and r["unit"] == "Gdraw/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert 0.0 < r["draw_fraction"] <= 1.0 and r["hbm_context"]["algorithmic_bytes_per_launch"] == 2048 * 2048 * 17 / 16 / 8
    c8 = r["hbm_contract_u8"]                             # the north_star's formula: updates/s x 17 B / peak
    assert abs(c8["achieved"] - 8.0 * r["hbm_context"]["achieved"]) < 1e-6 * c8["achieved"]
    st = r["streaming_kernel_u8"]                         # the in-place streaming kernel, timed in the same run
    assert st["variant"] == 6 and st["bound"] == "hbm" and st["algorithmic_bytes_per_launch"] == 2048 * 2048 * 17 / 16
    assert st["updates_per_s"] > 0 and abs(st["frac"] - st["achieved"] / st["peak"]) < 1e-9
    assert d["ceilings"]["philox_step_draws_per_s"] > 1e10
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == "updates/s"
    assert c["one_thread"]["cores"] == 1 and c["one_thread"]["value"] > 0 and "MCS 0" in c["sample"]
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


def test_bench_line_for_the_streaming_kernel():
    """--variant ring: in place on the uint8 rows, the HBM roofline with the 17 B/update contract bytes."""
    d = run_bench("--variant", "ring", "--no-cpu-baseline")
    assert d["dtype"] == "u8" and d["config"]["variant"] == 6
    assert d["gpu_launches"] == 2 * ((1 + 1) + (1 + 1 + 1 + 16 * 20 + 1))
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert r["algorithmic_bytes_per_launch"] == 2048 * 2048 * 17 / 16
    a = r["alu_context"]                                  # the draws against the Philox-only ceiling
    assert a["unit"] == "Gdraw/s" and 0.0 < a["draw_fraction"] <= 1.0 and 0.0 < a["frac"] < 1.5


def test_bench_reference_arm_line():
    cmd = [sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--L", "512", "--steps", "2", "--warmup", "1"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads([ln for ln in p.stdout.splitlines() if ln.startswith("{")][0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_bench_line_for_the_papers_schedule():
    """--order dtile: same contract line, 4 launches per MCS, no class-order kernel."""
    d = run_bench("--order", "dtile", "--no-cpu-baseline")
    assert d["config"]["order_mode"] == "dtile" and d["config"]["variant"] == 10
    assert d["gpu_launches"] == 2 * ((1 + 1) + (1 + 1 + 4 * 20 + 1))
    r = d["roofline"]
    assert r["algorithmic_bytes_per_launch"] == 2048 * 2048 * 1.25 and "dtile_part_kernel" in r["kernel"]
    assert d["value"] > 0 and d["e2e"]["value"] > 0 and 0.0 <= d["final_rho_C"] <= 1.0


def test_bench_line_for_the_bit_packed_layout():
    """--fmt bits: the packed lattice is L2-resident, so the roofline object is the ALU one (STEP draws per
    second against the Philox-only ceiling) with the HBM view kept as context."""
    d = run_bench("--fmt", "bits", "--no-cpu-baseline")
    r = d["roofline"]
    assert d["dtype"].startswith("u1") and d["config"]["variant"] == 11      # AUTO -> LEAN at L = 2048, one lattice
    assert r["bound"] == "alu" and r["unit"] == "Gdraw/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert 0.0 < r["draw_fraction"] <= 1.0 and r["hbm_context"]["algorithmic_bytes_per_launch"] == 2048 * 2048 * 17 / 16 / 8
