"""-m "not gpu": the reference arm of bench.py (the oracle on the host cores) runs without a GPU and
prints one JSON line carrying the contract's keys."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "2",
                          "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "demag_Hd_evals_per_s" and d["unit"] == "evals/s"
    for key in ("value", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in d["config"] and d["vs_baseline"] is None


def test_reference_arm_on_other_ranks_prints_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "2",
                          "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


import pytest


@pytest.mark.gpu
def test_our_arm_prints_the_contract_line_on_a_small_grid():
    """The GPU arm end to end on a debug grid (marked as not a BASELINE config): one JSON line with the keys
    the contract asks for — roofline of the dominant kernel, cpu_baseline (oracle), e2e with declared copy
    bytes, launches counted inside the timed region, clocks sampled during it."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--grid", "24,16,4", "--steps", "5", "--warmup", "3"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks",
                "measured_peaks", "assembly", "llg_rhs", "batch8"):
        assert key in d, key
    assert d["metric"] == "demag_Hd_evals_per_s" and d["n_gpus"] == 1 and d["steps"] == 5 and d["vs_baseline"] is None
    assert "DEBUG grid" in d["config"]["workload"] and d["dtype"] == "f32" and d["data"] == "synthetic"
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert r["traffic"] is None            # no ncu capture exists for a debug grid
    assert d["gpu_launches"] >= 2 * d["steps"] and d["value"] > 0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 3 * 1536 * 8 and e["d2h_bytes_per_step"] == 3 * 1536 * 8 and e["value"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["single_thread"]["cores"] == 1
    assert d["assembly"]["every_pair_evaluated"] and d["assembly"]["pairs"] == 1536 * 1536
