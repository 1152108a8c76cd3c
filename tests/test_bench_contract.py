"""bench.py's reference arm runs on the host cores only (the oracle), so its JSON line can be checked here without a GPU:
the keys the driver reads, the tier's extra objects, and that metric / unit / config agree with the GPU arm's constants."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0", *args],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    return json.loads(out.stdout.strip().splitlines()[-1])


def test_reference_line_config4():
    d = _run("--config", "4", "--log2-points", "16")
    assert d["impl"] == "reference" and d["metric"] == "atom_grid_evals_per_s" and d["unit"] == "evals/s"
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["cpu_baseline"]["value"] == d["value"] and d["e2e"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["gpu_launches"] == 0
    assert "workload" in d["config"]


def test_reference_line_config0():
    d = _run("--config", "0")
    assert d["impl"] == "reference" and d["metric"] == "replica_md_steps_per_s" and d["unit"] == "replica-steps/s"
    assert d["value"] > 0 and d["config"]["n_replicas"] == 64 and d["config"]["atoms"] == 12
    assert "sample" in d["cpu_baseline"] and d["steps"] == 1


def test_non_zero_rank_of_the_reference_arm_prints_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], capture_output=True, text=True,
                         timeout=300, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
