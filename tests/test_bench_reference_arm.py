"""bench.py --impl reference runs the oracle only (no CUDA library, no GPU) and prints one JSON line with the
keys the measurement contract names, on the same `config` keys as the CUDA arm."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_json_line_c1():
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["unit"] == "ms" and out["higher_is_better"] is False
    assert out["value"] > 0 and out["ms_per_step"] == out["value"] and out["vs_baseline"] is None
    assert out["cpu_baseline"]["kind"] == "oracle" and out["cpu_baseline"]["cores"] >= 1 and out["cpu_baseline"]["sample"]
    assert out["e2e"] == {"value": out["value"], "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    cfg = out["config"]
    assert cfg["workload"] == "C1-tiny" and cfg["n"] == 256 and cfg["heads"] == 2 and cfg["D"] == 64
    for k in ("cell_q", "cell_k", "win", "iters", "top_p", "merge_rounds", "tile", "l2", "parallelism"):
        assert k in cfg


def test_reference_arm_other_ranks_do_no_work():
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert r.returncode == 0 and r.stdout.strip() == ""
