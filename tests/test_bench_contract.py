"""bench.py prints ONE JSON line with the keys the driver reads (both arms)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
             "scaling", "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches"}


def _run(args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _run(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0", "--ref-segments", "12"])
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["metric"] == "segments_per_s" and d["unit"] == "segments/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["config"]["workload"] == "cfg1_single_track" and "model" not in d["config"]


def test_gpus_2_without_a_launcher_starts_two_ranks():
    """`bench.py --gpus 2` run as a plain script starts its own two ranks (torch.distributed.run,
    127.0.0.1); on the reference arm rank 0 alone works and prints, the other exits 0: still ONE line."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference",
                          "--config", "1", "--steps", "1", "--warmup", "0", "--ref-segments", "12"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1, out.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["impl"] == "reference" and d["value"] > 0
    # a launcher's world size that contradicts --gpus is refused, not silently reported as N
    bad = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=dict(env, WORLD_SIZE="1", RANK="0"))
    assert bad.returncode == 2 and "WORLD_SIZE" in bad.stderr


@pytest.mark.gpu
def test_cuda_arm_line():
    d = _run(["--config", "1", "--steps", "3", "--warmup", "3", "--ref-segments", "12"])
    assert BASE_KEYS | {"roofline", "cpu_baseline", "clocks", "stage_ms"} <= set(d)
    assert d["n_gpus"] == 1 and d["scaling"] == "weak" and d["dtype"].startswith("f32") and d["vs_baseline"] is None
    assert d["config"]["mac_mode_ran"] in (1, 2, 3, 5, 6, 7) and d["fma_tflops_measured"] > 10
    assert "tred_simulate" in d["e2e"]["through"] and d["config"]["host_reads"] == 1
    assert d["gpu_launches"] > 0 and d["value"] > 0 and d["e2e"]["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    r = d["roofline"]
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(r)
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
