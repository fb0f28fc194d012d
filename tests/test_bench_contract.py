"""bench.py contract checks that need no GPU: the reference arm (`--impl reference`, the CPU oracle) prints
one JSON line with the keys the driver reads."""
import json
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def test_reference_arm_prints_one_json_line():
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                        "--ref-states", "2"], capture_output=True, text=True, timeout=600, cwd=str(ROOT))
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "states/s" and d["higher_is_better"] is True
    assert d["metric"] == "counterfactual_state_renders_per_s" and d["value"] > 0
    assert d["config"]["workload"] == "cfg1_object_centric_800x800_B256"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": "states/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0 and d["steps"] == 1 and d["warmup"] == 0


def test_our_arm_refuses_to_run_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("this check is for the CPU-only box")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--steps", "1", "--warmup", "0"], capture_output=True,
                       text=True, timeout=600, cwd=str(ROOT))
    assert r.returncode != 0 and "CUDA" in (r.stderr + r.stdout)


def test_gpus_n_without_torchrun_fails_loudly_when_the_box_has_fewer_gpus():
    """`python bench.py --gpus N` starts its N ranks itself; with fewer than N devices it must refuse, not time one
    GPU and print n_gpus: 1."""
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        import pytest
        pytest.skip("needs a box with fewer than 2 GPUs")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, cwd=str(ROOT))
    assert r.returncode != 0
    assert "--gpus 2" in (r.stderr + r.stdout) and not [l for l in r.stdout.splitlines() if l.startswith("{")]


def test_reference_arm_with_gpus_2_is_one_line_from_rank_0():
    """Under N > 1 the reference arm (the CPU oracle) is run by rank 0 alone: one line, n_gpus as asked."""
    import os
    base = [sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
            "--ref-states", "2"]
    r0 = subprocess.run(base, capture_output=True, text=True, timeout=600, cwd=str(ROOT),
                        env=dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0"))
    r1 = subprocess.run(base, capture_output=True, text=True, timeout=600, cwd=str(ROOT),
                        env=dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1"))
    assert r0.returncode == 0 and r1.returncode == 0
    lines = [l for l in r0.stdout.splitlines() if l.strip()]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2
    assert not r1.stdout.strip()
