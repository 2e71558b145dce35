"""bench.py command line on a box without a GPU: the reference arm and the self-spawned multi-rank launch."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*argv, env=None):
    e = dict(os.environ)
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        e.pop(k, None)
    e.update(env or {})
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True, env=e, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    return [json.loads(l) for l in lines]


def test_reference_arm_line():
    out = _run("--impl", "reference", "--workload", "C1", "--steps", "2", "--warmup", "3")
    assert len(out) == 1
    d = out[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 1 and d["unit"] == "sample-steps/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"].startswith("C1: n=4 m=1 d=8 N=1024/GPU")


def test_gpus_flag_starts_the_ranks_itself():
    """`python bench.py --gpus 2` without a launcher re-executes under torch.distributed.run with two ranks (127.0.0.1);
    in the reference arm rank 0 alone works and prints, n_gpus is the real world size and the workload is the
    2-rank global candidate set."""
    out = _run("--gpus", "2", "--impl", "reference", "--workload", "C1", "--steps", "1", "--warmup", "3")
    assert len(out) == 1, out
    d = out[0]
    assert d["n_gpus"] == 2 and d["impl"] == "reference"
    assert "N=1024/GPU" in d["config"]["workload"] and "of 2048 candidates" in d["config"]["sample"]
