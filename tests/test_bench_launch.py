"""CPU-only: `python bench.py --gpus N` with WORLD_SIZE unset starts its N ranks itself (the
driver calls it that way; PAPER.md:89-101 is the partition those ranks then share).  No GPU: the
ranks only join a gloo group and are counted."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra, env_extra=None):
    env = {k: v for k, v in os.environ.items()
           if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env.update(env_extra or {})
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--launch-check", *extra],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout          # rank 0 alone prints
    return json.loads(lines[0])


def test_gpus_n_spawns_n_ranks():
    line = _run(["--gpus", "2"])
    assert line == {"launch_check": True, "n_gpus": 2, "ranks_answered": 2}


def test_single_gpu_and_torchrun_environments_do_not_respawn():
    assert _run(["--gpus", "1"])["n_gpus"] == 1
    # under torchrun the environment already carries the ranks: bench.py must not start more
    line = _run(["--gpus", "2"], {"WORLD_SIZE": "1", "RANK": "0", "LOCAL_RANK": "0"})
    assert line["n_gpus"] == 1 and line["ranks_answered"] == 1
