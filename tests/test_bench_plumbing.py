"""bench.py's N-rank entry point on CPU: `python bench.py --gpus 2 ...` launched PLAINLY (no torchrun environment) must
re-execute itself under torch.distributed.run, bring up 2 ranks (gloo here, nccl on the GPU box), and print ONE line
from rank 0 with n_gpus = 2; a --gpus that contradicts WORLD_SIZE must fail loudly; the reference arm under torchrun
prints one line from rank 0 only."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env_extra=None, timeout=600):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env.update(env_extra or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, env=env, cwd=ROOT, capture_output=True,
                          text=True, timeout=timeout)


def _json_lines(out):
    return [json.loads(ln) for ln in out.splitlines() if ln.startswith("{")]


def test_gpus_2_spawns_two_ranks_and_prints_one_line():
    p = _run(["--gpus", "2", "--plumbing-check"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = _json_lines(p.stdout)
    assert len(lines) == 1
    assert lines[0]["n_gpus"] == 2 and lines[0]["ranks_seen"] == 2 and lines[0]["max_over_ranks_ms"] == 11.0
    assert len(set(lines[0]["seeds"])) == 2                   # weak scaling: each rank draws its own batch


def test_gpus_must_match_world_size():
    p = _run(["--gpus", "3", "--plumbing-check"], {"RANK": "0", "LOCAL_RANK": "0", "WORLD_SIZE": "1"})
    assert p.returncode != 0 and "WORLD_SIZE" in (p.stderr + p.stdout)


def test_reference_arm_under_two_ranks_prints_one_line():
    p = _run(["--gpus", "2", "--impl", "reference", "--steps", "1", "--warmup", "0"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = _json_lines(p.stdout)
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2
    assert lines[0]["cpu_baseline"]["kind"] == "oracle" and lines[0]["value"] > 0
    assert lines[0]["e2e"]["h2d_bytes_per_step"] == 0
