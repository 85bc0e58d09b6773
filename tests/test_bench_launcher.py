"""bench.py --gpus N outside torchrun starts the N ranks itself.  CPU only:
the ranks join a gloo group (no GPU here), and the reference arm, which needs no GPU, runs under the
same launcher with rank 0 alone printing the line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*argv, timeout=600):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True, timeout=timeout, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    return [json.loads(ln) for ln in lines]


def test_gpus_2_spawns_two_ranks_gloo():
    out = _run("--gpus", "2", "--launch-selftest")
    assert len(out) == 1                                   # rank 0 alone prints
    assert out[0]["n_gpus"] == 2 and out[0]["ranks_counted"] == 2
    assert out[0]["max_ms"] == 2.0                         # max over ranks of (1 + rank) ms


def test_gpus_1_does_not_spawn():
    out = _run("--launch-selftest")
    assert len(out) == 1 and out[0]["n_gpus"] == 1 and out[0]["ranks_counted"] == 1


def test_reference_arm_under_the_launcher_names_what_it_times():
    out = _run("--gpus", "2", "--impl", "reference", "--workload", "8^4", "--steps", "2", "--warmup", "1")
    assert len(out) == 1
    line = out[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["steps"] == 2
    assert line["config"]["lattice"] == [8, 8, 8, 8] and line["config"]["workload"].startswith("8^4 ")
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
