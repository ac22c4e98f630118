"""bench.py's command line on CPU: `--gpus N` outside torchrun starts N ranks itself (here the
reference arm, which rendezvouses over gloo), both arms print the same `config` object, `e2e.unit`
is the metric's unit, and the uep arm refuses to run on fewer GPUs than asked for."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*argv, timeout=300):
    env = {k: v for k, v in os.environ.items()
           if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], cwd=ROOT, env=env,
                          capture_output=True, text=True, timeout=timeout)


def test_gpus_2_reference_arm_starts_two_ranks():
    r = _run("--gpus", "2", "--impl", "reference", "--workload", "tiny", "--steps", "2", "--warmup", "1")
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["ranks_started"] == 2
    assert d["unit"] == "us/layer" and d["e2e"]["unit"] == "us/layer" and d["e2e"]["value"] == d["value"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["higher_is_better"] is False
    sys.path.insert(0, ROOT)
    import bench
    args = bench.parse_args(["--gpus", "2", "--impl", "reference", "--workload", "tiny", "--steps", "2"])
    assert d["config"] == bench.config_of(args, bench.workload("tiny"))    # same object as the uep arm prints
    assert d["config"]["workload"] == "tiny"


def test_single_rank_reference_arm_and_config_keys():
    r = _run("--impl", "reference", "--workload", "tiny", "--steps", "1", "--warmup", "0")
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    assert d["n_gpus"] == 1 and d["ranks_started"] == 1
    assert {"workload", "T", "k", "E", "R", "n_slot", "u_min", "beta", "floor_mode", "gate",
            "state_bytes_per_expert", "zipf_s", "instances", "l2", "parallelism", "state_scale"} == set(d["config"])


def test_uep_arm_refuses_fewer_gpus_than_requested():
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        return                                               # only meaningful where 2 GPUs are NOT there
    r = _run("--gpus", "2", "--steps", "1", "--warmup", "0", timeout=120)
    assert r.returncode != 0
    assert "refusing to run on fewer GPUs" in (r.stderr + r.stdout)


def test_gpus_must_match_world_size():
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--impl", "reference"],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode != 0 and "WORLD_SIZE=2" in (r.stderr + r.stdout)
