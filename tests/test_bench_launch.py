"""CPU: `python bench.py --gpus 2` as the driver types it (no launcher around it) must start two ranks itself, shard the
reads by rank, take the max over ranks of the timed region and have rank 0 alone print one JSON line.  --plumbing-only
runs exactly that host path over gloo with the device work replaced by a rank-dependent sleep (no GPU here)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra, env_extra=None):
    env = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    env.update(env_extra or {})
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--plumbing-only", "--steps", "3", "--warmup", "1", *extra]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    if r.returncode != 0 and ("address already in use" in r.stderr.lower() or "timed out" in r.stderr.lower()):
        # the rendezvous port is picked free and then bound by the launcher: another process can take it in between; once more
        r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout                       # rank 0 alone prints
    return json.loads(lines[0])


def test_gpus_2_spawns_two_ranks_and_takes_the_max():
    d = _run("--gpus", "2", "--reads", "48")
    assert d["n_gpus"] == 2 and d["steps"] == 3 and d["scaling"] == "weak"
    assert d["reads_per_gpu"] == 48                         # weak scaling: every rank maps its own batch of that size
    assert len(d["read_digests"]) == 2 and d["read_digests"][0] != d["read_digests"][1]   # per-rank seeds differ
    # rank 0 "works" 50 ms per step, rank 1 100 ms: the reported time is the slower rank's (sleep never returns early)
    assert d["ms_per_step"] >= 99.0 and d["ms_per_step"] * 3 >= d["own_ms_rank0"]


def test_gpus_1_stays_in_process():
    d = _run("--gpus", "1", "--reads", "48")
    assert d["n_gpus"] == 1 and len(d["read_digests"]) == 1


def test_under_an_external_launcher_the_env_decides():
    """torchrun-style launch of a single rank: WORLD_SIZE is set, so bench.py must not spawn anything itself."""
    d = _run("--gpus", "1", env_extra={"RANK": "0", "WORLD_SIZE": "1", "LOCAL_RANK": "0", "MASTER_ADDR": "127.0.0.1",
                                       "MASTER_PORT": "29591"})
    assert d["n_gpus"] == 1
