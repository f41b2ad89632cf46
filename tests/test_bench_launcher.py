"""`python bench.py --gpus N` must start N ranks by itself (the driver's scaling run issues exactly that), print one
line with the rank count it really used, and refuse to run fewer ranks than asked.  CPU only: the `--dry-run-ranks`
path does the rank plumbing (launcher, rendezvous on 127.0.0.1, gloo all-gather of the charge slices) without CUDA."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*argv, env=None):
    e = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        e.pop(k, None)
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + list(argv), capture_output=True, text=True,
                          timeout=600, env=e, cwd=ROOT)


def test_gpus_2_starts_two_ranks_and_prints_one_line():
    r = _run("--gpus", "2", "--dry-run-ranks")
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["gather_ok"] is True


def test_gpus_2_without_two_devices_fails_loudly():
    r = _run("--gpus", "2", "--steps", "1", "--warmup", "0", env={"CUDA_VISIBLE_DEVICES": ""})
    assert r.returncode != 0
    assert "--gpus 2" in r.stderr and "visible" in r.stderr
    assert not [ln for ln in r.stdout.splitlines() if ln.startswith("{")]


def test_world_size_must_match_gpus():
    r = _run("--gpus", "1", "--dry-run-ranks", env={"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0",
                                                      "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": "29999"})
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)
