"""N > 1 host logic of bench.py on CPU: two ranks over gloo (no GPU).  The path shards as independent fields, so the
only cross-rank steps are the barrier and the max-over-ranks time; the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(extra, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2"] + extra
    env = dict(os.environ, OMP_NUM_THREADS="2")
    out = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)
    assert out.returncode == 0, out.stderr[-2000:]
    return [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]


def test_two_ranks_max_reduction_and_seeds():
    lines = _torchrun(["--selftest-ranks"])
    assert len(lines) == 1                                      # rank 0 alone prints
    d = lines[0]
    assert d["selftest"] == "ok" and d["world"] == 2
    assert d["max_ms"] == 20.0                                  # max over ranks of (10, 20)
    assert d["seeds"][0] != d["seeds"][1]


def test_reference_arm_runs_on_rank0_only():
    lines = _torchrun(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"])
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["value"] > 0 and d["unit"] == "Gpts/s" and d["n_gpus"] == 2
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
