"""CPU, world_size 2 over gloo: the N>1 host logic of bench.py (max-over-ranks timing, per-rank trace shards, rank-0-only
output of the reference arm). The data path itself has no collective."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _torchrun(script_args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_port())] + script_args
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)
    assert r.returncode == 0, r.stderr[-2000:]
    return [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]


def test_max_over_ranks_and_shards():
    out = _torchrun([os.path.join(ROOT, "tests", "_gloo_worker.py")])
    assert len(out) == 1
    assert out[0]["world"] == 2 and out[0]["ms"] == 15.0                  # MAX over ranks, not rank 0's 10.0
    assert out[0]["digests"][0] != out[0]["digests"][1]                  # different seeds -> different traces per rank


def test_reference_arm_prints_once_under_torchrun():
    out = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                     "--traces", "2"])
    assert len(out) == 1 and out[0]["impl"] == "reference" and out[0]["n_gpus"] == 2
    assert out[0]["cpu_baseline"]["kind"] == "oracle" and out[0]["e2e"]["h2d_bytes_per_step"] == 0
