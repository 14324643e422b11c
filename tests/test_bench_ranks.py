"""The N > 1 path of bench.py on CPU: world_size-2 gloo run of the aggregation (max time over ranks, summed
work: "replicas only") and of the reference arm (rank 0 alone runs the oracle and prints)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(args, timeout=300):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py")] + args
    out = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)
    assert out.returncode == 0, out.stderr[-2000:]
    return [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]


def test_two_rank_aggregation_gloo():
    lines = _torchrun(["--gpus", "2", "--selftest-ranks"])
    assert len(lines) == 1                      # rank 0 alone prints
    d = lines[0]
    assert d["n_gpus"] == 2 and d["ms"] == 2.0  # max over ranks of (1 + rank) ms
    assert abs(d["value"] - 2 * 2 * 1000 * 1000 / (2.0 * 1e6)) < 1e-12     # work of both ranks / max time


def test_reference_arm_under_torchrun_prints_once():
    lines = _torchrun(["--gpus", "2", "--impl", "reference", "--steps", "1", "--warmup", "0", "--L", "16384"])
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0
