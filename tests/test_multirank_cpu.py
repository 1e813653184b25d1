"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path is "replicas only" (DESIGN.md
section 8), so what there is to test is the plumbing - max-over-ranks timing, whole-job aggregation,
and that only rank 0 of the reference arm works and prints."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, 2, "cpu")          # rank 1 is the slow one
dist.barrier()
val = bench.aggregate_throughput(1000, 10, 4, 2, ms)
print(json.dumps({{"rank": rank, "ms": ms, "value": val}}))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (out, err) in zip(procs, outs):
        assert p.returncode == 0, err
    rows = [json.loads(out.strip().splitlines()[-1]) for out, _ in outs]
    for r in rows:
        assert r["ms"] == 15.0                                    # the slowest rank's clock, on every rank
        assert r["value"] == pytest.approx(2 * 1000 * 10 * 4 / 15e-3)


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun (N > 1) rank 0 alone times the oracle and prints; the other ranks exit 0 silently."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0", "--config", "2", "--cells", "6", "--cpu-seconds", "1"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
