"""Multi-process launch logic of bench.py on CPU (gloo, world_size 2).

DESIGN.md section 9: the path does not shard (BASELINE north_star: one B200, no collectives), so `bench.py --gpus N`
runs N independent replicas and only the TIMING is reduced (max over ranks).  What can be covered without a GPU:
  * the reference arm under torchrun: rank 0 alone runs the oracle and prints ONE JSON line, the other rank exits 0;
  * the max-over-ranks reduction bench.py uses, on the gloo backend.
"""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_reference_arm_under_torchrun_prints_one_line():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference",
           "--gpus", "2", "--steps", "2", "--warmup", "3", "--config", "c1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "macro-particle-turns/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["n_gpus"] == 2 and d["steps"] == 2


_WORKER = r"""
import os, sys, torch, torch.distributed as dist
dist.init_process_group("gloo")
rank = dist.get_rank()
sec = torch.tensor([0.25 + 0.5 * rank], dtype=torch.float64)      # per-rank device seconds of the timed region
dist.all_reduce(sec, op=dist.ReduceOp.MAX)                         # bench.py: slowest rank's time
n_part, K, world = 1000, 4, dist.get_world_size()
value = world * n_part * K / float(sec.item())                    # whole-job throughput of the replicas
assert abs(float(sec.item()) - 0.75) < 1e-12 and abs(value - 2 * 1000 * 4 / 0.75) < 1e-9
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_replica_timing_reduction_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), str(w)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.count("ok") == 2
