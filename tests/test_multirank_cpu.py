"""N > 1 path of bench.py on CPU: two gloo ranks, 127.0.0.1.  The path does not shard ("replicas
only"), so what needs covering is the host logic: the barrier, the max-over-ranks time and the
whole-job aggregate."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["SCAPE_ROOT"])
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks_ms(10.0 + 5.0 * rank, world, torch.device("cpu"))
assert ms == 15.0, ms
v = bench.whole_job_value(1000, 4, ms, world)
assert abs(v - 2 * 1000 * 4 / 0.015) < 1e-6, v
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_gloo_ranks_aggregate():
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), SCAPE_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
        assert "ok" in o


def test_single_rank_helpers():
    import torch
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks_ms(7.5, 1, torch.device("cpu")) == 7.5
    assert bench.whole_job_value(10, 2, 1000.0, 1) == 20.0
