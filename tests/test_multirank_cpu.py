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


def test_bench_gpus_2_launches_two_ranks_itself():
    """`python bench.py --gpus 2` with no launcher around it (WORLD_SIZE unset) must start two ranks:
    the line it prints says n_gpus = 2 and carries the max over the two ranks' (fake) region times.
    --plumbing-only keeps the CUDA step out so that this runs on a CPU box with the gloo backend."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "4", "--plumbing-only"],
                         env=env, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout                       # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["steps"] == 4
    assert line["plumbing_only"]["max_over_ranks_ms"] == 15.0          # rank 1's 15 ms, not rank 0's 10 ms
    assert abs(line["plumbing_only"]["aggregate_of_fake_region"] - 2 * 1000 * 4 / 0.015) < 1e-6


def test_single_rank_helpers():
    import torch
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks_ms(7.5, 1, torch.device("cpu")) == 7.5
    assert bench.whole_job_value(10, 2, 1000.0, 1) == 20.0


# ---------------------------------------------------------------------------------------------
# Workers mode (include/scape.h "Workers"): the host-side protocol on two gloo ranks.  The kernels
# need a GPU (tests/test_gpu_workers.py); what runs here is everything around them: every rank
# derives the same layer owners, the mask portions the owners produce are disjoint, and the
# integer all-reduce SUM the binding uses for them is a bitwise OR.
# ---------------------------------------------------------------------------------------------
WORKER_PROTOCOL = r"""
import os, sys
sys.path.insert(0, os.environ["SCAPE_ROOT"])
import numpy as np, torch, torch.distributed as dist
from paper_2607_01678_b200 import workers
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
sizes = [1000, 1, 5, 127, 129, 4099, 64, 20011, 2]
owner = workers.balance_layers(sizes, world)
got = [None] * world
dist.all_gather_object(got, owner)
assert all(g == owner for g in got), got                      # the same decision on every rank
offsets = np.concatenate([[0], np.cumsum(sizes)])
N = int(offsets[-1])
rng = np.random.default_rng(7)                                # same stream on both ranks
full = rng.integers(0, 2, N).astype(np.uint8)                 # a "true" M_t
mine = np.zeros(N, np.uint8)
for l, o in enumerate(owner):
    if o == rank:
        mine[offsets[l]:offsets[l + 1]] = full[offsets[l]:offsets[l + 1]]
pad = (-N) % 32
bits = np.packbits(np.concatenate([mine, np.zeros(pad, np.uint8)]), bitorder="little").view(np.uint32)
words = torch.from_numpy(bits.view(np.int32).copy())
dist.all_reduce(words, op=dist.ReduceOp.SUM)                  # disjoint portions: SUM == OR
out = np.unpackbits(words.numpy().view(np.uint8), bitorder="little")[:N]
assert np.array_equal(out, full)
# the word ranges a rank may touch cover its layers and nothing is lost when only those are exchanged
rngs = workers.owned_word_ranges(offsets, owner, rank)
cover = np.zeros(bits.size, bool)
for a, b in rngs:
    cover[a:b] = True
assert not bits[~cover].any()
# the exchange the library performs (scape_step_exchange; Scape.step_workers over torch.distributed):
# every word range broadcast from its owner, the shared words summed -- nothing else moves
ranges, shared = workers.exchange_plan(offsets, owner, N)
w2 = torch.from_numpy(bits.view(np.int32).copy())
moved = 0
for a, b, o in ranges:
    dist.broadcast(w2[a:b], src=o)
    moved += b - a
if shared:
    ix = torch.tensor(shared, dtype=torch.int64)
    sw = w2[ix]
    dist.all_reduce(sw, op=dist.ReduceOp.SUM)
    w2[ix] = sw
assert np.array_equal(np.unpackbits(w2.numpy().view(np.uint8), bitorder="little")[:N], full)
assert moved + len(shared) == bits.size and len(shared) < len(sizes)       # every word exactly once
sums = torch.full((5,), float(rank + 1))
dist.all_reduce(sums, op=dist.ReduceOp.SUM)
assert float(sums[0]) == sum(range(1, world + 1))
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_two_gloo_ranks_workers_protocol():
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), SCAPE_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER_PROTOCOL], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
        assert "ok" in o


def test_balance_layers_is_even_and_deterministic():
    sys.path.insert(0, ROOT)
    from paper_2607_01678_b200 import workers
    sizes = [50257 * 1024, 1024 * 1024] + [3072 * 1024, 1024 * 1024, 4096 * 1024, 4096 * 1024] * 24
    for world in (1, 2, 4, 8, 64):
        owner = workers.balance_layers(sizes, world)
        assert owner == workers.balance_layers(list(sizes), world)
        load = [0] * world
        for s, o in zip(sizes, owner):
            load[o] += s
        assert max(load) - min(load) <= max(sizes)            # within one (largest) layer of even
    assert workers.owned_word_ranges([0, 40, 64, 100], [0, 1, 0], 0) == [(0, 4)]
    assert workers.owned_word_ranges([0, 40, 64, 100], [0, 1, 0], 1) == [(1, 2)]
    assert workers.owned_word_ranges([0, 64, 640, 700], [0, 1, 0], 0) == [(0, 2), (20, 22)]
    # the plan of the exchange: runs of one owner become exclusive word ranges, boundary words are shared
    assert workers.exchange_plan([0, 64, 640, 700], [0, 1, 0], 700) == ([(0, 2, 0), (2, 20, 1), (20, 22, 0)], [])
    assert workers.exchange_plan([0, 37, 40, 128, 1128, 1141, 5148], [0, 1, 0, 1, 0, 1], 5148) == \
        ([(0, 1, 0), (2, 4, 0), (4, 35, 1), (36, 161, 1)], [1, 35])
    assert workers.exchange_plan([0, 10, 20], [1, 1], 20) == ([(0, 1, 1)], [])
