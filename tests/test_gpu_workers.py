"""Parity of the workers mode — `-m gpu`.

One GPU: W workers are W handles in ONE process, stepped one after the other (no kernel waits
on another), and the exchange between scape_step_local and scape_step_apply is done here with
torch adds in worker order — exactly what an all-reduce SUM delivers for W = 2 (one addition,
commutative) and the order the oracle's two-level sum fixes for W > 2.  Bar: masks / indices
bit-exact, theta / m / e to the bit, on every worker, against the oracle with R = W * R_local
replicas and the same layer owners.
"""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.scape_oracle import ScapeOracle  # noqa: E402
from paper_2607_01678_b200 import synth, workers  # noqa: E402
from test_gpu_parity import HYP, B, assert_close, to_np32  # noqa: E402,F401

pytestmark = pytest.mark.gpu


def exchange(handles):
    """Sum of the workers' exchange buffers, in worker order, written back to every worker."""
    bufs = [h.exchange_tensors() for h in handles]
    tot = bufs[0][0].clone()
    for s, _ in bufs[1:]:
        tot += s
    for s, _ in bufs:
        s.copy_(tot)
    if bufs[0][1] is not None:
        wt = bufs[0][1].clone()
        for _, w in bufs[1:]:
            assert int((wt & w).ne(0).sum()) == 0, "the workers' mask portions overlap"
            wt += w                                  # disjoint bits: SUM == OR, what the all-reduce computes
        for _, w in bufs:
            w.copy_(wt)


def run_workers(B, sizes, comp, W, Rl, s, gdt, steps, seed, schedule=None, owner=None):
    R = W * Rl
    w = synth.Workload(f"workers/W{W}xR{Rl}", [(f"t{i}", n) for i, n in enumerate(sizes)], R=R, sparsity=s,
                       dist="t3", rho=0.9, grad_dtype=gdt, steps=steps)
    offsets = w.offsets()
    owner = workers.balance_layers(sizes, W) if owner is None else owner
    gs = synth.GradStream(w, device="cuda", seed=seed)
    th0 = gs.theta0()
    ora = ScapeOracle(w.numel, R, s, **w.hyper)
    ora.set_layers(offsets, comp)
    ora.set_workers(W, owner)
    th_ora = th0.cpu().numpy().copy()
    hs, ths = [], []
    for r in range(W):
        h = B.Scape(w.numel, Rl, s, **w.hyper)
        h.set_layers(offsets, comp)
        h.set_workers(W, r, owner)
        hs.append(h)
        ths.append(th0.clone())
    for t in range(1, steps + 1):
        grads = gs.next()
        if schedule is not None:
            ora.set_sparsity(schedule(t))
            for h in hs:
                h.set_sparsity(schedule(t))
        for r, h in enumerate(hs):
            h.step_local(ths[r], grads[r * Rl:(r + 1) * Rl])
        exchange(hs)
        for r, h in enumerate(hs):
            h.step_apply(ths[r])
        ora.step(th_ora, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        mk = ora.mask()
        for r, h in enumerate(hs):
            tag = f"W={W} Rl={Rl} step {t} worker {r}"
            assert h.count_last() == ora.K_last, tag
            np.testing.assert_array_equal(h.idx_last(), ora.idx(), err_msg=tag + " idx_last")
            np.testing.assert_array_equal(h.mask_next(), mk, err_msg=tag + " mask_next")
            np.testing.assert_array_equal(h.idx_next(), np.nonzero(mk)[0].astype(np.int32), err_msg=tag + " idx_next")
            th = ths[r].cpu().numpy()
            assert_close(th, th_ora, tag + " theta")
            assert np.array_equal(th.view(np.uint32), th_ora.view(np.uint32)), tag + " theta not bit-exact"
            assert np.array_equal(h.moment().view(np.uint32), ora.m().view(np.uint32)), tag + " m not bit-exact"
            assert np.array_equal(h.packed_mean().view(np.uint32), ora.bbar().view(np.uint32)), tag + " bbar"
            for q in range(Rl):
                assert np.array_equal(h.residual(q).view(np.uint32), ora.e(r * Rl + q).view(np.uint32)), tag + f" e[{q}]"
                if ora.K_last < w.numel:
                    assert np.array_equal(h.packed(q).view(np.uint32), ora.b(r * Rl + q).view(np.uint32)), tag + f" b[{q}]"
    for h in hs:
        h.close()


RAGGED = ([1000, 1, 5, 127, 129, 4096 + 3, 64, 20_000 + 11, 2], [1, 1, 1, 1, 1, 1, 0, 1, 1])
BIG = ([128 * 700 + 5, 128 * 500, 1024, 128 * 900 + 77, 4096 * 3], [1, 1, 0, 1, 1])     # > 148 tiles: staged kernel


@pytest.mark.parametrize("W,Rl,s,gdt", [(2, 1, 0.9, "f32"), (2, 2, 0.99, "bf16"), (4, 1, 0.9, "f32"), (3, 2, 0.5, "f32")])
def test_workers_ragged_layers(B, W, Rl, s, gdt):
    sizes, comp = RAGGED
    run_workers(B, sizes, comp, W, Rl, s, gdt, steps=8, seed=W + Rl)


@pytest.mark.parametrize("W,Rl,s,gdt", [(2, 4, 0.99, "bf16"), (2, 3, 0.9, "f32")])
def test_workers_staged_kernel(B, W, Rl, s, gdt):
    sizes, comp = BIG
    run_workers(B, sizes, comp, W, Rl, s, gdt, steps=10, seed=5)


def test_workers_owner_layouts_and_boundaries_inside_words(B):
    # neighbouring layers of different owners meet inside one 32-bit word and inside one chunk
    sizes = [37, 3, 88, 1000, 13, 4000 + 7]
    run_workers(B, sizes, [1] * 6, 2, 1, 0.75, "f32", steps=6, seed=9, owner=[0, 1, 0, 1, 0, 1])
    run_workers(B, sizes, [1, 0, 1, 1, 0, 1], 3, 1, 0.75, "f32", steps=6, seed=9, owner=[2, 1, 0, 0, 1, 2])


def test_workers_density_warmup_and_back_to_dense(B):
    sizes, comp = RAGGED
    sched = lambda t: [0.0, 0.5, 0.9, 0.99, 0.99, 0.0, 0.0, 0.9][t - 1]     # noqa: E731
    run_workers(B, sizes, comp, 2, 2, 0.0, "f32", steps=8, seed=4, schedule=sched)


def test_split_step_with_one_worker_is_the_whole_step(B):
    sizes, comp = RAGGED
    w = synth.Workload("workers/one", [(f"t{i}", n) for i, n in enumerate(sizes)], R=3, sparsity=0.9,
                       dist="gauss", rho=0.9, grad_dtype="f32", steps=6)
    gs = synth.GradStream(w, device="cuda", seed=1)
    th_a = gs.theta0(); th_b = th_a.clone(); th_c = th_a.clone()
    a = B.Scape(w.numel, 3, 0.9, **w.hyper); a.set_layers(w.offsets(), comp)
    b = B.Scape(w.numel, 3, 0.9, **w.hyper); b.set_layers(w.offsets(), comp); b.set_workers(1, 0, [0] * len(sizes))
    c = B.Scape(w.numel, 3, 0.9, **w.hyper); c.set_workers(1, 0)          # flat top-k, split step
    d = B.Scape(w.numel, 3, 0.9, **w.hyper); th_d = th_a.clone()
    for t in range(6):
        g = gs.next()
        a.step(th_a, g)
        b.step_local(th_b, g); b.step_apply(th_b)
        c.step_local(th_c, g); c.step_apply(th_c)
        d.step(th_d, g)
        torch.cuda.synchronize()
        assert torch.equal(th_a, th_b) and torch.equal(th_c, th_d), t
        np.testing.assert_array_equal(a.mask_next(), b.mask_next())
        np.testing.assert_array_equal(c.mask_next(), d.mask_next())
        np.testing.assert_array_equal(a.idx_next(), b.idx_next())
        assert np.array_equal(a.moment().view(np.uint32), b.moment().view(np.uint32))
        assert np.array_equal(c.moment().view(np.uint32), d.moment().view(np.uint32))
    for h in (a, b, c, d):
        h.close()


def test_workers_api_errors(B):
    N = 4096
    h = B.Scape(N, 1, 0.9, **HYP)
    th = torch.zeros(N, device="cuda"); g = [torch.zeros(N, device="cuda")]
    with pytest.raises(B.ScapeError):
        h.set_workers(2, 0, [0, 1])              # owners need layers
    with pytest.raises(B.ScapeError):
        h.step_apply(th)                         # nothing in flight
    with pytest.raises(B.ScapeError):
        h.step_local(th, g)                      # set_workers first
    h.set_layers([0, 1000, N])
    with pytest.raises(B.ScapeError):
        h.set_workers(2, 2, [0, 1])              # rank out of range
    with pytest.raises(B.ScapeError):
        h.set_workers(2, 0, [0, 2])              # owner out of range
    with pytest.raises(B.ScapeError):
        h.set_workers(2, 0)                      # more than one worker needs owners
    h.set_workers(2, 0, [0, 1])
    with pytest.raises(B.ScapeError):
        h.step(th, g)                            # one of two workers: split step only
    with pytest.raises(B.ScapeError):
        h.set_layers([0, N])                     # not while it is one of several workers
    h.step_local(th, g)
    with pytest.raises(B.ScapeError):
        h.step_local(th, g)                      # apply first
    with pytest.raises(B.ScapeError):
        h.set_sparsity(0.5)
    sums, words = h.exchange_tensors()
    assert sums.numel() == N and words.numel() == N // 32      # first step: all-ones mask, dense payload
    h.step_apply(th)
    h.set_clip_grad(1.0)
    with pytest.raises(B.ScapeError):
        h.step_local(th, g)                      # clip_grad is not available in this mode
    h.close()


def test_step_workers_over_nccl_world_of_one(B, tmp_path):
    """The torch.distributed path itself (all-reduce on the handle's own buffers), world size 1."""
    import torch.distributed as dist
    if dist.is_initialized():
        pytest.skip("a process group already exists")
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    dist.init_process_group("nccl", init_method=f"file://{tmp_path}/pg", rank=0, world_size=1,
                            device_id=torch.device("cuda", torch.cuda.current_device()))
    try:
        sizes, comp = RAGGED
        w = synth.Workload("workers/nccl1", [(f"t{i}", n) for i, n in enumerate(sizes)], R=2, sparsity=0.9,
                           dist="gauss", rho=0.9, grad_dtype="f32", steps=5)
        gs = synth.GradStream(w, device="cuda", seed=2)
        th_a = gs.theta0(); th_b = th_a.clone()
        a = B.Scape(w.numel, 2, 0.9, **w.hyper); a.set_layers(w.offsets(), comp)
        b = B.Scape(w.numel, 2, 0.9, **w.hyper); b.set_layers(w.offsets(), comp); b.set_workers(1, 0, [0] * len(sizes))
        for t in range(5):
            g = gs.next()
            a.step(th_a, g)
            b.step_workers(th_b, g)
            torch.cuda.synchronize()
            assert torch.equal(th_a, th_b), t
            np.testing.assert_array_equal(a.mask_next(), b.mask_next())
        a.close(); b.close()
    finally:
        dist.destroy_process_group()


# ---- the exchange inside the library (scape_step_exchange) and the asynchronous refresh ----------
def test_exchange_plan_of_the_library_is_the_documented_one(B):
    sizes = [37, 3, 88, 1000, 13, 4000 + 7, 64, 32, 5]
    off = np.concatenate([[0], np.cumsum(sizes)]).tolist()
    for W, owner in ((2, [0, 1, 0, 1, 0, 1, 1, 0, 0]), (3, [2, 2, 0, 0, 1, 2, 2, 2, 1]), (2, [0] * 9), (1, [0] * 9)):
        h = B.Scape(off[-1], 1, 0.9, **HYP)
        h.set_layers(off, [1] * len(sizes))
        h.set_workers(W, 0, owner)
        ranges, shared = h.exchange_plan()
        want = workers.exchange_plan(off, owner, off[-1]) if W > 1 else ([(0, (off[-1] + 31) // 32, 0)], [])
        assert (ranges, shared) == (want[0], want[1]), (W, owner, ranges, shared, want)
        # every word is covered exactly once: by one range or as a shared word
        cover = np.zeros((off[-1] + 31) // 32, dtype=np.int32)
        for a, b, _ in ranges:
            cover[a:b] += 1
        cover[shared] += 1
        assert (cover == 1).all(), (W, owner)
        h.close()


@pytest.mark.parametrize("two_comms", [False, True])
def test_step_exchange_over_nccl_world_of_one(B, two_comms):
    """scape_step_exchange really calls NCCL (all-reduce of the sums, grouped broadcasts of the word
    ranges, all-reduce of the shared words); with a communicator of its own the mask part runs on the
    handle's stream.  One rank: the pair must equal scape_step to the bit."""
    sizes, comp = BIG
    w = synth.Workload("workers/nccl1", [(f"t{i}", n) for i, n in enumerate(sizes)], R=4, sparsity=0.99,
                       dist="t3", rho=0.9, grad_dtype="bf16", steps=8)
    gs = synth.GradStream(w, device="cuda", seed=2)
    th_a = gs.theta0(); th_b = th_a.clone()
    a = B.Scape(w.numel, 4, 0.99, **w.hyper); a.set_layers(w.offsets(), comp)
    b = B.Scape(w.numel, 4, 0.99, **w.hyper); b.set_layers(w.offsets(), comp); b.set_workers(1, 0, [0] * len(sizes))
    comm = B.scape_nccl_comm_create(1, 0, B.scape_nccl_unique_id())
    mcomm = B.scape_nccl_comm_create(1, 0, B.scape_nccl_unique_id()) if two_comms else None
    try:
        for t in range(8):
            g = gs.next()
            a.step(th_a, g)
            b.step_workers(th_b, g, comm=comm, mask_comm=mcomm)
            torch.cuda.synchronize()
            assert torch.equal(th_a, th_b), t
            np.testing.assert_array_equal(a.mask_next(), b.mask_next())
            np.testing.assert_array_equal(a.idx_next(), b.idx_next())
            assert np.array_equal(a.packed_mean().view(np.uint32), b.packed_mean().view(np.uint32))
    finally:
        a.close(); b.close()
        B.scape_nccl_comm_destroy(comm)
        if mcomm:
            B.scape_nccl_comm_destroy(mcomm)


_TWO_PROC = r'''
import os, sys, numpy as np, torch, torch.distributed as dist
sys.path.insert(0, os.environ["SCAPE_ROOT"]); sys.path.insert(0, os.path.join(os.environ["SCAPE_ROOT"], "tests"))
from oracle.scape_oracle import ScapeOracle
from paper_2607_01678_b200 import binding as B, synth, workers
dist.init_process_group("gloo")
rank, W = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)
sizes = [37, 3, 88, 1000, 13, 4000 + 7, 128 * 300 + 5, 64, 20011]
comp = [1, 1, 1, 1, 0, 1, 1, 1, 1]
Rl, s = 2, 0.9
w = synth.Workload("workers/2proc", [(f"t{i}", n) for i, n in enumerate(sizes)], R=W * Rl, sparsity=s, dist="t3", rho=0.9,
                   grad_dtype="f32", steps=8)
owner = workers.balance_layers(sizes, W)
gs = synth.GradStream(w, device="cuda", seed=3)            # same seed: every rank draws all W * Rl gradients, keeps its own
th = gs.theta0(); th_ora = th.cpu().numpy().copy()
ora = ScapeOracle(w.numel, W * Rl, s, **w.hyper); ora.set_layers(w.offsets(), comp); ora.set_workers(W, owner)
h = B.Scape(w.numel, Rl, s, **w.hyper); h.set_layers(w.offsets(), comp); h.set_workers(W, rank, owner)
for t in range(8):
    g = gs.next()
    h.step_workers(th, g[rank * Rl:(rank + 1) * Rl])          # torch.distributed path: plan-driven broadcasts over gloo
    ora.step(th_ora, [x.to(torch.float32).cpu().numpy() for x in g])
    torch.cuda.synchronize()
    assert np.array_equal(h.mask_next(), ora.mask()), (rank, t, "mask")
    assert np.array_equal(h.idx_last(), ora.idx()), (rank, t, "idx")
    assert np.array_equal(th.cpu().numpy().view(np.uint32), th_ora.view(np.uint32)), (rank, t, "theta")
    assert np.array_equal(h.packed_mean().view(np.uint32), ora.bbar().view(np.uint32)), (rank, t, "bbar")
    for q in range(Rl):
        assert np.array_equal(h.residual(q).view(np.uint32), ora.e(rank * Rl + q).view(np.uint32)), (rank, t, "e", q)
h.close()
dist.barrier()
if rank == 0:
    print("TWO_PROC_OK")
dist.destroy_process_group()
'''


def test_two_processes_on_one_gpu_over_gloo(tmp_path):
    """Two real processes, each with its own handle on cuda:0, exchanging through torch.distributed's
    gloo backend on CUDA tensors (NCCL refuses two ranks on one device): the word ranges from their
    owners, the shared words and the sums summed.  Every rank bit-exact against the oracle's workers
    reading, 8 steps."""
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "two_proc.py"
    script.write_text(_TWO_PROC)
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    env = dict(os.environ, SCAPE_ROOT=root)
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
                          "127.0.0.1", "--master-port", str(port), str(script)], capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0 and "TWO_PROC_OK" in res.stdout, res.stdout[-2000:] + res.stderr[-4000:]


def _busy(x, n):
    for _ in range(n):
        x.mul_(1.0000001)


@pytest.mark.parametrize("layered", [False, True])
def test_async_refresh_is_the_same_step(B, layered):
    """scape_set_async_refresh: stage 2 on the handle's own stream, the caller's stream free after the
    streaming kernel (other work enqueued between the steps); every output bit-exact against the oracle
    and against the in-stream form; accessors and the next step wait for the refresh by themselves."""
    sizes, comp = BIG
    w = synth.Workload("async", [(f"t{i}", n) for i, n in enumerate(sizes)], R=4, sparsity=0.99, dist="t3", rho=0.9,
                       grad_dtype="bf16", steps=10)
    gs = synth.GradStream(w, device="cuda", seed=7)
    th_a = gs.theta0(); th_b = th_a.clone(); th_o = th_a.cpu().numpy().copy()
    a = B.Scape(w.numel, 4, 0.99, **w.hyper)
    b = B.Scape(w.numel, 4, 0.99, **w.hyper); b.set_async_refresh(True)
    ora = ScapeOracle(w.numel, 4, 0.99, **w.hyper)
    if layered:
        for x in (a, b, ora):
            x.set_layers(w.offsets(), comp)
    other = torch.ones(1 << 24, device="cuda")
    side = torch.cuda.Stream()
    for t in range(10):
        g = gs.next()
        a.step(th_a, g)
        if t % 2:                                   # alternate the caller's stream: the dependency follows the handle
            with torch.cuda.stream(side):
                side.wait_stream(torch.cuda.current_stream())
                b.step(th_b, g)
                _busy(other, 3)
            torch.cuda.current_stream().wait_stream(side)
        else:
            b.step(th_b, g)
            _busy(other, 3)                         # the caller's next work overlaps the refresh
        ora.step(th_o, [to_np32(x) for x in g])
        if t in (2, 5, 9):
            np.testing.assert_array_equal(b.mask_next(), ora.mask())          # accessors join by themselves
            np.testing.assert_array_equal(b.idx_next(), np.nonzero(ora.mask())[0].astype(np.int32))
            torch.cuda.synchronize()
            assert torch.equal(th_a, th_b), t
            assert np.array_equal(th_b.cpu().numpy().view(np.uint32), th_o.view(np.uint32)), t
    torch.cuda.synchronize()
    assert b.last_kernel == "scape_fused_tma_kernel"
    # a captured step runs the refresh in-stream; replaying one rotation period stays exact
    b.join_refresh()
    torch.cuda.synchronize()
    ring = [gs.next() for _ in range(6)]
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr):
        for g in ring:
            b.step(th_b, g)
    for g in ring:
        a.step(th_a, g)
    gr.replay()
    torch.cuda.synchronize()
    assert torch.equal(th_a, th_b)
    a.close(); b.close()
