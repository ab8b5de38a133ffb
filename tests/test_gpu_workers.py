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
