"""Parity of the per-layer refresh and of the sparsity schedule — `-m gpu`.

Same bar as test_gpu_parity.py: masks / indices / counts bit-exact against the oracle, fp32 state
within 1e-6 (and in fact to the bit), through the C-ABI.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.scape_oracle import ScapeOracle  # noqa: E402
from paper_2607_01678_b200 import synth  # noqa: E402
from test_gpu_parity import HYP, B, compare_step, load_state, to_np32  # noqa: E402,F401

pytestmark = pytest.mark.gpu


def make_pair(B, w, offsets=None, compress=None, sparsity=None):
    s = w.sparsity if sparsity is None else sparsity
    gpu = B.Scape(w.numel, w.R, s, **w.hyper)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(w.numel, w.R, s, **w.hyper)
    if offsets is not None:
        gpu.set_layers(offsets, compress)
        ora.set_layers(offsets, compress)
    return gpu, ora


def run(B, w, steps, offsets=None, compress=None, reload=False, seed=0, schedule=None):
    """Chained (or per-step reloaded) parity; `schedule(t)` = sparsity of step t's refresh."""
    R = w.R
    gs = synth.GradStream(w, device="cuda", seed=seed)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu, ora = make_pair(B, w, offsets, compress, sparsity=None if schedule is None else schedule(1))
    for t in range(1, steps + 1):
        grads = gs.next()
        if schedule is not None:
            gpu.set_sparsity(schedule(t))
            ora.set_sparsity(schedule(t))
        if reload:
            load_state(gpu, ora, R)
            th_gpu = torch.from_numpy(th_ora.copy()).cuda()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        compare_step(gpu, ora, th_gpu, th_ora, R, f"{w.name} step {t}")
        if offsets is not None:             # exactly k_l per layer
            mk = gpu.mask_next()
            for l in range(len(offsets) - 1):
                assert int(mk[offsets[l]:offsets[l + 1]].sum()) == gpu.layer_k(l), (t, l)
            assert gpu.k == int(mk.sum())
    stats = gpu.select_stats()
    gpu.close()
    return stats


LAYOUTS = {
    # name: (tensor sizes, compress flags)
    "aligned": ([128 * 40, 128 * 3, 128 * 100, 128 * 7], [1, 1, 1, 1]),
    "ragged": ([1000, 1, 5, 127, 129, 4096 + 3, 64, 20_000 + 11, 2], [1, 1, 1, 1, 1, 1, 0, 1, 1]),
    "norms": ([1024 * 48, 1024, 1024, 1024 * 16, 1024, 4096 * 12, 4096], [1, 0, 0, 1, 0, 1, 0]),
    "one": ([50_000 + 5], [1]),
    "all_uncompressed_but_one": ([300, 5000, 300], [0, 1, 0]),
}


@pytest.mark.parametrize("layout", sorted(LAYOUTS))
@pytest.mark.parametrize("R,s,gdt", [(1, 0.9, "f32"), (4, 0.99, "bf16"), (3, 0.5, "f32")])
def test_layers_chained_parity(B, layout, R, s, gdt):
    sizes, comp = LAYOUTS[layout]
    w = synth.Workload(f"layers/{layout}", [(f"t{i}", n) for i, n in enumerate(sizes)], R=R, sparsity=s,
                       dist="t3", rho=0.9, grad_dtype=gdt, steps=8)
    run(B, w, steps=8, offsets=w.offsets(), compress=comp, seed=len(sizes) + R)


@pytest.mark.parametrize("layout", ["ragged", "norms"])
def test_layers_reload_parity(B, layout):
    sizes, comp = LAYOUTS[layout]
    w = synth.Workload(f"layers-reload/{layout}", [(f"t{i}", n) for i, n in enumerate(sizes)], R=2, sparsity=0.95,
                       dist="gauss", rho=0.9, grad_dtype="f32", steps=5)
    run(B, w, steps=5, offsets=w.offsets(), compress=comp, reload=True, seed=3)


def test_layers_take_the_candidate_route_in_steady_state(B):
    sizes = [128 * 600, 128 * 900 + 17, 128 * 300, 4096, 128 * 1200]
    w = synth.Workload("layers/steady", [(f"t{i}", n) for i, n in enumerate(sizes)], R=4, sparsity=0.99,
                       dist="t4", rho=0.9, grad_dtype="f32", steps=30)
    fast, general = run(B, w, steps=30, offsets=w.offsets(), compress=[1, 1, 1, 0, 1], seed=11)
    assert fast + general == 30 * len(sizes)
    assert fast >= 20 * len(sizes), (fast, general)      # the per-layer brackets hold once predicted


def test_layers_model_shaped_with_uncompressed_norms(B):
    """GPT-345M-shaped tensor list /256 with LayerNorm / bias tensors added (not compressed,
    PAPER.md:286), one layer per tensor."""
    base = synth.workload("gpt345m", div=256)
    tensors = []
    for name, n in base.tensors:
        tensors.append((name, n))
        if name.endswith(("qkv", "fc")):
            tensors += [(name + ".bias", 1024 if name.endswith("qkv") else 4096), (name + ".ln_w", 1024)]
    w = synth.Workload("gpt345m/div256+norms", tensors, R=4, sparsity=0.99, dist="t4", rho=0.9, grad_dtype="f32", steps=6)
    comp = w.compress_flags()
    assert 0 in comp and 1 in comp
    run(B, w, steps=6, offsets=w.offsets(), compress=comp, seed=2)


def test_layers_crafted_ties_across_and_inside_layers(B):
    rng = np.random.default_rng(0)
    offsets = [0, 700, 1403, 5000, 9000 + 13]
    N, R, s = offsets[-1], 2, 0.9
    w = synth.Workload("layers/ties", [("x", N)], R=R, sparsity=s, dist="gauss", rho=0.0, grad_dtype="f32", steps=6)
    gpu, ora = make_pair(B, w, offsets, [1, 1, 0, 1])
    th_ora = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th_gpu = torch.from_numpy(th_ora.copy()).cuda()
    for t in range(1, 7):
        base = (rng.integers(-3, 4, N) * 0.25).astype(np.float32)
        base[:300] = 0.0
        if t == 4:
            base[:] = 0.5
        if t == 5:
            base[:] = 0.0
        grads = [torch.from_numpy(base.copy()).cuda() for _ in range(R)]
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [base.copy() for _ in range(R)])
        compare_step(gpu, ora, th_gpu, th_ora, R, f"layer ties step {t}")
    gpu.close()


def warmup(t, d_final, T_w):
    """Exponential density warm-up 1 -> d_final over T_w steps (PAPER.md:279 gives only the shape)."""
    return 1.0 - max(d_final, d_final ** (t / T_w))


@pytest.mark.parametrize("layered", [False, True])
def test_density_warmup_schedule(B, layered):
    sizes = [128 * 200 + 9, 640, 128 * 333, 128 * 150 + 100]
    w = synth.Workload("warmup", [(f"t{i}", n) for i, n in enumerate(sizes)], R=3, sparsity=0.0, dist="t4", rho=0.9,
                       grad_dtype="bf16", steps=16)
    off = w.offsets() if layered else None
    comp = [1, 0, 1, 1] if layered else None
    # step 1 refreshes at density 1 ** ... < 1 already; the mask sizes shrink every step up to step 10
    run(B, w, steps=16, offsets=off, compress=comp, seed=4, schedule=lambda t: warmup(t, 0.02, 10))


def test_sparsity_can_go_back_to_dense_and_up_again(B):
    w = synth.Workload("updown", [("a", 30_000 + 7)], R=2, sparsity=0.9, dist="gauss", rho=0.9, grad_dtype="f32", steps=9)
    sched = {1: 0.9, 2: 0.9, 3: 0.0, 4: 0.0, 5: 0.5, 6: 0.99, 7: 0.99, 8: 0.2, 9: 0.9}
    run(B, w, steps=9, seed=6, schedule=lambda t: sched[t])


def test_layers_can_change_between_steps(B):
    """scape_set_layers in the middle of a run (the cached select graphs hold the old layer tables' addresses and
    item counts and must go): layout A, another layout, the flat top-k, layout A again; every step against the oracle."""
    w = synth.Workload("relayer", [("a", 128 * 700 + 77)], R=2, sparsity=0.9, dist="gauss", rho=0.9, grad_dtype="f32", steps=18)
    N = w.numel
    lay_a = [0, 1000, 1000 + 128 * 300 + 5, 60_000, N]
    lay_b = [0, 128 * 100, 128 * 100 + 3, 20_000, 20_001, 70_000 + 9, N]
    plan = {1: (lay_a, [1, 1, 0, 1]), 6: (lay_b, [1, 0, 1, 1, 1, 1]), 11: None, 14: (lay_a, [1, 1, 0, 1])}
    gs = synth.GradStream(w, device="cuda", seed=9)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu, ora = make_pair(B, w)
    for t in range(1, 19):
        if t in plan:
            if plan[t] is None:                      # flat: one top-k over the shard = one compressed layer
                gpu.clear_layers()
                ora.set_layers([0, N], [1])
            else:
                gpu.set_layers(*plan[t])
                ora.set_layers(*plan[t])
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        compare_step(gpu, ora, th_gpu, th_ora, w.R, f"relayer step {t}")
    gpu.close()


def test_set_layers_api_errors(B):
    gpu = B.Scape(1000, 1, 0.9, **HYP)
    for bad in ([0, 500], [1, 1000], [0, 500, 500, 1000], [0, 600, 400, 1000]):
        with pytest.raises(B.ScapeError):
            gpu.set_layers(bad)
    with pytest.raises(B.ScapeError):
        gpu.set_sparsity(1.0)
    gpu.set_layers([0, 10, 1000], [0, 1])
    assert gpu.layer_k(0) == 10 and gpu.layer_k(1) == 990 - int(np.floor(0.9 * 990)) and gpu.k == 10 + gpu.layer_k(1)
    gpu.clear_layers()
    assert gpu.k == 100
    gpu.close()


@pytest.mark.parametrize("n_tiles,extra", [(149, 77), (150, 0), (151, 1023), (296 * 4 + 2, 5)])
def test_grouped_staged_kernel_short_last_group(B, n_tiles, extra):
    """Per-layer refresh runs the grouped form of the staged kernel (groups of 4 tiles, mask words by bulk
    copy): shards whose number of full tiles is not a multiple of 4, with and without a ragged tail, layer
    boundaries inside tiles and chunks, an uncompressed layer; 7 chained steps against the oracle."""
    N = n_tiles * 1024 + extra
    sizes = [1024 * 37 + 5, 333, 1024 * 60 - 338]
    sizes.append(N - sum(sizes))
    w = synth.Workload(f"grouped/{n_tiles}+{extra}", [(f"t{i}", n) for i, n in enumerate(sizes)], R=4, sparsity=0.99,
                       dist="t3", rho=0.9, grad_dtype="bf16", steps=7)
    gs = synth.GradStream(w, device="cuda", seed=11)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu, ora = make_pair(B, w, w.offsets(), [1, 0, 1, 1])
    for t in range(1, 8):
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        compare_step(gpu, ora, th_gpu, th_ora, 4, f"{w.name} step {t}")
        if t >= 3:
            assert gpu.last_kernel == "scape_fused_tma_kernel"
    gpu.close()
