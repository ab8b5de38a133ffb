"""Parity at BASELINE.json's full size, in the launch configuration bench.py times — `-m gpu`.

The headline workload (Llama-1.8B-shaped shard: N = 1,775,239,168, R = 4 bf16 gradient buffers,
99 % sparsity) is far too large for the CPU oracle as a whole, so the step is checked
  (a) element by element on a SAMPLE of positions: the inputs of the sampled positions (theta, m,
      e^r, g^r, mask bit) are gathered before the step, handed to the oracle as a small problem
      of their own, and its outputs compared bit for bit with what the kernels wrote there; and
  (b) through properties that hold at any size: exactly k bits in M_t, ascending in-range index
      list, and the top-k property itself (every selected key >= every unselected key, ties to
      the lower index), evaluated with plain torch ops on the statistic |m~^0| rebuilt from the
      new e^0 and b^0 (pin P2).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.scape_oracle import ScapeOracle  # noqa: E402
from paper_2607_01678_b200 import synth  # noqa: E402

pytestmark = pytest.mark.gpu


def unpack_bits(words_t, n):
    """uint32 words (torch, device) -> bool tensor [n]"""
    shifts = torch.arange(32, device=words_t.device, dtype=torch.int32)
    bits = (words_t.to(torch.int32).unsqueeze(1) >> shifts) & 1
    return bits.reshape(-1)[:n].bool()


def get_mask_device(B, sc, which, N):
    nw = (N + 31) // 32
    buf = torch.empty(nw, dtype=torch.int32, device="cuda")
    B.scape_get(sc.h, which, 0, buf.data_ptr(), nw * 4, torch.cuda.current_stream().cuda_stream)
    return unpack_bits(buf, N)


def get_f32_device(B, sc, what, r, n):
    buf = torch.empty(n, dtype=torch.float32, device="cuda")
    B.scape_get(sc.h, what, r, buf.data_ptr(), n * 4, torch.cuda.current_stream().cuda_stream)
    return buf


def _workload(name):
    if name == "max_int32_index":
        # the largest shard the int32 index list allows (N < 2^31); odd, so the last chunk is ragged
        return synth.Workload(name, [("a", 2**30), ("b", 2**30 - 1)], R=3, sparsity=0.99, dist="t3", rho=0.9,
                              grad_dtype="bf16", steps=4), "scape_fused_tma_kernel", 80e9
    if name == "max_int32_index_R1":
        return synth.Workload(name, [("a", 2**31 - 1)], R=1, sparsity=0.999, dist="gauss", rho=0.9,
                              grad_dtype="f32", steps=4, per_tensor_scale=False), "scape_fused_step_kernel", 60e9
    if name == "llama1p8b_layers_split":
        # the same shard with the per-layer refresh (one top-k per tensor: 194 layers) and the split step of
        # the workers mode (a world of one): SURVEY.md §8(f) ranks 2 and 3 at full size
        return synth.workload("llama1p8b"), "scape_fused_tma_kernel", 130e9
    return synth.workload(name), "scape_fused_tma_kernel", 120e9


@pytest.mark.parametrize("name", ["llama1p8b", "llama1p8b_layers_split", "max_int32_index", "max_int32_index_R1"])
def test_fullsize_sampled_and_property_parity(name):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    w, want_kernel, need = _workload(name)
    free, _ = torch.cuda.mem_get_info()
    if free < need:
        pytest.skip(f"needs ~{need / 1e9:.0f} GB of free HBM")
    from paper_2607_01678_b200 import binding as B
    B.lib()
    N, R, k = w.numel, w.R, None
    gs = synth.GradStream(w, device="cuda", seed=0)
    theta = gs.theta0()
    sc = B.Scape(N, R, w.sparsity, **w.hyper)
    layered = name.endswith("_layers_split")
    offsets = w.offsets()
    if layered:
        sc.set_layers(offsets, w.compress_flags())
        sc.set_workers(1, 0, [0] * (len(offsets) - 1))

    def step(th, g):
        if layered:
            sc.step_local(th, g)
            sc.step_apply(th)
        else:
            sc.step(th, g)
    k = sc.k
    # reach the steady state bench.py times: dense first step, then sparse steps with m stored sparsely
    for _ in range(3):
        step(theta, gs.next())
    torch.cuda.synchronize()
    fast0, gen0 = sc.select_stats()

    # ---- sample positions: random ones plus every kind of edge (first/last element, tile and
    # chunk boundaries) plus a few hundred positions that ARE in the mask the step will use
    rng = np.random.default_rng(0)
    cur = get_mask_device(B, sc, B.SCAPE_MASK_NEXT, N)
    on_idx = torch.nonzero(cur).flatten()
    pick_on = on_idx[torch.from_numpy(rng.integers(0, on_idx.numel(), 600)).cuda()]
    edges = [0, 1, 127, 128, 1023, 1024, N - 1, N - 2, N - 1024, (N // 1024) * 1024 - 1, (N // 1024) * 1024]
    edges = [e for e in edges if 0 <= e < N]
    samp = torch.cat([torch.from_numpy(rng.integers(0, N, 3000)).cuda(), pick_on, torch.tensor(edges, device="cuda")])
    samp = torch.unique(samp)            # sorted ascending
    S = samp.numel()

    grads = gs.next()
    m_before = get_f32_device(B, sc, B.SCAPE_MOMENT, 0, N)[samp].cpu().numpy()
    e_before = [get_f32_device(B, sc, B.SCAPE_RESIDUAL, r, N)[samp].cpu().numpy() for r in range(R)]
    th_before = theta[samp].cpu().numpy()
    g_s = [g[samp].to(torch.float32).cpu().numpy() for g in grads]
    cur_s = cur[samp].cpu().numpy().astype(np.uint8)
    del cur, on_idx

    step(theta, grads)                   # the step under test (steady state, full size)
    torch.cuda.synchronize()
    fast1, gen1 = sc.select_stats()

    # ---- (a) sampled positions through the oracle, bit for bit
    ora = ScapeOracle(S, R, 0.5, **w.hyper)          # its own top-k is irrelevant here
    ora.set_m(m_before)
    for r in range(R):
        ora.set_e(r, e_before[r])
    ora.set_mask(cur_s)
    th_o = th_before.copy()
    ora.step(th_o, g_s)
    th_g = theta[samp].cpu().numpy()
    assert np.array_equal(th_g.view(np.uint32), th_o.view(np.uint32)), "theta differs on sampled positions"
    m_g = get_f32_device(B, sc, B.SCAPE_MOMENT, 0, N)[samp].cpu().numpy()
    assert np.array_equal(m_g.view(np.uint32), ora.m().view(np.uint32)), "m differs on sampled positions"
    e0_new = get_f32_device(B, sc, B.SCAPE_RESIDUAL, 0, N)
    for r in range(R):
        e_g = (e0_new if r == 0 else get_f32_device(B, sc, B.SCAPE_RESIDUAL, r, N))[samp].cpu().numpy()
        assert np.array_equal(e_g.view(np.uint32), ora.e(r).view(np.uint32)), f"e[{r}] differs on sampled positions"

    # ---- (b) properties at full size
    assert sc.count_last() == k and sc.count_next() == k
    nxt = get_mask_device(B, sc, B.SCAPE_MASK_NEXT, N)
    assert int(nxt.sum()) == k
    idx_next = torch.from_numpy(sc.idx_next()).cuda()
    assert idx_next.numel() == k and bool((idx_next[1:] > idx_next[:-1]).all()) and int(idx_next[-1]) < N
    assert bool(nxt[idx_next.long()].all())
    # statistic |m~^0|: new e^0 off the mask the step used, b^0 on it
    keys = e0_new.abs_()
    idx_last = torch.from_numpy(sc.idx_last()).cuda().long()
    b0 = get_f32_device(B, sc, B.SCAPE_PACKED, 0, k)
    keys[idx_last] = b0.abs()
    # ---- (a') the sparse buffer itself at the sampled on-mask positions: b^r and b- (l.9, l.10) sit at
    # packed position j with idx_last[j] = i; the small oracle's packed order is the sampled positions'
    on_s = torch.from_numpy(cur_s.astype(bool)).cuda()
    samp_on = samp[on_s]
    j_on = torch.searchsorted(idx_last, samp_on)
    assert bool((idx_last[j_on] == samp_on).all()), "a sampled on-mask position is missing from the index list"
    assert samp_on.numel() == ora.K_last and samp_on.numel() >= 300
    for r in range(R):
        b_g = (b0 if r == 0 else get_f32_device(B, sc, B.SCAPE_PACKED, r, k))[j_on].cpu().numpy()
        assert np.array_equal(b_g.view(np.uint32), ora.b(r).view(np.uint32)), f"b[{r}] differs on sampled on-mask positions"
    bb_g = get_f32_device(B, sc, B.SCAPE_PACKED_MEAN, 0, k)[j_on].cpu().numpy()
    assert np.array_equal(bb_g.view(np.uint32), ora.bbar().view(np.uint32)), "b-bar differs on sampled on-mask positions"

    def check_topk(keys_l, nxt_l, k_l):
        assert int(nxt_l.sum()) == k_l
        if k_l == keys_l.numel():
            return
        sel_min = keys_l[nxt_l].min()
        unsel_max = torch.where(nxt_l, torch.full_like(keys_l, -1.0), keys_l).max()
        assert float(sel_min) >= float(unsel_max), (float(sel_min), float(unsel_max))
        if float(sel_min) == float(unsel_max):       # tie class straddles the threshold: lower indices win
            tie = keys_l == sel_min
            last_sel = torch.nonzero(tie & nxt_l).flatten().max()
            first_unsel = torch.nonzero(tie & ~nxt_l).flatten().min()
            assert int(last_sel) < int(first_unsel)

    if layered:                                      # the top-k property inside every layer, exactly k_l each
        for l in range(len(offsets) - 1):
            a, b = offsets[l], offsets[l + 1]
            check_topk(keys[a:b], nxt[a:b], sc.layer_k(l))
        assert fast1 - fast0 + gen1 - gen0 == len(offsets) - 1      # counted per layer and step
    else:
        check_topk(keys, nxt, k)
        # the timed configuration: fast select route with the bulk-copy staged kernel
        assert fast1 - fast0 + gen1 - gen0 == 1
    assert sc.last_kernel == want_kernel
    sc.close()
    del theta, grads, keys, nxt, e0_new
    torch.cuda.empty_cache()
