"""Parity of the CUDA path (through the C-ABI) against the CPU oracle — `-m gpu`.

Bar (BASELINE.json north_star): from identical state each step, masks / indices / counts
bit-exact (ties to the lower index) and fp32 theta, m, e within max relative error 1e-6; after
100 chained steps theta within 1e-4 relative and masks agreeing on >= 99.99 % of entries.
With the pinned operation order the expectation is 0 ulp, which the tests also report.
"""
import json
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.scape_oracle import ScapeOracle  # noqa: E402
from paper_2607_01678_b200 import synth  # noqa: E402

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
HYP = dict(beta1=0.9, beta2=0.95, eps=1e-8, lr=1e-3, wd=0.1)
REL_TOL = 1e-6          # north_star: per-step max relative error on fp32 state


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01678_b200 import binding
    binding.lib()       # raises if libscape.so is missing: no fallback
    return binding


def max_rel(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    den = np.maximum(np.abs(a), np.abs(b))
    with np.errstate(invalid="ignore", divide="ignore"):
        r = np.where(den > 0, np.abs(a - b) / den, 0.0)
    return float(r.max()) if r.size else 0.0


def assert_close(a, b, what, tol=REL_TOL):
    assert a.shape == b.shape, what
    r = max_rel(a, b)
    assert r <= tol, f"{what}: max rel err {r:.3e} > {tol}"


def to_np32(g):
    return g.detach().to(torch.float32).cpu().numpy()


def load_state(gpu, ora, R, moment=True):
    """Copy the oracle's state (m, e^r, mask the coming step uses, t) into the CUDA handle.
    moment=False leaves m as the handle carries it (sparsely, as the previous step's packed mean:
    loading a dense m would switch the next step to the dense-m kernel variant); compare_step has
    already shown it equal to the oracle's to the bit."""
    if moment:
        gpu.set_moment(ora.m())
    for r in range(R):
        gpu.set_residual(r, ora.e(r))
    gpu.set_mask_next(ora.mask())
    gpu.set_step_count(ora.t)


def compare_step(gpu, ora, th_gpu, th_ora, R, tag, exact=True):
    """Everything one step produces, GPU vs oracle."""
    K = ora.K_last
    assert gpu.count_last() == K, tag
    np.testing.assert_array_equal(gpu.idx_last(), ora.idx(), err_msg=f"{tag} idx_last")
    mk_g, mk_o = gpu.mask_next(), ora.mask()
    np.testing.assert_array_equal(mk_g, mk_o, err_msg=f"{tag} mask_next")
    assert gpu.count_next() == int(mk_o.sum()), tag
    np.testing.assert_array_equal(gpu.idx_next(), np.nonzero(mk_o)[0].astype(np.int32), err_msg=f"{tag} idx_next")
    th = th_gpu.cpu().numpy()
    assert_close(th, th_ora, f"{tag} theta")
    assert_close(gpu.moment(), ora.m(), f"{tag} m")
    for r in range(R):
        assert_close(gpu.residual(r), ora.e(r), f"{tag} e[{r}]")
        assert_close(gpu.packed(r), ora.b(r), f"{tag} b[{r}]")
    assert_close(gpu.packed_mean(), ora.bbar(), f"{tag} bbar")
    if exact:   # the pinned operation order makes the two sides agree to the bit
        assert np.array_equal(th.view(np.uint32), th_ora.view(np.uint32)), f"{tag} theta not bit-exact"
        assert np.array_equal(gpu.moment().view(np.uint32), ora.m().view(np.uint32)), f"{tag} m not bit-exact"
        for r in range(R):
            assert np.array_equal(gpu.residual(r).view(np.uint32), ora.e(r).view(np.uint32)), f"{tag} e[{r}] not bit-exact"


def run_reload_parity(B, w, steps, seed=0, hyp=HYP, setup=None, reload_moment=True, kernels=None):
    """Per-step parity 'when both start from identical state each step'.
    kernels: optional {step number: expected scape_last_kernel}."""
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=seed)
    th0 = gs.theta0()
    gpu = B.Scape(N, R, w.sparsity, **hyp)
    gpu.keep_dense_pack(True)
    if setup is not None:
        setup(gpu)
    ora = ScapeOracle(N, R, w.sparsity, **hyp)
    assert gpu.k == ora.k
    th_ora = th0.cpu().numpy().copy()
    for t in range(1, steps + 1):
        grads = gs.next()
        load_state(gpu, ora, R, moment=reload_moment)
        th_gpu = torch.from_numpy(th_ora.copy()).cuda()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        compare_step(gpu, ora, th_gpu, th_ora, R, f"{w.name} step {t}")
        if kernels and t in kernels:
            assert gpu.last_kernel == kernels[t], (t, gpu.last_kernel)
    gpu.close()


# ------------------------------------------------------------------------------------------
def test_config1_pr1_per_step_parity(B):
    """BASELINE.json configs[0]: N = 2^20, R = 2, s = 0.9, 10 steps, seed 0."""
    run_reload_parity(B, synth.workload("pr1"), steps=10, seed=0)


def test_config1_pr1_chained_parity_is_exact(B):
    """Same config, no reload: the GPU carries its own state for 10 steps."""
    w = synth.workload("pr1")
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=0)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu = B.Scape(N, R, w.sparsity, **HYP)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(N, R, w.sparsity, **HYP)
    for t in range(1, 11):
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        compare_step(gpu, ora, th_gpu, th_ora, R, f"chained step {t}")
    fast, general = gpu.select_stats()
    assert fast + general == 10 and general >= 1      # step 1 (all-ones mask) is always general
    assert fast >= 5, (fast, general)                 # the predicted bracket holds in steady state
    gpu.close()


def test_chained_100_steps(B):
    """north_star: after 100 chained steps theta within 1e-4 relative, masks agree >= 99.99 %."""
    w = synth.Workload("chain100", [("flat", 300_000 + 77)], R=3, sparsity=0.99, dist="t4", rho=0.9,
                       grad_dtype="f32", steps=100, per_tensor_scale=False, const_scale=1e-3)
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=5)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu = B.Scape(N, R, w.sparsity, **HYP)
    ora = ScapeOracle(N, R, w.sparsity, **HYP)
    for _ in range(100):
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
    agree = float((gpu.mask_next() == ora.mask()).mean())
    assert agree >= 0.9999, agree
    fast, general = gpu.select_stats()
    assert fast + general == 100 and fast >= 80, (fast, general)
    assert_close(th_gpu.cpu().numpy(), th_ora, "theta after 100 chained steps", tol=1e-4)
    assert_close(gpu.moment(), ora.m(), "m after 100 chained steps", tol=1e-4)
    gpu.close()


@pytest.mark.parametrize("N,R,s,gdt", [
    (1, 1, 0.0, "f32"), (3, 2, 0.5, "f32"), (127, 1, 0.9, "f32"), (128, 2, 0.9, "bf16"),
    (129, 3, 0.99, "f32"), (1000, 4, 0.999, "bf16"), (4099, 5, 0.9, "f32"), (128 * 37 + 5, 8, 0.99, "bf16"),
    (131072 + 1, 2, 0.5, "f32"), (200_003, 7, 0.9, "f32"), (150_000, 6, 0.0, "bf16"), (40_000, 4, 0.25, "f32"),
])
def test_ragged_sizes_replica_counts_and_dtypes(B, N, R, s, gdt):
    w = synth.Workload(f"ragged{N}", [("a", N // 2), ("b", N - N // 2)], R=R, sparsity=s, dist="t3", rho=0.9,
                       grad_dtype=gdt, steps=4)
    run_reload_parity(B, w, steps=4, seed=N)


@pytest.mark.parametrize("name,div", [("gpt345m", 256), ("llama500m", 256), ("llama1p8b", 512)])
def test_scaled_model_shaped_shards(B, name, div):
    """Configs 2-4 with every tensor `div` times smaller (same structure, scales, distributions).
    Loading a dense m makes every sparse step take the register-staged kernel with dense m in."""
    w = synth.workload(name, div=div)
    run_reload_parity(B, w, steps=3, seed=1, kernels={2: "scape_fused_step_kernel", 3: "scape_fused_step_kernel"})


@pytest.mark.parametrize("name,div,sparsity", [("gpt345m", 256, None), ("llama500m", 256, 0.9), ("llama500m", 256, None),
                                               ("llama1p8b", 512, None)])
def test_scaled_model_shaped_shards_reload_keeps_m_sparse(B, name, div, sparsity):
    """The same per-step reload (e^r, mask, theta, t from the oracle) but m stays as the handle keeps it
    in steady state -- the previous step's packed mean -- so from step 3 on the step under test is the
    steady-state instantiation bench.py times (m gathered through the previous mask)."""
    w = synth.workload(name, div=div, sparsity=sparsity)
    steady = STEADY_KERNEL[name]
    run_reload_parity(B, w, steps=5, seed=2, reload_moment=False,
                      kernels={1: "scape_fused_step_kernel", 2: "scape_fused_step_kernel", 3: steady, 4: steady, 5: steady})


# streaming kernel each model-shaped workload takes in steady state (what bench.py times)
STEADY_KERNEL = {"gpt345m": "scape_fused_tma_kernel", "llama500m": "scape_fused_step_kernel", "llama1p8b": "scape_fused_tma_kernel"}


@pytest.mark.parametrize("name,div,sparsity", [("llama1p8b", 512, None), ("gpt345m", 128, None), ("llama500m", 128, 0.9),
                                               ("llama500m", 128, None)])
def test_headline_instantiations_chained_element_by_element(B, name, div, sparsity):
    """The exact instantiations bench.py times (llama1p8b: staged kernel <bf16, R = 4>, flat select;
    gpt345m: <f32, 4>; llama500m: <f32, 8> at 90 % and 99 %), chained for 8 steps WITHOUT reloading any
    state, every output of every step compared with the oracle element by element: masks, index lists,
    theta, m, e^r, b^r, b-bar.  N = 2.8-3.9 M: thousands of tiles per CTA ring and a ragged tail."""
    w = synth.workload(name, div=div, sparsity=sparsity)
    w.tensors.append(("ragged_tail", 1024 * 3 + 128 * 2 + 77))       # chunks past the last full tile, the last one ragged
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=11)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu = B.Scape(N, R, w.sparsity, **w.hyper)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(N, R, w.sparsity, **w.hyper)
    for t in range(1, 9):
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        compare_step(gpu, ora, th_gpu, th_ora, R, f"{w.name} chained step {t}")
        if t >= 3:
            assert gpu.last_kernel == STEADY_KERNEL[name], (t, gpu.last_kernel)
    fast, general = gpu.select_stats()
    assert fast + general == 8 and fast >= 3, (fast, general)
    gpu.close()


def test_crafted_ties_and_zeros(B):
    """Quantised gradients: many exactly equal |m~| straddle the threshold; zero regions."""
    rng = np.random.default_rng(0)
    N, R, s = 10_000 + 13, 2, 0.9
    gpu = B.Scape(N, R, s, **HYP)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(N, R, s, **HYP)
    th_ora = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th_gpu = torch.from_numpy(th_ora.copy()).cuda()
    for t in range(1, 7):
        base = (rng.integers(-3, 4, N) * 0.25).astype(np.float32)     # 7 distinct values
        base[: N // 3] = 0.0                                          # a zero region
        if t == 4:
            base[:] = 0.5                                             # every key equal
        if t == 5:
            base[:] = 0.0                                             # all-zero gradients
        grads = [torch.from_numpy(base.copy()).cuda() for _ in range(R)]
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [base.copy() for _ in range(R)])
        compare_step(gpu, ora, th_gpu, th_ora, R, f"ties step {t}")
    gpu.close()


def test_general_route_when_the_recovery_pass_overflows(B):
    """All-zero gradients on a shard of 2^20: every key is 0, the sampled bracket makes every key a candidate, the
    candidate list overflows, and the plain general route (radix passes over every key) must take over; ties go to
    the lowest indices.  Then ordinary gradients again (recovery pass, then the predicted bracket)."""
    N, R, s = (1 << 20) + 77, 1, 0.9
    rng = np.random.default_rng(3)
    gpu = B.Scape(N, R, s, **HYP)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(N, R, s, **HYP)
    th_ora = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th_gpu = torch.from_numpy(th_ora.copy()).cuda()
    for t in range(1, 8):
        base = np.zeros(N, np.float32) if t <= 3 else (1e-3 * rng.standard_normal(N)).astype(np.float32)
        gpu.step(th_gpu, [torch.from_numpy(base.copy()).cuda()])
        ora.step(th_ora, [base.copy()])
        compare_step(gpu, ora, th_gpu, th_ora, R, f"overflow step {t}")
    fast, general = gpu.select_stats()
    rec = gpu.select_recovered()
    assert general - rec >= 2 and rec >= 1, (fast, general, rec)
    gpu.close()


def test_p9_worked_example_on_gpu(B):
    with open(os.path.join(HERE, "golden", "p9_worked_example.json")) as f:
        G = json.load(f)
    gpu = B.Scape(G["N"], G["R"], G["sparsity"], G["beta1"], G["beta2"], G["eps"], G["lr"], G["wd"])
    gpu.keep_dense_pack(True)
    assert gpu.k == G["k"]
    th = torch.tensor(G["theta0"], dtype=torch.float32, device="cuda")
    for s in G["steps"]:
        g = [torch.tensor(s[k], dtype=torch.float32, device="cuda") * G["grad_scale"] for k in ("g0", "g1")]
        gpu.step(th, g)
        np.testing.assert_array_equal(gpu.idx_last(), np.array(s["cur"], np.int32))
        np.testing.assert_array_equal(np.nonzero(gpu.mask_next())[0], np.array(s["next"]))
        np.testing.assert_array_equal(gpu.packed(0), np.array(s["b0"], np.float32))
        np.testing.assert_array_equal(gpu.packed(1), np.array(s["b1"], np.float32))
        np.testing.assert_array_equal(gpu.residual(0), np.array(s["e0_after"], np.float32))
        np.testing.assert_array_equal(gpu.residual(1), np.array(s["e1_after"], np.float32))
        np.testing.assert_array_equal(gpu.moment(), np.array(s["m_after"], np.float32))
        np.testing.assert_allclose(th.cpu().numpy(), np.array(s["theta_after"], np.float32), rtol=1e-6, atol=0)
    gpu.close()


def test_sparsity_zero_stays_dense(B):
    w = synth.Workload("dense", [("flat", 50_000 + 3)], R=2, sparsity=0.0, dist="gauss", rho=0.5,
                       grad_dtype="f32", steps=3, per_tensor_scale=False)
    run_reload_parity(B, w, steps=3)


def test_api_errors(B):
    import ctypes
    L = B.lib()
    assert not L.scape_create(0, 1, 0.5, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert "shard_numel" in B.scape_last_error()
    assert not L.scape_create(1 << 31, 1, 0.5, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 0, 0.5, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 9, 0.5, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 1, 1.0, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 1, 0.5, 1.0, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 1, 0.5, 0.9, 0.95, -1.0, 1e-3, 0.1)
    assert not L.scape_create(16, 1, float("nan"), 0.9, 0.95, 1e-8, 1e-3, 0.1)
    g = B.Scape(1024, 2, 0.9)
    th = torch.zeros(1024 + 4, device="cuda")
    gr = [torch.zeros(1024, device="cuda") for _ in range(2)]
    arr = (ctypes.c_void_p * 2)(*[x.data_ptr() for x in gr])
    assert L.scape_step(g.h, th.data_ptr() + 4, arr, None) == B.SCAPE_EINVAL      # misaligned param
    assert "aligned" in B.scape_last_error()
    assert L.scape_step(None, th.data_ptr(), arr, None) == B.SCAPE_EINVAL
    assert L.scape_step(g.h, None, arr, None) == B.SCAPE_EINVAL
    assert g.t == 0                                                              # state unchanged
    with pytest.raises(B.ScapeError):
        g.packed(0)                                                              # no step has run yet
    with pytest.raises(B.ScapeError):
        B.scape_set_grad_dtype(g.h, 7)
    L.scape_destroy(None)                                                        # NULL is a no-op
    g.close()


def test_step_host_matches_device_step(B):
    w = synth.Workload("host", [("flat", 70_001)], R=2, sparsity=0.9, dist="gauss", rho=0.9,
                       grad_dtype="bf16", steps=3, per_tensor_scale=False)
    gs = synth.GradStream(w, device="cuda", seed=3)
    th_d = gs.theta0()
    th_h = th_d.cpu().pin_memory()
    a, b = B.Scape(w.numel, w.R, w.sparsity), B.Scape(w.numel, w.R, w.sparsity)
    for _ in range(3):
        grads = gs.next()
        a.step(th_d, grads)
        b.step_host(th_h, [g.cpu().pin_memory() for g in grads])
        torch.cuda.synchronize()
        assert torch.equal(th_d.cpu(), th_h)
        np.testing.assert_array_equal(a.mask_next(), b.mask_next())
    a.close()
    b.close()


@pytest.mark.parametrize("R,gdt,s", [(4, "bf16", 0.99), (2, "f32", 0.9), (8, "f32", 0.99)])
def test_step_host_pipeline_in_parts(B, R, gdt, s):
    """scape_step_host on a shard large enough to be pipelined in 16 parts (upload / sub-range launch of the
    streaming kernel / download, both kernels): every step equal to scape_step on device buffers -- theta, the
    mask, the index list, b-, b^r and the residuals -- and to the oracle on the last step."""
    n = 148 * 2 * 16 * 1024 + 3 * 1024 + 77                # just above the pipeline's threshold, ragged tail
    w = synth.Workload("hostparts", [("a", n // 3), ("b", n - n // 3)], R=R, sparsity=s, dist="t3", rho=0.9, grad_dtype=gdt, steps=6)
    gs = synth.GradStream(w, device="cuda", seed=8)
    th_d = gs.theta0()
    th_h = th_d.cpu().pin_memory()
    th_o = th_d.cpu().numpy().copy()
    a, b = B.Scape(w.numel, R, s, **w.hyper), B.Scape(w.numel, R, s, **w.hyper)
    ora = ScapeOracle(w.numel, R, s, **w.hyper)
    for t in range(6):
        grads = gs.next()
        a.step(th_d, grads)
        b.step_host(th_h, [g.cpu().pin_memory() for g in grads])
        ora.step(th_o, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        assert torch.equal(th_d.cpu(), th_h), t
        np.testing.assert_array_equal(a.mask_next(), b.mask_next())
        np.testing.assert_array_equal(a.idx_next(), b.idx_next())
        assert np.array_equal(a.packed_mean().view(np.uint32), b.packed_mean().view(np.uint32)), t
        for r in range(R):
            assert np.array_equal(a.residual(r).view(np.uint32), b.residual(r).view(np.uint32)), (t, r)
            if t > 0:
                assert np.array_equal(a.packed(r).view(np.uint32), b.packed(r).view(np.uint32)), (t, r)
    assert np.array_equal(th_h.numpy().view(np.uint32), th_o.view(np.uint32))
    np.testing.assert_array_equal(b.mask_next(), ora.mask())
    a.close()
    b.close()


@pytest.mark.parametrize("R,gdt", [(2, "f32"), (1, "bf16")])
def test_step_host_pipeline_with_the_first_digit_histogram(B, R, gdt):
    """The pipelined scape_step_host on the register-staged kernel at N >= 2^24: every part's launch adds its
    candidates' first-digit histogram to the global one; results equal to scape_step on device buffers."""
    n = (1 << 24) + 5 * 1024 + 33
    w = synth.Workload("hosthist", [("a", n)], R=R, sparsity=0.9, dist="t3", rho=0.9, grad_dtype=gdt, steps=6)
    gs = synth.GradStream(w, device="cuda", seed=5)
    th_d = gs.theta0()
    th_h = th_d.cpu().pin_memory()
    a, b = B.Scape(n, R, 0.9, **w.hyper), B.Scape(n, R, 0.9, **w.hyper)
    for t in range(6):
        g = gs.next()
        a.step(th_d, g)
        b.step_host(th_h, [x.cpu().pin_memory() for x in g])
        torch.cuda.synchronize()
        assert torch.equal(th_d.cpu(), th_h), t
        np.testing.assert_array_equal(a.mask_next(), b.mask_next())
        np.testing.assert_array_equal(a.idx_next(), b.idx_next())
        assert np.array_equal(a.packed_mean().view(np.uint32), b.packed_mean().view(np.uint32)), t
    assert b.select_stats()[0] >= 2
    a.close()
    b.close()


def test_first_radix_digit_made_by_the_streaming_kernel(B):
    """From 2^24 parameters on, the register-staged kernel histograms the candidates' first radix digit as it
    flushes them and the select skips its first pass over the candidate list: 8 chained steps, every buffer
    against the oracle, and the fast route must have been taken once the bracket exists."""
    n = (1 << 24) + 4099
    w = synth.Workload("fusedhist", [("a", n // 2 + 17), ("b", n - n // 2 - 17)], R=1, sparsity=0.9, dist="t3", rho=0.9,
                       grad_dtype="f32", steps=8)
    gs = synth.GradStream(w, device="cuda", seed=12)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu = B.Scape(w.numel, 1, 0.9, **w.hyper)
    gpu.keep_dense_pack(True)                      # compare_step also reads b^r of the dense first step
    ora = ScapeOracle(w.numel, 1, 0.9, **w.hyper)
    for t in range(1, 9):
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        torch.cuda.synchronize()
        compare_step(gpu, ora, th_gpu, th_ora, 1, f"fusedhist step {t}")
    fast, general = gpu.select_stats()
    assert fast >= 5, (fast, general)
    assert gpu.last_kernel == "scape_fused_step_kernel"
    gpu.close()


def test_cuda_graph_capture_of_a_step(B):
    """scape_step allocates nothing and never synchronises, so it can be captured."""
    w = synth.Workload("graph", [("flat", 100_000)], R=2, sparsity=0.9, dist="gauss", rho=0.9,
                       grad_dtype="f32", steps=4, per_tensor_scale=False)
    gs = synth.GradStream(w, device="cuda", seed=4)
    th = gs.theta0()
    th2 = th.clone()
    ref, cap = B.Scape(w.numel, w.R, w.sparsity), B.Scape(w.numel, w.R, w.sparsity)
    grads = gs.next()
    for sc, p in ((ref, th), (cap, th2)):       # step 1 (dense) and 2 eagerly on both
        sc.step(p, grads)
        sc.step(p, grads)
    # steps 3 and 4 use different internal buffers (mask double buffer): capture both
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            cap.step(th2, grads)
            cap.step(th2, grads)
    torch.cuda.current_stream().wait_stream(s)
    graph.replay()
    ref.step(th, grads)
    ref.step(th, grads)
    torch.cuda.synchronize()
    assert torch.equal(th, th2)
    np.testing.assert_array_equal(ref.mask_next(), cap.mask_next())
    ref.close()
    cap.close()


def test_cuda_graph_replays_a_whole_rotation_period(B):
    """include/scape.h: the handle rotates three mask slots and two packed-mean buffers and bakes their
    addresses into the launches, so a graph must hold a multiple of SCAPE_GRAPH_PERIOD = 6 steady-state
    steps.  Capture 6 steps once, replay the graph three times on fresh gradients (18 steps) and compare
    with 18 eager steps of a second handle and with the oracle."""
    w = synth.Workload("graph6", [("a", 200_000), ("b", 131_072 + 333)], R=3, sparsity=0.99, dist="t4", rho=0.9,
                       grad_dtype="f32", steps=24)
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=8)
    th_ref = gs.theta0()
    th_cap = th_ref.clone()
    th_ora = th_ref.cpu().numpy().copy()
    ref, cap = B.Scape(N, R, w.sparsity, **HYP), B.Scape(N, R, w.sparsity, **HYP)
    ora = ScapeOracle(N, R, w.sparsity, **HYP)
    static = [[torch.empty(N, device="cuda") for _ in range(R)] for _ in range(6)]     # the graph's gradient buffers

    def feed(i):
        grads = gs.next()
        for dst, src in zip(static[i], grads):
            dst.copy_(src)
        return grads

    for i in range(4):                                   # dense step, dense-m step, two steady-state steps: eagerly
        grads = feed(i)
        ref.step(th_ref, grads)
        cap.step(th_cap, static[i])
        ora.step(th_ora, [to_np32(g) for g in grads])
    assert cap.last_kernel == "scape_fused_tma_kernel"
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            for i in range(6):
                cap.step(th_cap, static[i])
    torch.cuda.current_stream().wait_stream(s)
    for rep in range(3):
        for i in range(6):
            grads = feed(i)
            ref.step(th_ref, grads)
            ora.step(th_ora, [to_np32(g) for g in grads])
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(th_ref, th_cap), f"replay {rep + 1}: theta of the replayed graph differs from eager steps"
        np.testing.assert_array_equal(cap.mask_next(), ora.mask(), err_msg=f"replay {rep + 1} mask")
        np.testing.assert_array_equal(cap.idx_next(), np.nonzero(ora.mask())[0].astype(np.int32))
        assert np.array_equal(th_cap.cpu().numpy().view(np.uint32), th_ora.view(np.uint32)), f"replay {rep + 1}: theta vs oracle"
        assert np.array_equal(cap.moment().view(np.uint32), ora.m().view(np.uint32)), f"replay {rep + 1}: m vs oracle"
        for r in range(R):
            assert np.array_equal(cap.residual(r).view(np.uint32), ora.e(r).view(np.uint32)), f"replay {rep + 1}: e[{r}]"
    ref.close()
    cap.close()


def test_select_survives_threshold_jumps(B):
    """Gradient scale jumps by 100x up and down between steps: the predicted bracket misses in both
    directions (and overflows when everything becomes a candidate); every step must stay exact."""
    rng = np.random.default_rng(7)
    N, R, s = 300_000 + 5, 2, 0.99
    gpu = B.Scape(N, R, s, **HYP)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(N, R, s, **HYP)
    th_ora = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th_gpu = torch.from_numpy(th_ora.copy()).cuda()
    scales = [1e-3, 1e-3, 1e-3, 1e-1, 1e-1, 1e-5, 1e-5, 1e-3, 1e-3, 1e-3, 0.0, 1e-3, 1e-3]
    for t, sc in enumerate(scales, 1):
        base = [(sc * rng.standard_normal(N)).astype(np.float32) for _ in range(R)]
        if t == 9:
            for b in base:
                b[:] = 1e-3          # constant gradient: huge tie class around the threshold
        gpu.step(th_gpu, [torch.from_numpy(b).cuda() for b in base])
        ora.step(th_ora, base)
        compare_step(gpu, ora, th_gpu, th_ora, R, f"jump step {t}")
    fast, general = gpu.select_stats()
    assert fast >= 2 and general >= 3, (fast, general)
    # most misses are completed by the recovery pass (sampled bracket + one classification pass) ...
    assert gpu.select_recovered() >= 3, (fast, general, gpu.select_recovered())
    gpu.close()


# ------------------------------------------------------------------------------------------
# Optional parts of Alg. 1: learning-rate schedule, bias correction, clip_grad (l.14)
# ------------------------------------------------------------------------------------------
def run_options_parity(B, w, steps, seed, bias_correction=False, clip=0.0, lr_schedule=False, exact=True):
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=seed)
    th_gpu = gs.theta0()
    th_ora = th_gpu.cpu().numpy().copy()
    gpu = B.Scape(N, R, w.sparsity, **HYP)
    gpu.keep_dense_pack(True)
    ora = ScapeOracle(N, R, w.sparsity, **HYP)
    for o in (gpu, ora):
        o.set_bias_correction(bias_correction)
        o.set_clip_grad(clip)
    clipped = 0
    for t in range(1, steps + 1):
        if lr_schedule:
            lr = HYP["lr"] * (0.25 + 0.25 * t)
            gpu.set_lr(lr)
            ora.set_lr(lr)
        grads = gs.next()
        gpu.step(th_gpu, grads)
        ora.step(th_ora, [to_np32(g) for g in grads])
        if clip > 0:
            norm, coef = gpu.last_grad_norm()
            np.testing.assert_allclose(norm, ora.last_norm(), rtol=1e-12)
            np.testing.assert_allclose(coef, ora.last_coef(), rtol=2e-7)
            clipped += coef < 1.0
            same_coef = np.float32(coef) == np.float32(ora.last_coef())
        else:
            same_coef = True
        compare_step(gpu, ora, th_gpu, th_ora, R, f"{w.name} opt step {t}", exact=exact and same_coef)
    gpu.close()
    return clipped


def small_workload(name, N, R, s, gdt="f32"):
    return synth.Workload(name, [("a", N // 3), ("b", N - N // 3)], R=R, sparsity=s, dist="t4", rho=0.9,
                          grad_dtype=gdt, steps=6)


def test_bias_correction_and_lr_schedule(B):
    run_options_parity(B, small_workload("bc", 200_003, 3, 0.99), 6, seed=21, bias_correction=True, lr_schedule=True)
    run_options_parity(B, small_workload("bc_dense", 50_001, 2, 0.0, "bf16"), 4, seed=22, bias_correction=True, lr_schedule=True)


@pytest.mark.parametrize("N,R,s,gdt,clip", [
    (300_007, 4, 0.99, "bf16", 1e-3),      # staged kernel, clip bites every step
    (300_007, 2, 0.9, "f32", 2e-3),        # register-staged kernel
    (40_001, 3, 0.0, "f32", 1e-2),         # all-ones mask every step: the deferred update covers all N
])
def test_clip_grad(B, N, R, s, gdt, clip):
    clipped = run_options_parity(B, small_workload("clip", N, R, s, gdt), 6, seed=N, clip=clip, bias_correction=True)
    assert clipped >= 3


def test_clip_grad_above_the_norm_is_a_bitwise_noop(B):
    w = small_workload("clip_noop", 150_011, 3, 0.99)
    gs = synth.GradStream(w, device="cuda", seed=5)
    th_a = gs.theta0()
    th_b = th_a.clone()
    a, b = B.Scape(w.numel, w.R, w.sparsity, **HYP), B.Scape(w.numel, w.R, w.sparsity, **HYP)
    b.set_clip_grad(1e9)
    for _ in range(5):
        grads = gs.next()
        a.step(th_a, grads)
        b.step(th_b, grads)
        assert b.last_grad_norm()[1] == 1.0
        assert torch.equal(th_a, th_b)
    np.testing.assert_array_equal(a.mask_next(), b.mask_next())
    a.close()
    b.close()


@pytest.mark.parametrize("form", [1, 2])
def test_both_compaction_forms(B, form):
    """rank128 + index list from the mask bits: the three-kernel form (large shards) and the single-pass
    chained scan (small shards) are chosen by size; scape_set_compaction forces either on the same
    ragged shard."""
    w = synth.Workload(f"compact{form}", [("a", 300_000), ("b", 1024 * 700 + 77)], R=2, sparsity=0.97, dist="t3", rho=0.9,
                       grad_dtype="f32", steps=5)
    run_reload_parity(B, w, steps=5, seed=form, setup=lambda gpu: gpu.set_compaction(form))
