"""Algorithm 2, parameter side (Eq. 6 :207-211) on the GPU against the oracle — `-m gpu`.

scape_param_pack (l.2) and scape_param_apply (l.3-4) through the C-ABI, bit for bit against
oracle.param_pack / oracle.param_apply: the payload in fp32 and bf16, the FP32 copy w, the bf16
compute copy w^.  The owner's parameters come from the handle's own scape_step (itself checked
against the oracle elsewhere); the non-owner's copy must equal them to the bit with an fp32 payload.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import scape_oracle as O  # noqa: E402
from oracle.scape_oracle import ScapeOracle  # noqa: E402
from paper_2607_01678_b200 import synth  # noqa: E402

pytestmark = pytest.mark.gpu
HYP = dict(beta1=0.9, beta2=0.95, eps=1e-8, lr=1e-3, wd=0.1)


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01678_b200 import binding
    binding.lib()
    return binding


def bits16(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


@pytest.mark.parametrize("N,R,s,gdt", [
    (1, 1, 0.0, "f32"), (127, 2, 0.5, "f32"), (129, 1, 0.9, "f32"), (128 * 37 + 5, 2, 0.99, "bf16"),
    (300_000 + 77, 3, 0.99, "f32"), (262_144, 4, 0.9, "bf16"), (70_001, 2, 0.999, "f32"), (50_000, 2, 0.0, "f32"),
])
def test_pack_and_apply_match_the_oracle_and_the_copy_tracks_the_owner(B, N, R, s, gdt):
    w_ = synth.Workload(f"alg2_{N}", [("a", N // 2), ("b", N - N // 2)] if N > 1 else [("a", 1)], R=R, sparsity=s, dist="t3",
                        rho=0.9, grad_dtype=gdt, steps=5)
    gs = synth.GradStream(w_, device="cuda", seed=N)
    theta = gs.theta0()                                   # the owner's parameters
    th_ora = theta.cpu().numpy().copy()
    gpu = B.Scape(N, R, s, **HYP)
    ora = ScapeOracle(N, R, s, **HYP)
    # two non-owners: one fed with fp32 payloads, one with bf16 payloads; GPU and oracle versions of each
    w32, wbf = theta.clone(), theta.clone()
    hat32 = torch.zeros(N, dtype=torch.bfloat16, device="cuda")
    hatbf = torch.zeros(N, dtype=torch.bfloat16, device="cuda")
    o32, obf = th_ora.copy(), th_ora.copy()
    for t in range(1, 6):
        if t == 4:                                        # a learning-rate schedule: the decay uses the eta of the step just taken
            gpu.set_lr(5e-4)
            ora.set_lr(5e-4)
        lr = 5e-4 if t >= 4 else HYP["lr"]
        grads = gs.next()
        used = ora.mask().copy()                          # M_{t-1}
        gpu.step(theta, grads)
        ora.step(th_ora, [g.to(torch.float32).cpu().numpy() for g in grads])
        assert np.array_equal(theta.cpu().numpy().view(np.uint32), th_ora.view(np.uint32))
        K = gpu.count_last()
        assert K == int(used.sum())
        # l.2
        p32 = gpu.param_pack(theta)
        pbf = gpu.param_pack(theta, dtype=torch.bfloat16)
        q32, qbf = O.param_pack(th_ora, used, "f32"), O.param_pack(th_ora, used, "bf16")
        assert np.array_equal(p32.cpu().numpy().view(np.uint32), q32.view(np.uint32)), f"step {t}: fp32 payload"
        assert np.array_equal(bits16(pbf), qbf), f"step {t}: bf16 payload"
        # a worker that owns a range of the sparse buffer packs just that range, into its own place
        if K >= 3:
            parts = torch.empty(K, dtype=torch.float32, device="cuda")
            cuts = [0, K // 3, K // 3 + 1, K]
            for a, b in zip(cuts[:-1], cuts[1:]):
                gpu.param_pack(theta, first=a, count=b - a, out=parts[a:b])
            assert torch.equal(parts, p32)
        # l.3-4
        gpu.param_apply(w32, p32, w_hat=hat32)
        gpu.param_apply(wbf, pbf, w_hat=hatbf)
        oh32, ohbf = np.zeros(N, np.uint16), np.zeros(N, np.uint16)
        O.param_apply(o32, used, q32, lr, HYP["wd"], w_hat=oh32)
        O.param_apply(obf, used, qbf, lr, HYP["wd"], w_hat=ohbf)
        torch.cuda.synchronize()
        assert np.array_equal(w32.cpu().numpy().view(np.uint32), o32.view(np.uint32)), f"step {t}: w (fp32 payload)"
        assert np.array_equal(bits16(hat32), oh32), f"step {t}: w^ (fp32 payload)"
        assert np.array_equal(wbf.cpu().numpy().view(np.uint32), obf.view(np.uint32)), f"step {t}: w (bf16 payload)"
        assert np.array_equal(bits16(hatbf), ohbf), f"step {t}: w^ (bf16 payload)"
        # the point of the exercise: the non-owner's FP32 copy IS the owner's theta
        assert torch.equal(w32, theta), f"step {t}: the FP32 copy left the owner's parameters"
    # without a compute copy
    w_only = w32.clone()
    gpu.param_apply(w_only, p32)
    gpu.close()


def test_param_calls_reject_bad_arguments(B):
    N = 4096
    g = B.Scape(N, 1, 0.9, **HYP)
    th = torch.zeros(N, device="cuda")
    out = torch.zeros(N, device="cuda")
    L = B.lib()
    assert L.scape_param_pack(g.h, th.data_ptr(), 0, 1, out.data_ptr(), 0, None) == B.SCAPE_EINVAL        # no step yet
    assert L.scape_param_apply(g.h, th.data_ptr(), None, out.data_ptr(), 0, None) == B.SCAPE_EINVAL
    g.step(th, [torch.zeros(N, device="cuda")])
    K = g.count_last()
    assert K == N
    assert L.scape_param_pack(g.h, th.data_ptr(), 0, K + 1, out.data_ptr(), 0, None) == B.SCAPE_EINVAL     # range
    assert L.scape_param_pack(g.h, th.data_ptr(), -1, 1, out.data_ptr(), 0, None) == B.SCAPE_EINVAL
    assert L.scape_param_pack(g.h, th.data_ptr(), 0, 1, out.data_ptr(), 7, None) == B.SCAPE_EINVAL         # dtype
    assert L.scape_param_pack(g.h, th.data_ptr(), 0, 1, out.data_ptr() + 2, 0, None) == B.SCAPE_EINVAL     # alignment
    assert L.scape_param_apply(g.h, th.data_ptr() + 4, None, out.data_ptr(), 0, None) == B.SCAPE_EINVAL
    assert L.scape_param_apply(None, th.data_ptr(), None, out.data_ptr(), 0, None) == B.SCAPE_EINVAL
    assert L.scape_param_pack(g.h, th.data_ptr(), 0, 0, None, 0, None) == B.SCAPE_OK                       # empty range: no-op
    g.close()


def test_fullsize_param_exchange_sampled(B):
    """Llama-1.8B-shaped shard (N = 1,775,239,168): pack + apply at full size in steady state; the FP32
    copy equals the owner's parameters everywhere (torch.equal on the device), the compute copy equals
    torch's own bf16 rounding of it, and sampled positions go through the oracle."""
    w_ = synth.workload("llama1p8b")
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        pytest.skip("needs ~120 GB of free HBM")
    N, R = w_.numel, w_.R
    gs = synth.GradStream(w_, device="cuda", seed=0)
    theta = gs.theta0()
    sc = B.Scape(N, R, w_.sparsity, **w_.hyper)
    for _ in range(3):
        sc.step(theta, gs.next())
    w = theta.clone()
    hat = torch.empty(N, dtype=torch.bfloat16, device="cuda")
    grads = gs.next()
    del gs
    sc.step(theta, grads)
    del grads
    payload = sc.param_pack(theta)
    idx = torch.from_numpy(sc.idx_last()).cuda().long()
    assert torch.equal(payload, theta[idx])
    sc.param_apply(w, payload, w_hat=hat)
    torch.cuda.synchronize()
    assert torch.equal(w, theta), "the FP32 copy differs from the owner's parameters at full size"
    assert torch.equal(hat, theta.to(torch.bfloat16))
    # sampled positions through the oracle (bf16 payload this time)
    rng = np.random.default_rng(1)
    samp = torch.unique(torch.cat([torch.from_numpy(rng.integers(0, N, 4000)).cuda(), idx[torch.from_numpy(rng.integers(0, idx.numel(), 500)).cuda()],
                                   torch.tensor([0, 127, 128, N - 1], device="cuda")]))
    mask_s = torch.zeros(N, dtype=torch.bool, device="cuda")
    mask_s[idx] = True
    used_s = mask_s[samp].cpu().numpy().astype(np.uint8)
    del mask_s
    w2 = theta.clone()
    w2.mul_(1.25)                                        # a copy that is NOT equal to the owner's, so that l.4 is visible
    before = w2[samp].cpu().numpy()
    pbf = sc.param_pack(theta, dtype=torch.bfloat16)
    sc.param_apply(w2, pbf, w_hat=hat)
    torch.cuda.synchronize()
    th_s = theta[samp].cpu().numpy()
    o = before.copy()
    oh = np.zeros(o.size, np.uint16)
    O.param_apply(o, used_s, O.param_pack(th_s, used_s, "bf16"), w_.hyper["lr"], w_.hyper["wd"], w_hat=oh)
    assert np.array_equal(w2[samp].cpu().numpy().view(np.uint32), o.view(np.uint32))
    assert np.array_equal(bits16(hat[samp]), oh)
    sc.close()
