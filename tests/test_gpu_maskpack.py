"""Mask bit pack / unpack kernels against the oracle's plain loop — `-m gpu`.
Byte / bit work: the bar is bit-exact."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import scape_oracle as ora  # noqa: E402
from test_gpu_parity import HYP, B  # noqa: E402,F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [1, 2, 15, 16, 17, 31, 32, 33, 63, 64, 65, 255, 4096, 4097, 100_003, 8192 * 32 + 5])
def test_pack_unpack_against_the_oracle(B, n):
    rng = np.random.default_rng(n)
    m = (rng.random(n) < [0.01, 0.1, 0.5][n % 3]).astype(np.uint8)
    m[rng.integers(0, n)] = 200                      # any non-zero byte counts as selected
    want = ora.mask_pack(m) if n <= 100_003 else np.packbits(np.concatenate([m != 0, np.zeros((-n) % 32, bool)]),
                                                             bitorder="little").view(np.uint32)
    words = B.mask_pack(torch.from_numpy(m).cuda())
    got = words.cpu().numpy().view(np.uint32)
    np.testing.assert_array_equal(got, want)
    back = B.mask_unpack(words, n).cpu().numpy()
    np.testing.assert_array_equal(back, (m != 0).astype(np.uint8))
    if n <= 100_003:
        np.testing.assert_array_equal(back, ora.mask_unpack(want, n))


def test_unaligned_views_and_padding_bits(B):
    n = 1000
    base = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
    m = (torch.rand(n, device="cuda") < 0.3).to(torch.uint8)
    for off in (1, 3, 16, 17):                       # 16-byte accesses are not possible: the byte path
        v = base[off:off + n]
        v.copy_(m)
        words = B.mask_pack(v)
        np.testing.assert_array_equal(words.cpu().numpy().view(np.uint32), ora.mask_pack(m.cpu().numpy()))
        out = torch.full((n + 64,), 7, dtype=torch.uint8, device="cuda")
        B.scape_mask_unpack(words.data_ptr(), n, out[off:off + n].data_ptr(), torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert torch.equal(out[off:off + n], m)
        assert int(out[:off].min()) == 7 and int(out[off + n:].min()) == 7      # nothing written outside
    # bits at positions >= n are zero even when the bytes behind the mask are not
    base.fill_(1)
    words = B.mask_pack(base[:n])
    assert int(words[-1].item()) & ~((1 << (n % 32)) - 1) == 0


def test_the_handle_masks_are_in_this_format(B):
    """SCAPE_MASK_NEXT as the library keeps it == pack(mask bytes); unpack(that) == the oracle's mask."""
    from oracle.scape_oracle import ScapeOracle
    from paper_2607_01678_b200 import synth
    w = synth.Workload("maskpack", [("a", 30_000), ("b", 20_011)], R=2, sparsity=0.9, dist="gauss", rho=0.9,
                       grad_dtype="f32", steps=3)
    gs = synth.GradStream(w, device="cuda", seed=0)
    th = gs.theta0(); th_o = th.cpu().numpy().copy()
    gpu = B.Scape(w.numel, 2, 0.9, **w.hyper); o = ScapeOracle(w.numel, 2, 0.9, **w.hyper)
    for _ in range(3):
        g = gs.next()
        gpu.step(th, g); o.step(th_o, [x.cpu().numpy() for x in g])
    mk = o.mask()
    words = B.mask_pack(torch.from_numpy(mk).cuda())
    np.testing.assert_array_equal(B.mask_unpack(words, w.numel).cpu().numpy(), gpu.mask_next())
    np.testing.assert_array_equal(words.cpu().numpy().view(np.uint32)[: (w.numel + 31) // 32],
                                  ora.mask_pack(gpu.mask_next()))
    gpu.close()


def test_api_errors(B):
    with pytest.raises(B.ScapeError):
        B.scape_mask_pack(0, 10, 0)
    with pytest.raises(B.ScapeError):
        B.scape_mask_pack(0, -1, 0)
    B.scape_mask_pack(0, 0, 0)                        # n = 0: no-op
    t = torch.zeros(64, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.ScapeError):
        B.scape_mask_pack(t.data_ptr(), 8, t.data_ptr() + 1)      # misaligned words
