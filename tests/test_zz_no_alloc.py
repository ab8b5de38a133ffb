"""scape_mask_indices_static — the ordered compaction of a bit mask with NO allocation (scratch in a
file-scope __device__ array of the library; include/scape.h) — against the existing path: the index
list a handle makes for the same mask (scape_set SCAPE_MASK_NEXT -> mask_compact / mask_rank_idx
kernels with cudaMalloc'ed scratch -> scape_get SCAPE_IDX_NEXT).  Index work: the bar is bit-exact.
`-m gpu`.  Collected last on purpose (the suite runs with pytest -x); self-contained, so it passes
alone in a fresh process and after the other tests."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01678_b200 import binding
    binding.lib()       # raises if libscape.so is missing: no fallback
    return binding


def _mask(n, density, seed, dense_head=0):
    rng = np.random.default_rng(seed)
    m = (rng.random(n) < density).astype(np.uint8)
    m[:dense_head] = 1                                 # chunks with more than 32 set bits: the warp-cooperative writer
    m[n - 1] = 1                                       # the last valid position, inside the ragged last word
    return m


def _words(m):
    """bit i % 32 of word i / 32; the padding bits of the last word are SET: the entry point must ignore them."""
    n = m.size
    pad = (-n) % 32
    return np.packbits(np.concatenate([m, np.ones(pad, np.uint8)]), bitorder="little").view(np.uint32)


def _existing_path(B, m, sparsity):
    """index list + count through a handle: cudaMalloc'ed scratch, the kernels every step uses"""
    s = B.Scape(m.size, 1, sparsity)
    try:
        assert int(m.sum()) <= s.k
        s.set_mask_next(m)
        return s.idx_next().copy(), s.count_next()
    finally:
        s.close()


def _static_path(B, m, idx_cap=None, guard=64):
    n = m.size
    words = torch.from_numpy(_words(m).view(np.int32)).cuda()
    cap = int(m.sum()) if idx_cap is None else idx_cap
    idx = torch.full((cap + guard,), -7, dtype=torch.int32, device="cuda")
    count = torch.full((1,), 123456, dtype=torch.int32, device="cuda")
    B.scape_mask_indices_static(words.data_ptr(), n, idx.data_ptr(), cap, count.data_ptr(),
                                torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    out = idx.cpu().numpy()
    assert (out[cap:] == -7).all(), "wrote past idx_cap"
    return out[:cap], int(count.item())


def test_static_scratch_matches_the_handle_path_on_calls_in_a_row(B):
    # several CTAs of 1024 chunks (look-back across blocks), a ragged tail, dense chunks; then a SMALLER mask, so that
    # the array still holds the first call's state beyond the second call's blocks; then a large one again
    cases = [(128 * 1024 * 3 + 77, 0.08, 0.9, 5000), (128 * 1024 + 5, 0.004, 0.99, 0), (128 * 1024 * 5 + 1, 0.3, 0.5, 300)]
    free = []
    for seed, (n, density, sparsity, head) in enumerate(cases):
        m = _mask(n, density, seed, head)
        want_idx, want_count = _existing_path(B, m, sparsity)
        got_idx, got_count = _static_path(B, m)
        assert got_count == want_count == int(m.sum())
        np.testing.assert_array_equal(got_idx, want_idx)
        np.testing.assert_array_equal(got_idx, np.flatnonzero(m).astype(np.int32))
        # the same call again, directly after: the array keeps the last call's contents
        again_idx, again_count = _static_path(B, m)
        assert again_count == want_count
        np.testing.assert_array_equal(again_idx, want_idx)
        free.append(torch.cuda.mem_get_info()[0])
    # the calls allocate nothing on the device: the free memory after each case's handle is gone does not shrink
    assert free[-1] >= free[0] - (1 << 20)


def test_static_scratch_capacity_count_only_and_empty(B):
    m = _mask(128 * 1024 + 333, 0.05, 11)
    total = int(m.sum())
    got, count = _static_path(B, m, idx_cap=1000)
    assert count == total
    np.testing.assert_array_equal(got, np.flatnonzero(m)[:1000].astype(np.int32))
    # count only
    words = torch.from_numpy(_words(m).view(np.int32)).cuda()
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    B.scape_mask_indices_static(words.data_ptr(), m.size, None, 0, cnt.data_ptr(), st)
    assert int(cnt.item()) == total
    # empty mask, n = 0
    z = torch.zeros(4, dtype=torch.int32, device="cuda")
    got, count = _static_path(B, np.zeros(1000, np.uint8))
    assert count == 0 and got.size == 0
    cnt.fill_(9)
    B.scape_mask_indices_static(z.data_ptr(), 0, None, 0, cnt.data_ptr(), st)
    assert int(cnt.item()) == 0


def test_static_scratch_rejects_sizes_beyond_the_maximum(B):
    z = torch.zeros(4, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    with pytest.raises(B.ScapeError, match="SCAPE_STATIC_MAX_BITS"):
        B.scape_mask_indices_static(z.data_ptr(), B.SCAPE_STATIC_MAX_BITS + 1, z.data_ptr(), 4, cnt.data_ptr(), 0)
    with pytest.raises(B.ScapeError):
        B.scape_mask_indices_static(z.data_ptr(), -1, z.data_ptr(), 4, cnt.data_ptr(), 0)
    with pytest.raises(B.ScapeError):
        B.scape_mask_indices_static(z.data_ptr() + 4, 64, z.data_ptr(), 4, cnt.data_ptr(), 0)      # misaligned mask
    with pytest.raises(B.ScapeError):
        B.scape_mask_indices_static(z.data_ptr(), 64, None, 4, cnt.data_ptr(), 0)                  # NULL idx_out with a capacity
