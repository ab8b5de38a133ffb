"""Thin ctypes binding of libscape.so (include/scape.h).  Argument marshalling only: every step
of the path runs in the CUDA kernels.  There is no fallback: if the library is missing, cannot be
loaded, or no CUDA device exists, the calls raise.

The module-level functions carry the C names (scape_create, scape_step, ...) and take raw
pointers (ints); `Scape` is a small convenience wrapper over torch tensors (torch is used for
device memory and streams only).
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libscape.so")

SCAPE_OK, SCAPE_EINVAL, SCAPE_ECUDA, SCAPE_ENOMEM = 0, -1, -2, -3
SCAPE_GRAD_F32, SCAPE_GRAD_BF16 = 0, 1
SCAPE_PARAM_F32, SCAPE_PARAM_BF16 = 0, 1
(SCAPE_MOMENT, SCAPE_RESIDUAL, SCAPE_MASK_NEXT, SCAPE_MASK_LAST, SCAPE_IDX_NEXT, SCAPE_IDX_LAST,
 SCAPE_PACKED, SCAPE_PACKED_MEAN) = range(8)

# every symbol include/scape.h declares: name -> (restype, argtypes)
_VP, _I64, _I, _D, _SZ = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
SYMBOLS = {
    "scape_create": (_VP, [_I64, _I, _D, _D, _D, _D, _D, _D]),
    "scape_step": (_I, [_VP, _VP, _VP, _VP]),
    "scape_step_host": (_I, [_VP, _VP, _VP, _VP]),
    "scape_destroy": (None, [_VP]),
    "scape_k": (_I64, [_VP]),
    "scape_step_count": (_I64, [_VP]),
    "scape_launch_count": (_I64, [_VP]),
    "scape_last_kernel": (ctypes.c_char_p, [_VP]),
    "scape_count": (_I64, [_VP, _I]),
    "scape_set_grad_dtype": (_I, [_VP, _I]),
    "scape_set_keep_dense_pack": (_I, [_VP, _I]),
    "scape_set_compaction": (_I, [_VP, _I]),
    "scape_set_lr": (_I, [_VP, _D]),
    "scape_set_bias_correction": (_I, [_VP, _I]),
    "scape_set_clip_grad": (_I, [_VP, _D]),
    "scape_last_grad_norm": (_I, [_VP, _VP, _VP, _VP]),
    "scape_set_layers": (_I, [_VP, _I, _VP, _VP]),
    "scape_set_sparsity": (_I, [_VP, _D]),
    "scape_layer_k": (_I64, [_VP, _I]),
    "scape_set_workers": (_I, [_VP, _I, _I, _VP]),
    "scape_step_local": (_I, [_VP, _VP, _VP, _VP]),
    "scape_exchange_buffers": (_I, [_VP, _VP, _VP, _VP, _VP]),
    "scape_step_apply": (_I, [_VP, _VP, _VP]),
    "scape_step_exchange": (_I, [_VP, _VP, _VP, _VP]),
    "scape_exchange_plan": (_I, [_VP, _VP, _VP, _VP, _I, _VP, _VP, _I, _VP]),
    "scape_nccl_unique_id": (_I, [_VP]),
    "scape_nccl_comm_create": (_I, [_I, _I, _VP, _VP]),
    "scape_nccl_comm_destroy": (_I, [_VP]),
    "scape_set_async_refresh": (_I, [_VP, _I]),
    "scape_join_refresh": (_I, [_VP, _VP]),
    "scape_param_pack": (_I, [_VP, _VP, _I64, _I64, _VP, _I, _VP]),
    "scape_param_apply": (_I, [_VP, _VP, _VP, _VP, _I, _VP]),
    "scape_mask_pack": (_I, [_VP, _I64, _VP, _VP]),
    "scape_mask_unpack": (_I, [_VP, _I64, _VP, _VP]),
    "scape_mask_indices_static": (_I, [_VP, _I64, _VP, _I64, _VP, _VP]),
    "scape_get": (_I, [_VP, _I, _I, _VP, _SZ, _VP]),
    "scape_set": (_I, [_VP, _I, _I, _VP, _SZ, _VP]),
    "scape_set_step_count": (_I, [_VP, _I64]),
    "scape_select_stats": (_I, [_VP, _VP, _VP, _VP]),
    "scape_select_recovered": (_I, [_VP, _VP, _VP]),
    "scape_select_debug": (_I, [_VP, _VP, _VP]),
    "scape_profile": (_I, [_VP, _I]),
    "scape_profile_read": (_I, [_VP, _VP, _VP, _VP]),
    "scape_last_error": (ctypes.c_char_p, []),
}

_LIB = None


def _device_view(ptr, n, dtype):
    """torch tensor over n elements of device memory owned by the library (current device)."""
    import torch

    class _Mem:
        pass
    m = _Mem()
    m.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "<f4" if dtype == "float32" else "<i4",
                                  "data": (int(ptr), False), "version": 3, "strides": None}
    return torch.as_tensor(m, device="cuda")


class ScapeError(RuntimeError):
    pass


def lib():
    """Load libscape.so (once).  Raises if it has not been built — there is no fallback."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ScapeError(f"{LIB_PATH} is missing: run `python -m paper_2607_01678_b200.build` "
                             "(or __graft_entry__.build()); there is no CPU or PyTorch fallback")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _LIB = L
    return _LIB


def scape_last_error() -> str:
    return lib().scape_last_error().decode()


def _check(rc, what):
    if rc != SCAPE_OK:
        raise ScapeError(f"{what} failed ({rc}): {scape_last_error()}")


def scape_create(shard_numel, R, sparsity, beta1, beta2, eps, lr, wd):
    h = lib().scape_create(int(shard_numel), int(R), float(sparsity), float(beta1), float(beta2),
                           float(eps), float(lr), float(wd))
    if not h:
        raise ScapeError(f"scape_create failed: {scape_last_error()}")
    return h


def scape_step(h, param_ptr, grad_ptrs, stream=0):
    arr = (ctypes.c_void_p * len(grad_ptrs))(*grad_ptrs)
    _check(lib().scape_step(h, param_ptr, arr, stream), "scape_step")


def scape_step_host(h, param_ptr, grad_ptrs, stream=0):
    arr = (ctypes.c_void_p * len(grad_ptrs))(*grad_ptrs)
    _check(lib().scape_step_host(h, param_ptr, arr, stream), "scape_step_host")


def scape_destroy(h):
    lib().scape_destroy(h)


def scape_k(h):
    return int(lib().scape_k(h))


def scape_step_count(h):
    return int(lib().scape_step_count(h))


def scape_launch_count(h):
    return int(lib().scape_launch_count(h))


def scape_last_kernel(h):
    return lib().scape_last_kernel(h).decode()


def scape_count(h, which):
    n = int(lib().scape_count(h, which))
    if n < 0:
        raise ScapeError(f"scape_count failed ({n}): {scape_last_error()}")
    return n


def scape_set_grad_dtype(h, dtype):
    _check(lib().scape_set_grad_dtype(h, dtype), "scape_set_grad_dtype")


def scape_set_keep_dense_pack(h, on):
    _check(lib().scape_set_keep_dense_pack(h, int(on)), "scape_set_keep_dense_pack")


def scape_set_compaction(h, form):
    _check(lib().scape_set_compaction(h, int(form)), "scape_set_compaction")


def scape_set_lr(h, lr):
    _check(lib().scape_set_lr(h, float(lr)), "scape_set_lr")


def scape_set_bias_correction(h, on):
    _check(lib().scape_set_bias_correction(h, int(on)), "scape_set_bias_correction")


def scape_set_clip_grad(h, max_norm):
    _check(lib().scape_set_clip_grad(h, float(max_norm)), "scape_set_clip_grad")


def scape_last_grad_norm(h, stream=0):
    """-> (||g^||_2, factor applied) of the last step"""
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(lib().scape_last_grad_norm(h, ctypes.byref(a), ctypes.byref(b), stream), "scape_last_grad_norm")
    return a.value, b.value


def scape_set_layers(h, offsets, compress=None):
    """offsets: n_layers+1 ints (0 ... shard_numel); compress: n_layers flags or None (all compressed)."""
    n = len(offsets) - 1
    off = (ctypes.c_int64 * (n + 1))(*[int(x) for x in offsets])
    cp = None if compress is None else (ctypes.c_uint8 * n)(*[int(bool(x)) for x in compress])
    _check(lib().scape_set_layers(h, n, off, cp), "scape_set_layers")


def scape_set_workers(h, world, rank, layer_owner=None):
    ow = None if layer_owner is None else np.ascontiguousarray(layer_owner, dtype=np.int32)
    _check(lib().scape_set_workers(h, int(world), int(rank), None if ow is None else ow.ctypes.data), "scape_set_workers")


def scape_step_local(h, param_ptr, grad_ptrs, stream=0):
    arr = (ctypes.c_void_p * len(grad_ptrs))(*grad_ptrs)
    _check(lib().scape_step_local(h, param_ptr, arr, stream), "scape_step_local")


def scape_exchange_buffers(h):
    """-> (sums device pointer, n_sums, mask words device pointer, n_mask_words)"""
    ps, pw = ctypes.c_void_p(), ctypes.c_void_p()
    ns, nw = ctypes.c_int64(), ctypes.c_int64()
    _check(lib().scape_exchange_buffers(h, ctypes.byref(ps), ctypes.byref(ns), ctypes.byref(pw), ctypes.byref(nw)),
           "scape_exchange_buffers")
    return ps.value or 0, ns.value, pw.value or 0, nw.value


def scape_step_apply(h, param_ptr, stream=0):
    _check(lib().scape_step_apply(h, param_ptr, stream), "scape_step_apply")


def scape_step_exchange(h, comm, mask_comm=None, stream=0):
    _check(lib().scape_step_exchange(h, comm, mask_comm, stream), "scape_step_exchange")


def scape_exchange_plan(h):
    """-> ([(first word, end word, owner)], [shared word numbers]): what scape_step_exchange moves of M_t"""
    nr, ns = ctypes.c_int(), ctypes.c_int()
    lib().scape_exchange_plan(h, None, None, None, 0, ctypes.byref(nr), None, 0, ctypes.byref(ns))
    a, b = (ctypes.c_int64 * max(1, nr.value))(), (ctypes.c_int64 * max(1, nr.value))()
    o, sh = (ctypes.c_int32 * max(1, nr.value))(), (ctypes.c_int64 * max(1, ns.value))()
    _check(lib().scape_exchange_plan(h, a, b, o, nr.value, ctypes.byref(nr), sh, ns.value, ctypes.byref(ns)), "scape_exchange_plan")
    return [(a[i], b[i], o[i]) for i in range(nr.value)], [sh[i] for i in range(ns.value)]


SCAPE_NCCL_ID_BYTES = 128


def scape_nccl_unique_id() -> bytes:
    buf = ctypes.create_string_buffer(SCAPE_NCCL_ID_BYTES)
    _check(lib().scape_nccl_unique_id(buf), "scape_nccl_unique_id")
    return buf.raw


def scape_nccl_comm_create(world, rank, uid: bytes):
    assert len(uid) == SCAPE_NCCL_ID_BYTES
    comm = ctypes.c_void_p()
    _check(lib().scape_nccl_comm_create(int(world), int(rank), ctypes.create_string_buffer(uid, SCAPE_NCCL_ID_BYTES), ctypes.byref(comm)),
           "scape_nccl_comm_create")
    return comm.value


def scape_nccl_comm_destroy(comm):
    _check(lib().scape_nccl_comm_destroy(comm), "scape_nccl_comm_destroy")


def scape_set_async_refresh(h, on):
    _check(lib().scape_set_async_refresh(h, int(on)), "scape_set_async_refresh")


def scape_join_refresh(h, stream=0):
    _check(lib().scape_join_refresh(h, stream), "scape_join_refresh")


def scape_param_pack(h, param_ptr, first, count, out_ptr, dtype, stream=0):
    _check(lib().scape_param_pack(h, param_ptr, int(first), int(count), out_ptr, int(dtype), stream), "scape_param_pack")


def scape_param_apply(h, w_ptr, w_hat_ptr, payload_ptr, dtype, stream=0):
    _check(lib().scape_param_apply(h, w_ptr, w_hat_ptr, payload_ptr, int(dtype), stream), "scape_param_apply")


def scape_mask_pack(mask_bytes_ptr, n, words_ptr, stream=0):
    _check(lib().scape_mask_pack(mask_bytes_ptr, int(n), words_ptr, stream), "scape_mask_pack")


def scape_mask_unpack(words_ptr, n, mask_bytes_ptr, stream=0):
    _check(lib().scape_mask_unpack(words_ptr, int(n), mask_bytes_ptr, stream), "scape_mask_unpack")


SCAPE_STATIC_MAX_BITS = 1 << 29


def scape_mask_indices_static(words_ptr, n, idx_ptr, idx_cap, count_ptr, stream=0):
    _check(lib().scape_mask_indices_static(words_ptr, n, idx_ptr, idx_cap, count_ptr, stream), "scape_mask_indices_static")


def mask_pack(mask_bytes):
    """torch uint8 [n] on the GPU -> torch int32 [ceil(n/32)] bit-packed."""
    import torch
    assert mask_bytes.is_cuda and mask_bytes.dtype == torch.uint8 and mask_bytes.is_contiguous()
    n = mask_bytes.numel()
    words = torch.empty((n + 31) // 32, dtype=torch.int32, device=mask_bytes.device)
    with torch.cuda.device(mask_bytes.device):
        scape_mask_pack(mask_bytes.data_ptr(), n, words.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return words


def mask_unpack(words, n):
    """torch int32 bit-packed words on the GPU -> torch uint8 [n] of 0 / 1."""
    import torch
    assert words.is_cuda and words.dtype == torch.int32 and words.is_contiguous() and words.numel() >= (n + 31) // 32
    out = torch.empty(n, dtype=torch.uint8, device=words.device)
    with torch.cuda.device(words.device):
        scape_mask_unpack(words.data_ptr(), n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return out


def scape_set_sparsity(h, sparsity):
    _check(lib().scape_set_sparsity(h, float(sparsity)), "scape_set_sparsity")


def scape_layer_k(h, layer):
    n = int(lib().scape_layer_k(h, int(layer)))
    if n < 0:
        raise ScapeError(f"scape_layer_k failed ({n}): {scape_last_error()}")
    return n


def scape_set_step_count(h, t):
    _check(lib().scape_set_step_count(h, int(t)), "scape_set_step_count")


def scape_get(h, what, r, buf_ptr, nbytes, stream=0):
    _check(lib().scape_get(h, what, r, buf_ptr, nbytes, stream), "scape_get")


def scape_set(h, what, r, buf_ptr, nbytes, stream=0):
    _check(lib().scape_set(h, what, r, buf_ptr, nbytes, stream), "scape_set")


def scape_select_stats(h, stream=0):
    """-> (steps whose select used the fused candidate list, steps that took the general path)"""
    a, b = ctypes.c_int64(), ctypes.c_int64()
    _check(lib().scape_select_stats(h, ctypes.byref(a), ctypes.byref(b), stream), "scape_select_stats")
    return a.value, b.value


def scape_select_recovered(h, stream=0):
    """-> "general" steps that the recovery pass (sampled bracket + one classification pass) completed"""
    a = ctypes.c_int64()
    _check(lib().scape_select_recovered(h, ctypes.byref(a), stream), "scape_select_recovered")
    return a.value


def scape_select_debug(h, stream=0):
    out = (ctypes.c_double * 8)()
    _check(lib().scape_select_debug(h, out, stream), "scape_select_debug")
    keys = ("hit", "n_above", "n_cand", "delta", "lnT", "ln_pred_next", "cand_cap", "n_seg")
    return dict(zip(keys, list(out)))


def scape_profile(h, on):
    _check(lib().scape_profile(h, int(on)), "scape_profile")


def scape_profile_read(h):
    """-> (fused_ms_total, select_ms_total, steps)"""
    a, b, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_int64()
    _check(lib().scape_profile_read(h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(n)), "scape_profile_read")
    return a.value, b.value, n.value


class Scape:
    """Convenience wrapper: one partition's SCAPE state on the current CUDA device.

    step(param, grads) takes torch CUDA tensors (param fp32 [N]; grads: R tensors [N], all fp32 or
    all bf16) and enqueues the step on torch's current stream.
    """

    def __init__(self, shard_numel, R, sparsity, beta1=0.9, beta2=0.95, eps=1e-8, lr=1e-3, wd=0.1):
        self.N, self.R = int(shard_numel), int(R)
        self.h = scape_create(shard_numel, R, sparsity, beta1, beta2, eps, lr, wd)
        self._gdt = SCAPE_GRAD_F32

    def close(self):
        if getattr(self, "h", None):
            try:
                scape_destroy(self.h)
            except TypeError:       # interpreter shutdown: the module globals are already gone
                pass
            self.h = None

    __del__ = close

    @property
    def k(self):
        return scape_k(self.h)

    @property
    def t(self):
        return scape_step_count(self.h)

    @property
    def last_kernel(self):
        return scape_last_kernel(self.h)

    @property
    def launches(self):
        return scape_launch_count(self.h)

    @staticmethod
    def _stream():
        import torch
        return torch.cuda.current_stream().cuda_stream

    def _set_dtype_for(self, g0):
        import torch
        want = SCAPE_GRAD_BF16 if g0.dtype == torch.bfloat16 else SCAPE_GRAD_F32
        if want == SCAPE_GRAD_F32 and g0.dtype != torch.float32:
            raise TypeError("gradients must be float32 or bfloat16")
        if want != self._gdt:
            scape_set_grad_dtype(self.h, want)
            self._gdt = want

    def step(self, param, grads):
        import torch
        assert param.is_cuda and param.dtype == torch.float32 and param.is_contiguous() and param.numel() == self.N
        assert len(grads) == self.R
        for g in grads:
            assert g.is_cuda and g.is_contiguous() and g.numel() == self.N and g.dtype == grads[0].dtype
        self._set_dtype_for(grads[0])
        scape_step(self.h, param.data_ptr(), [g.data_ptr() for g in grads], self._stream())

    # ---- workers: split step (include/scape.h "Workers") ---------------------------------
    def set_workers(self, world, rank, layer_owner=None):
        scape_set_workers(self.h, world, rank, layer_owner)

    def step_local(self, param, grads):
        import torch
        assert param.is_cuda and param.dtype == torch.float32 and param.is_contiguous() and param.numel() == self.N
        assert len(grads) == self.R
        for g in grads:
            assert g.is_cuda and g.is_contiguous() and g.numel() == self.N and g.dtype == grads[0].dtype
        self._set_dtype_for(grads[0])
        scape_step_local(self.h, param.data_ptr(), [g.data_ptr() for g in grads], self._stream())

    def exchange_tensors(self):
        """The two buffers to be summed over the workers, as torch views of the handle's device
        memory (no copy): (float32 [n_sums], int32 [n_mask_words] or None)."""
        ps, ns, pw, nw = scape_exchange_buffers(self.h)
        sums = _device_view(ps, ns, "float32")
        words = _device_view(pw, nw, "int32") if nw else None
        return sums, words

    def step_apply(self, param):
        scape_step_apply(self.h, param.data_ptr(), self._stream())

    def set_async_refresh(self, on=True):
        scape_set_async_refresh(self.h, on)

    def join_refresh(self):
        scape_join_refresh(self.h, self._stream())

    def exchange_plan(self):
        return scape_exchange_plan(self.h)

    def step_exchange(self, comm, mask_comm=None):
        """The exchange inside the library (scape_step_exchange): comm / mask_comm are ncclComm_t values
        (scape_nccl_comm_create, or any NCCL binding's)."""
        scape_step_exchange(self.h, comm, mask_comm, self._stream())

    def step_workers(self, param, grads, group=None, comm=None, mask_comm=None):
        """One step of worker `rank` of `world`: the local half, the exchange of PAPER.md:155 / :178 /
        :218, the apply half.  comm given: the library's own exchange over NCCL (scape_step_exchange).
        Otherwise torch.distributed moves the same things on the handle's buffers -- the sums with an
        all-reduce, of the mask only what the plan says: every word range from its owner, the shared
        words summed -- which also works on backends NCCL does not cover (gloo: two ranks on one GPU)."""
        self.step_local(param, grads)
        if comm is not None:
            self.step_exchange(comm, mask_comm)
        else:
            import torch
            import torch.distributed as dist
            sums, words = self.exchange_tensors()
            dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=group)
            if words is not None:
                ranges, shared = self.exchange_plan()
                for a, b, owner in ranges:
                    dist.broadcast(words[a:b], src=dist.get_global_rank(group, owner) if group is not None else owner, group=group)
                if shared:
                    ix = torch.tensor(shared, dtype=torch.int64, device=words.device)
                    sw = words[ix]
                    dist.all_reduce(sw, op=dist.ReduceOp.SUM, group=group)     # disjoint bits: SUM == OR
                    words[ix] = sw
        self.step_apply(param)

    # ---- Algorithm 2, parameter side (include/scape.h) -----------------------------------
    def param_pack(self, param, dtype=None, first=0, count=None, out=None):
        """Alg. 2 l.2: the updated parameters on the mask the last step used, packed in index order.
        dtype: torch.float32 (default) or torch.bfloat16.  Returns the torch tensor written."""
        import torch
        dtype = dtype or torch.float32
        assert param.is_cuda and param.dtype == torch.float32 and param.is_contiguous() and param.numel() == self.N
        if count is None:
            count = self.count_last() - first
        if out is None:
            out = torch.empty(count, dtype=dtype, device=param.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == dtype and out.numel() >= count
        scape_param_pack(self.h, param.data_ptr(), first, count, out.data_ptr(),
                         SCAPE_PARAM_BF16 if dtype == torch.bfloat16 else SCAPE_PARAM_F32, self._stream())
        return out

    def param_apply(self, w, payload, w_hat=None):
        """Alg. 2 l.3-4 on a copy that did not take the update: w (fp32 [N]) in place, w_hat (bf16 [N]) optional."""
        import torch
        assert w.is_cuda and w.dtype == torch.float32 and w.is_contiguous() and w.numel() == self.N
        assert payload.is_cuda and payload.is_contiguous() and payload.dtype in (torch.float32, torch.bfloat16)
        assert payload.numel() == self.count_last()
        if w_hat is not None:
            assert w_hat.is_cuda and w_hat.dtype == torch.bfloat16 and w_hat.is_contiguous() and w_hat.numel() == self.N
        scape_param_apply(self.h, w.data_ptr(), None if w_hat is None else w_hat.data_ptr(), payload.data_ptr(),
                          SCAPE_PARAM_BF16 if payload.dtype == torch.bfloat16 else SCAPE_PARAM_F32, self._stream())

    def step_host(self, param, grads):
        """param / grads: CPU tensors (pinned for async DMA). Synchronises before returning."""
        assert not param.is_cuda and param.is_contiguous() and param.numel() == self.N
        self._set_dtype_for(grads[0])
        scape_step_host(self.h, param.data_ptr(), [g.data_ptr() for g in grads], self._stream())

    # ---- accessors (numpy in / out) -------------------------------------------------
    def _get(self, what, n, dtype, r=0):
        out = np.empty(n, dtype=dtype)
        scape_get(self.h, what, r, out.ctypes.data, out.nbytes, self._stream())
        return out

    def _set(self, what, arr, dtype, r=0):
        a = np.ascontiguousarray(arr, dtype=dtype)
        scape_set(self.h, what, r, a.ctypes.data, a.nbytes, self._stream())

    def moment(self):
        return self._get(SCAPE_MOMENT, self.N, np.float32)

    def set_moment(self, a):
        self._set(SCAPE_MOMENT, a, np.float32)

    def residual(self, r):
        return self._get(SCAPE_RESIDUAL, self.N, np.float32, r)

    def set_residual(self, r, a):
        self._set(SCAPE_RESIDUAL, a, np.float32, r)

    def _mask(self, what):
        words = self._get(what, (self.N + 31) // 32, np.uint32)
        return np.unpackbits(words.view(np.uint8), bitorder="little")[: self.N]

    def mask_next(self):
        return self._mask(SCAPE_MASK_NEXT)

    def mask_last(self):
        return self._mask(SCAPE_MASK_LAST)

    def set_mask_next(self, mask_u8):
        m = np.asarray(mask_u8, dtype=np.uint8)
        assert m.size == self.N
        pad = (-self.N) % 32
        bits = np.packbits(np.concatenate([m, np.zeros(pad, np.uint8)]), bitorder="little")
        self._set(SCAPE_MASK_NEXT, bits.view(np.uint32), np.uint32)

    def count_next(self):
        return scape_count(self.h, SCAPE_MASK_NEXT)

    def count_last(self):
        return scape_count(self.h, SCAPE_MASK_LAST)

    def idx_next(self):
        return self._get(SCAPE_IDX_NEXT, self.count_next(), np.int32)

    def idx_last(self):
        return self._get(SCAPE_IDX_LAST, self.count_last(), np.int32)

    def packed(self, r):
        return self._get(SCAPE_PACKED, self.count_last(), np.float32, r)

    def packed_mean(self):
        return self._get(SCAPE_PACKED_MEAN, self.count_last(), np.float32)

    def keep_dense_pack(self, on=True):
        scape_set_keep_dense_pack(self.h, on)

    def set_compaction(self, form):
        scape_set_compaction(self.h, form)

    def set_step_count(self, t):
        scape_set_step_count(self.h, t)

    def set_layers(self, offsets, compress=None):
        scape_set_layers(self.h, offsets, compress)

    def clear_layers(self):
        _check(lib().scape_set_layers(self.h, 0, None, None), "scape_set_layers")

    def set_sparsity(self, sparsity):
        scape_set_sparsity(self.h, sparsity)

    def layer_k(self, layer):
        return scape_layer_k(self.h, layer)

    def set_lr(self, lr):
        scape_set_lr(self.h, lr)

    def set_bias_correction(self, on=True):
        scape_set_bias_correction(self.h, on)

    def set_clip_grad(self, max_norm):
        scape_set_clip_grad(self.h, max_norm)

    def last_grad_norm(self):
        return scape_last_grad_norm(self.h, self._stream())

    def select_stats(self):
        return scape_select_stats(self.h, self._stream())

    def select_debug(self):
        return scape_select_debug(self.h, self._stream())

    def select_recovered(self):
        return scape_select_recovered(self.h, self._stream())

    def profile(self, on=True):
        scape_profile(self.h, on)

    def profile_read(self):
        return scape_profile_read(self.h)
