"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE ONLY — see scape_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this module.  It imports nothing from paper_2607_01678_b200.
"""
import ctypes

import numpy as np

from . import build as _build

_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(_build.build())
    return _LIB


class ScapeOracle:
    """One rank's partition of Algorithm 1 with R simulated replicas.

    dtype np.float32 is the graded arithmetic; np.float64 is the same source instantiated in
    double for the exact-arithmetic pins.
    """

    def __init__(self, shard_numel, R, sparsity, beta1, beta2, eps, lr, wd, dtype=np.float32):
        self.dtype = np.dtype(dtype)
        self.suf = {"float32": "f32", "float64": "f64"}[self.dtype.name]
        self.N, self.R = int(shard_numel), int(R)
        L = _lib()
        self._f = lambda name: getattr(L, f"oracle_{name}_{self.suf}")
        cr = self._f("create")
        cr.restype = ctypes.c_void_p
        cr.argtypes = [ctypes.c_int64, ctypes.c_int] + [ctypes.c_double] * 6
        self.h = cr(self.N, self.R, sparsity, beta1, beta2, eps, lr, wd)
        if not self.h:
            raise ValueError("oracle_create rejected the arguments")
        for name in ("k", "t", "K_last"):
            fn = self._f(name)
            fn.restype = ctypes.c_int64
            fn.argtypes = [ctypes.c_void_p]

    def __del__(self):
        if getattr(self, "h", None):
            d = self._f("destroy")
            d.argtypes = [ctypes.c_void_p]
            d(self.h)
            self.h = None

    # ---- scalars -------------------------------------------------------------------
    @property
    def k(self):
        return int(self._f("k")(self.h))

    @property
    def t(self):
        return int(self._f("t")(self.h))

    @property
    def K_last(self):
        return int(self._f("K_last")(self.h))

    def set_t(self, t):
        fn = self._f("set_t")
        fn.argtypes = [ctypes.c_void_p, ctypes.c_int64]
        fn(self.h, int(t))

    def set_layers(self, offsets, compress=None):
        """Per-layer refresh: layers [offsets[l], offsets[l+1]); compress[l] == 0
        marks a layer that is never sparsified."""
        off = np.ascontiguousarray(offsets, dtype=np.int64)
        L = off.size - 1
        cp = np.ones(L, np.uint8) if compress is None else np.ascontiguousarray(compress, dtype=np.uint8)
        assert cp.size == L
        fn = self._f("set_layers")
        fn.restype = ctypes.c_int
        fn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        if fn(self.h, int(L), off.ctypes.data, cp.ctypes.data) != 0:
            raise ValueError("oracle_set_layers rejected the offsets")

    def set_workers(self, workers, layer_owner=None):
        """the R replicas are `workers` groups of R/workers replicas; layer l's
        mask comes from worker layer_owner[l]'s statistic; l.10 sums per worker, then over workers."""
        fn = self._f("set_workers")
        fn.restype = ctypes.c_int
        fn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
        ow = None if layer_owner is None else np.ascontiguousarray(layer_owner, dtype=np.int32)
        if fn(self.h, int(workers), None if ow is None else ow.ctypes.data) != 0:
            raise ValueError("oracle_set_workers rejected the arguments")

    def set_sparsity(self, s):
        """Sparsity of the coming refreshes (density warm-up)."""
        fn = self._f("set_sparsity")
        fn.restype = ctypes.c_int
        fn.argtypes = [ctypes.c_void_p, ctypes.c_double]
        if fn(self.h, float(s)) != 0:
            raise ValueError("sparsity must be in [0, 1)")

    def set_lr(self, lr):
        fn = self._f("set_lr")
        fn.argtypes = [ctypes.c_void_p, ctypes.c_double]
        fn(self.h, float(lr))

    def set_bias_correction(self, on):
        fn = self._f("set_bias_correction")
        fn.argtypes = [ctypes.c_void_p, ctypes.c_int]
        fn(self.h, int(on))

    def set_clip_grad(self, max_norm):
        fn = self._f("set_clip_grad")
        fn.argtypes = [ctypes.c_void_p, ctypes.c_double]
        fn(self.h, float(max_norm))

    def last_norm(self):
        fn = self._f("last_norm")
        fn.restype, fn.argtypes = ctypes.c_double, [ctypes.c_void_p]
        return fn(self.h)

    def last_coef(self):
        fn = self._f("last_coef")
        fn.restype, fn.argtypes = ctypes.c_double, [ctypes.c_void_p]
        return fn(self.h)

    # ---- the step ------------------------------------------------------------------
    def step(self, theta, grads):
        """theta: contiguous array [N] of self.dtype, updated in place. grads: R arrays [N]."""
        assert theta.dtype == self.dtype and theta.flags.c_contiguous and theta.size == self.N
        gs = [np.ascontiguousarray(g, dtype=self.dtype) for g in grads]
        assert len(gs) == self.R and all(g.size == self.N for g in gs)
        arr = (ctypes.c_void_p * self.R)(*[g.ctypes.data for g in gs])
        fn = self._f("step")
        fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        fn(self.h, theta.ctypes.data, arr)

    # ---- state / last-step outputs ---------------------------------------------------
    def _get(self, name, n, dtype=None, r=None):
        out = np.empty(n, dtype=dtype or self.dtype)
        fn = self._f("get_" + name)
        if r is None:
            fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
            fn(self.h, out.ctypes.data)
        else:
            fn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
            fn(self.h, int(r), out.ctypes.data)
        return out

    def _set(self, name, arr, dtype=None, r=None):
        a = np.ascontiguousarray(arr, dtype=dtype or self.dtype)
        assert a.size == self.N
        fn = self._f("set_" + name)
        if r is None:
            fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
            fn(self.h, a.ctypes.data)
        else:
            fn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
            fn(self.h, int(r), a.ctypes.data)

    def m(self):
        return self._get("m", self.N)

    def set_m(self, a):
        self._set("m", a)

    def e(self, r):
        return self._get("e", self.N, r=r)

    def set_e(self, r, a):
        self._set("e", a, r=r)

    def mask(self):
        """The mask the NEXT step will use (M_t after step t), as uint8 [N]."""
        return self._get("mask", self.N, dtype=np.uint8)

    def set_mask(self, a):
        self._set("mask", a, dtype=np.uint8)

    def idx(self):
        """Ascending indices of the mask the LAST step used."""
        return self._get("idx", self.K_last, dtype=np.int32)

    def mt(self, r):
        return self._get("mt", self.N, r=r)

    def b(self, r):
        return self._get("b", self.K_last, r=r)

    def bbar(self):
        return self._get("bbar", self.K_last)

    def ghat(self):
        return self._get("ghat", self.K_last)

    def v(self):
        return self._get("v", self.K_last)

    def u(self):
        return self._get("u", self.K_last)


def topk_mask(x, k):
    """refresh_mask on its own: uint8 mask of the k largest |x|, ties to the lower index."""
    x = np.ascontiguousarray(x)
    suf = {"float32": "f32", "float64": "f64"}[x.dtype.name]
    fn = getattr(_lib(), f"oracle_topk_{suf}")
    fn.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p]
    out = np.zeros(x.size, dtype=np.uint8)
    fn(x.ctypes.data, x.size, int(k), out.ctypes.data)
    return out


def mask_pack(mask_bytes):
    """Mask bit pack written out from its definition (INT8 mask values to 1 bit
    each, 8 per byte; layout of include/scape.h: bit i % 32 of little-endian word i / 32): a plain
    loop over the entries, no library routine.  Returns uint32 words, ceil(n / 32) of them."""
    m = np.asarray(mask_bytes)
    n = m.size
    words = [0] * ((n + 31) // 32)
    for i in range(n):
        if m[i] != 0:
            words[i // 32] |= 1 << (i % 32)
    return np.array(words, dtype=np.uint32)


def mask_unpack(words, n):
    """The inverse of mask_pack, entry by entry: uint8 [n] of 0 / 1."""
    w = np.asarray(words, dtype=np.uint32)
    return np.array([(int(w[i // 32]) >> (i % 32)) & 1 for i in range(n)], dtype=np.uint8)


# ---- Algorithm 2, parameter side (scape_oracle.cpp "Algorithm 2") ----------------
def bf16_rne(x):
    """float32 array -> uint16 array of bfloat16 bit patterns, round to nearest even (the C++ definition, entry by entry)."""
    a = np.ascontiguousarray(x, dtype=np.float32).ravel()
    out = np.empty(a.size, np.uint16)
    fn = _lib().oracle_bf16_rne_array
    fn.restype, fn.argtypes = None, [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p]
    fn(a.ctypes.data, a.size, out.ctypes.data)
    return out


def bf16_widen(b):
    """uint16 bfloat16 bit patterns -> float32 (exact)."""
    return (np.asarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def param_pack(w_local, mask, dtype="f32"):
    """Alg. 2 l.2: the owner's parameters on the mask, packed in ascending index order.
    dtype "f32" -> float32 array, "bf16" -> uint16 bit patterns (RNE)."""
    w = np.ascontiguousarray(w_local, dtype=np.float32)
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    assert w.size == m.size
    K = int(np.count_nonzero(m))
    fn = _lib().oracle_param_pack
    fn.restype = ctypes.c_int64
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
    if dtype == "f32":
        out = np.empty(K, np.float32)
        n = fn(w.ctypes.data, m.ctypes.data, w.size, out.ctypes.data, None)
    else:
        out = np.empty(K, np.uint16)
        n = fn(w.ctypes.data, m.ctypes.data, w.size, None, out.ctypes.data)
    assert n == K
    return out


def param_apply(w, mask, payload, lr, wd, w_hat=None, form=0):
    """Alg. 2 l.3-4 on a non-owner: `w` (float32 [N]) is updated in place, `w_hat` (uint16 [N], optional)
    receives bf16(w).  payload: float32 or uint16 (bf16 bits), one value per set mask entry, index order."""
    assert w.dtype == np.float32 and w.flags.c_contiguous
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    p = np.ascontiguousarray(payload)
    assert p.dtype in (np.float32, np.uint16) and p.size == int(np.count_nonzero(m)) and m.size == w.size
    if w_hat is not None:
        assert w_hat.dtype == np.uint16 and w_hat.flags.c_contiguous and w_hat.size == w.size
    fn = _lib().oracle_param_apply
    fn.restype = None
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
                   ctypes.c_double, ctypes.c_double, ctypes.c_int]
    fn(w.ctypes.data, None if w_hat is None else w_hat.ctypes.data, m.ctypes.data, w.size,
       p.ctypes.data if p.dtype == np.float32 else None, p.ctypes.data if p.dtype == np.uint16 else None,
       float(lr), float(wd), int(form))
