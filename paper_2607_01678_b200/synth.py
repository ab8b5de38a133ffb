"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json `configs`).

This module holds NO arithmetic of the SCAPE method: only tensor lists, random draws and the
AR(1) recursion that correlates gradients across steps.  It serves both the CUDA path and the
oracle (tests and bench.py hand the very same bytes to both sides).

The paper trains GPT-345M on OpenWebText and Llama-500M / Llama-1.8B on SlimPajama-6B
(PAPER.md:279, :286, :343); those datasets are not available here and are not needed: the
optimizer step only sees gradient values.  The generators below stand in for them with the
shapes, sizes and peaked / heavy-tailed value distributions the paper reports
(Fig. 4-5) as BASELINE.json's configs spell them out.

Recipe (also stated in DESIGN.md §Inputs):
  theta_0 ~ N(0, 0.02^2)
  AR(1) signal shared by the replicas:  a_1 = xi_1,  a_t = rho a_{t-1} + sqrt(1-rho^2) xi_t
  per-replica gradient:                 g_t^r = scale_tensor * (a_t + n_t^r)
  xi, n: unit-variance Gaussian or Student-t_nu = Z / sqrt(chi2_nu/nu) * sqrt((nu-2)/nu)
  scale_tensor: one per weight tensor, 10^(-5+3u), u ~ U(0,1)   (configs 2-4), or a constant
"""
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import torch

# --------------------------------------------------------------------------------------
# Tensor lists (2-D weights only: the paper leaves LayerNorm / RMSNorm / bias uncompressed,
# PAPER.md:279, :286)
# --------------------------------------------------------------------------------------


def gpt345m_tensors() -> List[Tuple[str, int]]:
    h, ff, L = 1024, 4096, 24
    t = []
    for i in range(L):
        t += [(f"l{i}.qkv", 3 * h * h), (f"l{i}.attn_out", h * h),
              (f"l{i}.fc", ff * h), (f"l{i}.proj", h * ff)]
    t += [("wte", 50257 * h), ("wpe", 1024 * h)]
    return t  # 354,501,632


def llama500m_tensors() -> List[Tuple[str, int]]:
    h, ff, L = 1536, 4096, 16
    t = []
    for i in range(L):
        t += [(f"l{i}.q", h * h), (f"l{i}.k", h * h), (f"l{i}.v", h * h), (f"l{i}.o", h * h),
              (f"l{i}.gate_up", 2 * ff * h), (f"l{i}.down", h * ff)]
    t += [("embed", 32000 * h)]
    return t  # 502,136,832


def llama1p8b_tensors(layers: int = 32, separate_output: bool = True) -> List[Tuple[str, int]]:
    """hidden 2048, SwiGLU FFN 5632, vocab 32000.  BASELINE.json's literal 24 layers give
    1.36 B; 32 layers + separate embedding and output matrices give 1,775,239,168 (~1.8 B),
    the headline size."""
    h, ff = 2048, 5632
    t = []
    for i in range(layers):
        t += [(f"l{i}.q", h * h), (f"l{i}.k", h * h), (f"l{i}.v", h * h), (f"l{i}.o", h * h),
              (f"l{i}.gate_up", 2 * ff * h), (f"l{i}.down", h * ff)]
    t += [("embed", 32000 * h)]
    if separate_output:
        t += [("output", 32000 * h)]
    return t


@dataclass
class Workload:
    name: str
    tensors: List[Tuple[str, int]]
    R: int
    sparsity: float
    dist: str            # "gauss" | "t3" | "t4"
    rho: float
    grad_dtype: str      # "f32" | "bf16" (bf16 buffers) | "bf16_in_f32" (bf16-valued fp32 buffers)
    steps: int
    per_tensor_scale: bool = True
    const_scale: float = 1e-3
    hyper: dict = field(default_factory=lambda: dict(beta1=0.9, beta2=0.95, eps=1e-8,
                                                     lr=1e-3, wd=0.1))

    @property
    def numel(self) -> int:
        return sum(n for _, n in self.tensors)

    def offsets(self) -> List[int]:
        """Tensor boundaries in the flattened shard: the layers of a per-layer refresh."""
        off = [0]
        for _, n in self.tensors:
            off.append(off[-1] + n)
        return off

    def compress_flags(self) -> List[int]:
        """0 for the tensors the paper leaves uncompressed (LayerNorm, RMSNorm, bias: PAPER.md:246,
        :279, :286), recognised by name; 1 for the weight matrices."""
        return [0 if any(t in name for t in ("norm", "bias", "ln_")) else 1 for name, _ in self.tensors]


def scaled(tensors: List[Tuple[str, int]], div: int) -> List[Tuple[str, int]]:
    """Same structure, every tensor `div` times smaller (kept a multiple of 8 elements, so
    bf16 segment boundaries stay 16-byte aligned)."""
    if div <= 1:
        return list(tensors)
    return [(n, max(8, (s // div) // 8 * 8)) for n, s in tensors]


def workload(name: str, div: int = 1, sparsity: Optional[float] = None) -> Workload:
    """BASELINE.json configs by name; `div` shrinks every tensor (parity tests, CPU baseline)."""
    if name == "pr1":
        w = Workload("pr1", [("flat", 1 << 20)], R=2, sparsity=0.90, dist="gauss", rho=0.9,
                     grad_dtype="f32", steps=10, per_tensor_scale=False, const_scale=1e-3)
    elif name == "gpt345m":
        w = Workload("gpt345m", gpt345m_tensors(), R=4, sparsity=0.99, dist="t4", rho=0.9,
                     grad_dtype="f32", steps=50)
    elif name == "llama500m":
        w = Workload("llama500m", llama500m_tensors(), R=8, sparsity=0.99, dist="gauss",
                     rho=0.95, grad_dtype="bf16_in_f32", steps=50)
    elif name == "llama1p8b":
        w = Workload("llama1p8b", llama1p8b_tensors(32, True), R=4, sparsity=0.99, dist="t3",
                     rho=0.9, grad_dtype="bf16", steps=20)
    elif name == "llama1p8b_literal":
        w = Workload("llama1p8b_literal", llama1p8b_tensors(24, True), R=4, sparsity=0.99,
                     dist="t3", rho=0.9, grad_dtype="bf16", steps=20)
    else:
        raise ValueError(f"unknown workload {name!r}")
    w.tensors = scaled(w.tensors, div)
    if div > 1:
        w.name = f"{w.name}/div{div}"
    if sparsity is not None:
        w.sparsity = float(sparsity)
    return w


def sweep_point(log2n: int, sparsity: float, R: int) -> Workload:
    """Config 5: i.i.d. Gaussian std 1e-3 (rho = 0), fp32 gradients."""
    return Workload(f"sweep/2^{log2n}/s{sparsity}/R{R}", [("flat", 1 << log2n)], R=R,
                    sparsity=sparsity, dist="gauss", rho=0.0, grad_dtype="f32", steps=13,
                    per_tensor_scale=False, const_scale=1e-3)


# --------------------------------------------------------------------------------------
# Random draws
# --------------------------------------------------------------------------------------

_CHUNK = 1 << 25


def _unit_noise(out: torch.Tensor, dist: str, gen: torch.Generator) -> None:
    """Fill `out` (fp32, 1-D) with unit-variance draws, chunked to bound temporaries."""
    n = out.numel()
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        z = torch.randn(hi - lo, device=out.device, dtype=torch.float32, generator=gen)
        if dist == "gauss":
            out[lo:hi] = z
        else:
            nu = {"t3": 3, "t4": 4}[dist]
            chi2 = torch.zeros_like(z)
            for _ in range(nu):
                w = torch.randn(hi - lo, device=out.device, dtype=torch.float32, generator=gen)
                chi2.addcmul_(w, w)
            z.div_(torch.sqrt(chi2.div_(nu)))
            z.mul_(((nu - 2) / nu) ** 0.5)
            out[lo:hi] = z


class GradStream:
    """Yields, step after step, the R per-replica gradient buffers of one workload."""

    def __init__(self, w: Workload, device="cpu", seed: int = 0):
        self.w = w
        self.device = torch.device(device)
        self.gen = torch.Generator(device=self.device)
        self.gen.manual_seed(int(seed))
        self.N = w.numel
        self.t = 0
        self.a = torch.zeros(self.N, dtype=torch.float32, device=self.device)
        if w.per_tensor_scale:
            # drawn on the CPU so the scales do not depend on the device
            g = torch.Generator().manual_seed(int(seed) + 7919)
            u = torch.rand(len(w.tensors), generator=g, dtype=torch.float64)
            self.scales = (10.0 ** (-5.0 + 3.0 * u)).tolist()
        else:
            self.scales = [w.const_scale] * len(w.tensors)

    def theta0(self) -> torch.Tensor:
        return 0.02 * torch.randn(self.N, device=self.device, dtype=torch.float32,
                                  generator=self.gen)

    def _apply_scales(self, x: torch.Tensor) -> None:
        off = 0
        for (_, n), s in zip(self.w.tensors, self.scales):
            x[off:off + n].mul_(s)
            off += n

    def next(self) -> List[torch.Tensor]:
        w = self.w
        self.t += 1
        xi = torch.empty(self.N, dtype=torch.float32, device=self.device)
        _unit_noise(xi, w.dist, self.gen)
        if self.t == 1 or w.rho == 0.0:
            self.a.copy_(xi)
        else:
            self.a.mul_(w.rho).add_(xi, alpha=(1.0 - w.rho * w.rho) ** 0.5)
        out = []
        for _ in range(w.R):
            _unit_noise(xi, w.dist, self.gen)       # reuse the buffer for n_t^r
            g = xi + self.a
            self._apply_scales(g)
            if w.grad_dtype == "bf16":
                g = g.to(torch.bfloat16)
            elif w.grad_dtype == "bf16_in_f32":
                g = g.to(torch.bfloat16).to(torch.float32)
            out.append(g.contiguous())
        return out
