"""Seeded synthetic inputs for the GeoFP8 codec (the ONLY module shared by the CUDA path's tests /
bench and the oracle's tests).  It holds none of the method's arithmetic: it only draws gradients,
activation / output-gradient samples and start bases with the shapes, spectra and structure of
BASELINE.json's five configs.  These inputs stand in for the paper's
OpenWebText-trained Llama-300M / 600M gradients, which are not available.

Everything is generated in FP32 with torch on the requested device and, for BF16 configs, rounded
to BF16 once; both the oracle and the GPU library then read the SAME bits.
"""
from dataclasses import dataclass, field
from typing import List, Optional

import torch

SIDE_NONE, SIDE_IN, SIDE_OUT, SIDE_BOTH = 0, 1, 2, 3
E4M3, E5M2 = 0, 1
SCALE_TENSOR, SCALE_BLOCK128 = 0, 1


def _seed(*parts) -> int:
    """Mix a tuple of small integers into one 63-bit seed (splitmix-style, no method arithmetic)."""
    x = 0x9E3779B97F4A7C15
    for p in parts:
        x = (x ^ (int(p) + 0x9E3779B97F4A7C15 + ((x << 6) & 0xFFFFFFFFFFFFFFFF) + (x >> 2))) & 0xFFFFFFFFFFFFFFFF
        x = (x * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
        x ^= x >> 31
    return x & 0x7FFFFFFFFFFFFFFF


def _gen(device, *parts):
    g = torch.Generator(device=device)
    g.manual_seed(_seed(*parts))
    return g


def rand_orthonormal(rows: int, cols: int, device, *seed) -> torch.Tensor:
    """rows x cols matrix with orthonormal columns: Q of the QR of a seeded Gaussian."""
    z = torch.randn(rows, cols, generator=_gen(device, *seed), device=device, dtype=torch.float32)
    q, r = torch.linalg.qr(z.double())
    q = q * torch.sign(torch.diagonal(r)).unsqueeze(0)
    return q.float()


def gradient(m: int, n: int, device, *seed, max_rank: int = 256, noise: float = 0.01,
             power: float = 1.5) -> torch.Tensor:
    """G = U diag(i^-power) V^T + noise * N(0,1), U and V random orthonormal (configs 0-4).

    For min(m, n) > max_rank the low-rank term keeps its first max_rank singular triplets
    (i^-1.5 at i = 256 is 2.4e-4, far below the noise floor) -- DESIGN.md recipe D5."""
    r = min(m, n, max_rank)
    U = rand_orthonormal(m, r, device, *seed, 1)
    V = rand_orthonormal(n, r, device, *seed, 2)
    s = torch.arange(1, r + 1, device=device, dtype=torch.float32) ** (-power)
    G = (U * s.unsqueeze(0)) @ V.t()
    G = G + noise * torch.randn(m, n, generator=_gen(device, *seed, 3), device=device, dtype=torch.float32)
    return G.contiguous()


def rank_gradient(G: torch.Tensor, rank: int, *seed, frac: float = 0.1) -> torch.Tensor:
    """Simulated DP rank r: the shared G plus an independent N(0, (frac * std(G))^2) perturbation."""
    g = _gen(G.device, *seed, 7, rank)
    sigma = frac * float(G.float().std())
    return (G.float() + sigma * torch.randn(G.shape, generator=g, device=G.device, dtype=torch.float32)).contiguous()


def factor_samples(T: int, d: int, device, *seed, power: float = 1.0) -> torch.Tensor:
    """T samples x ~ N(0, Sigma), Sigma = Q diag(i^-2power) Q^T in a random orthogonal basis Q:
    X = Z diag(i^-power) Q^T  (T x d, FP32)."""
    Q = rand_orthonormal(d, d, device, *seed, 11)
    z = torch.randn(T, d, generator=_gen(device, *seed, 12), device=device, dtype=torch.float32)
    s = torch.arange(1, d + 1, device=device, dtype=torch.float32) ** (-power)
    return ((z * s.unsqueeze(0)) @ Q.t()).contiguous()


def start_basis(d: int, k: int, device, *seed) -> torch.Tensor:
    """V0 for subspace iteration: seeded Gaussian d x k (the library holds no RNG)."""
    return torch.randn(d, k, generator=_gen(device, *seed, 21), device=device, dtype=torch.float32).contiguous()


# ---- the five configs of BASELINE.json ------------------------------------------------------------
@dataclass
class TensorSpec:
    name: str
    d_out: int
    d_in: int
    side: int
    rank: int               # k for both sides
    tokens: int             # T samples per factor
    layer: int = 0
    matrix: int = 0


@dataclass
class Config:
    index: int
    name: str
    R: int
    dtype: str              # "f32" | "bf16"
    damping: float
    fmt: int
    scaling: int
    tensors: List[TensorSpec] = field(default_factory=list)

    @property
    def n_elements(self) -> int:
        return sum(t.d_out * t.d_in for t in self.tensors)


def _llama(index, name, R, hidden, ffn, vocab, layers, k, tokens) -> Config:
    ts = []
    for l in range(layers):
        shapes = [("q", hidden, hidden), ("k", hidden, hidden), ("v", hidden, hidden), ("o", hidden, hidden),
                  ("gate", ffn, hidden), ("up", ffn, hidden), ("down", hidden, ffn)]
        for mi, (nm, m, n) in enumerate(shapes):
            ts.append(TensorSpec(f"l{l}.{nm}", m, n, SIDE_BOTH, k, tokens, l, mi))
    # selective application: embedding and LM head stay Euclidean (BASELINE.json configs[1])
    ts.append(TensorSpec("embed", vocab, hidden, SIDE_NONE, 0, 0, layers, 0))
    ts.append(TensorSpec("lm_head", vocab, hidden, SIDE_NONE, 0, 0, layers, 1))
    return Config(index, name, R, "bf16", 1e-3, E4M3, SCALE_TENSOR, ts)


def config(index: int, layers: Optional[int] = None) -> Config:
    if index == 0:
        return Config(0, "tiny-256", 2, "f32", 1e-3, E4M3, SCALE_TENSOR,
                      [TensorSpec("tiny", 256, 256, SIDE_BOTH, 16, 512)])
    if index == 1:
        return _llama(1, "llama300m-shaped", 4, 1024, 2816, 32000, layers or 24, 32, 4096)
    if index == 2:
        return _llama(2, "llama600m-shaped", 8, 1536, 4096, 32000, layers or 24, 64, 8192)
    if index == 4:
        return _llama(4, "llama600m-shaped-stress", 16, 1536, 4096, 32000, layers or 24, 64, 8192)
    raise ValueError("config 3 is a sweep: use sweep_tensor(k)")


def sweep_tensor(k: int) -> TensorSpec:
    """Config 3: one 4096 x 4096 BF16 gradient, factors from 16384 tokens."""
    return TensorSpec(f"sweep-k{k}", 4096, 4096, SIDE_BOTH, k, 16384)


def tensor_gradient(cfg: Config, t: TensorSpec, device) -> torch.Tensor:
    """The shared (seed-0) gradient of one tensor, in the config's storage dtype."""
    G = gradient(t.d_out, t.d_in, device, cfg.index, t.layer, t.matrix)
    return G.to(torch.bfloat16) if cfg.dtype == "bf16" else G


def tensor_rank_gradient(cfg: Config, t: TensorSpec, G: torch.Tensor, rank: int) -> torch.Tensor:
    Gr = rank_gradient(G, rank, cfg.index, t.layer, t.matrix)
    return Gr.to(torch.bfloat16) if cfg.dtype == "bf16" else Gr


def tensor_factor_samples(cfg: Config, t: TensorSpec, side: str, device, refresh: int = 0) -> torch.Tensor:
    """Activation (side='in', T x d_in) or output-gradient (side='out', T x d_out) samples."""
    d = t.d_in if side == "in" else t.d_out
    X = factor_samples(t.tokens, d, device, cfg.index, t.layer, t.matrix, 0 if side == "in" else 1, refresh)
    return X.to(torch.bfloat16) if cfg.dtype == "bf16" else X


def tensor_start_basis(cfg: Config, t: TensorSpec, side: str, device) -> torch.Tensor:
    d = t.d_in if side == "in" else t.d_out
    return start_basis(d, t.rank, device, cfg.index, t.layer, t.matrix, 0 if side == "in" else 1)
