"""Seeded synthetic inputs shaped like the paper's agent workloads (BASELINE.json configs 1-5).

This module holds NO arithmetic of the method: only shapes, lengths, page permutations and
i.i.d. Gaussian bf16 values.  It serves both sides of the parity tests (the CUDA path and the
fp64 oracle receive the very same bits) and belongs to neither.

The paper's evaluation is the authors' own agent runs on Qwen3 weights (PAPER.md L422-428,
L450-452); none of that exists here and none is needed, because the cost and the correctness of
the path depend on lengths only.  The shapes below take the paper's regime (context transformed
at ~15K tokens, up to 32K, L422/L450) and BASELINE.json's extrapolation of it; DESIGN.md
"Input recipe" states every draw.

Draw order (reading R13): lengths and page permutations from numpy default_rng(seed); values of
session i from a torch generator seeded with seed*1000003 + i on the device the caller asks for,
always in the order k, v, q (fp32 normal, scaled, rounded to bf16).  A session can therefore be
regenerated alone (config 5 never holds all raw inputs at once).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np
import torch

K = 1024


@dataclass
class Layer:
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    rope_base: float


@dataclass
class SessionSpec:
    prefix: int          # retained prefix already in the pool (prefix_j)
    new: int             # tokens appended and queried: segment length, or 1 for a decode row
    chunk: Optional[int] = None  # re-prefill the segment in chunks of this many tokens (None: one shot)

    @property
    def total(self) -> int:
        return self.prefix + self.new


@dataclass
class Workload:
    name: str
    layer: Layer
    sessions: List[SessionSpec]
    num_pages: int
    value_scale: float
    seed: int
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def max_session_tokens(self) -> int:
        return max(s.total for s in self.sessions)

    def pair_count(self) -> int:
        """sum_j A_j over the prefill sessions, A_j = q*prefix + q(q+1)/2."""
        return sum(s.new * s.prefix + s.new * (s.new + 1) // 2 for s in self.sessions if s.new > 1)

    def decode_kv_tokens(self) -> int:
        return sum(s.total for s in self.sessions if s.new == 1)

    def page_order(self) -> np.ndarray:
        """Random permutation of the pool = the order in which pages are handed out."""
        return np.random.default_rng(self.seed + 7919).permutation(self.num_pages).astype(np.int32)


LLAMA8B = Layer(32, 8, 128, 64, 500000.0)


def config1() -> Workload:
    return Workload("cfg1_tiny", Layer(8, 2, 64, 16, 10000.0), [SessionSpec(256, 128)], num_pages=64,
                    value_scale=1.0, seed=0, note="tiny single session; correctness config")


def config2() -> Workload:
    return Workload("cfg2_summarize", LLAMA8B, [SessionSpec(24 * K, 8 * K, chunk=2 * K)], num_pages=1024,
                    value_scale=128 ** -0.5, seed=2,
                    note="summarization-style: 24,576-token retained prefix, 8,192-token segment in 2,048-token chunks")


def config3() -> Workload:
    rng = np.random.default_rng(3)
    prefix = rng.integers(1 * K, 16 * K, size=16, endpoint=True)
    new = rng.integers(512, 4 * K, size=16, endpoint=True)
    return Workload("cfg3_offload16", LLAMA8B, [SessionSpec(int(p), int(n)) for p, n in zip(prefix, new)],
                    num_pages=10240, value_scale=128 ** -0.5, seed=3,
                    note="16 ragged sessions, offloading-style segments, one call")


def config4(n_decode: int = 64) -> Workload:
    rng = np.random.default_rng(4)
    ctx = rng.integers(8 * K, 32 * K, size=n_decode, endpoint=True)
    sessions = [SessionSpec(p * K, 2 * K) for p in (8, 16, 24, 32)]
    sessions += [SessionSpec(int(c) - 1, 1) for c in ctx]
    pages = sum((s.total + 63) // 64 for s in sessions)
    return Workload("cfg4_mixed", LLAMA8B, sessions, num_pages=int(pages * 1.25) + 64, value_scale=128 ** -0.5, seed=4,
                    note="4 lookahead chunks of 2,048 on 8K-32K prefixes + %d decode rows on 8K-32K contexts" % n_decode)


def config5(scale_down: int = 1) -> Workload:
    """scale_down > 1 shrinks every length by that factor (tests on small boxes); 1 = BASELINE.json."""
    rng = np.random.default_rng(5)
    prefix = rng.integers(32 * K, 112 * K, size=8, endpoint=True)
    ctx = rng.integers(32 * K, 128 * K, size=128, endpoint=True)
    sd = scale_down
    sessions = [SessionSpec(int(p) // sd, 16 * K // sd) for p in prefix]
    sessions += [SessionSpec(max(int(c) // sd, 2) - 1, 1) for c in ctx]
    layer = Layer(64, 8, 128, 64, 500000.0)
    used = sum((s.total + 63) // 64 for s in sessions)
    # ~120 GB of pages at full size (K+V: 256 KiB per page)
    pages = 458752 // sd if sd == 1 else int(used * 1.25) + 64
    return Workload("cfg5_long", layer, sessions, num_pages=max(pages, used + 8), value_scale=128 ** -0.5, seed=5,
                    note="8 sessions re-prefilling 16K segments after 32K-112K prefixes + 128 decode rows on 32K-128K")


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def gen_session(w: Workload, idx: int, device="cpu", scale: Optional[float] = None, with_prefix: bool = True):
    """Raw (pre-RoPE) inputs of session idx: k, v [total, Hkv, D], q [new, Hq, D], bf16.

    `scale` overrides w.value_scale (the "sharp" parity variants use 1.0 or 4.0 on q and k)."""
    s = w.sessions[idx]
    L = w.layer
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(w.seed * 1000003 + idx)
    sc = w.value_scale if scale is None else scale
    n_kv = s.total

    def draw(n, h, mult):
        x = torch.randn((n, h, L.head_dim), generator=g, device=dev, dtype=torch.float32)
        return (x * mult).to(torch.bfloat16)

    k = draw(n_kv, L.num_kv_heads, sc)
    v = draw(n_kv, L.num_kv_heads, w.value_scale)
    q = draw(s.new, L.num_q_heads, sc)
    return k, v, q


# ---- dense operators of the layer: random-init weights of BASELINE.json's "Llama-3-8B-shaped layer"
@dataclass
class LayerShape:
    hidden: int
    ffn: int
    rms_eps: float = 1e-5


LLAMA8B_DENSE = LayerShape(4096, 14336)


def gen_layer_weights(layer: Layer, shape: LayerShape, seed: int, device="cpu") -> dict:
    """bf16 tensors, weights [out_features, in_features] ~ N(0,1)/sqrt(in_features), norm gains ~ 1 + 0.1 N(0,1).
    Draw order: norm1, w_qkv, w_o, norm2, w_gate, w_up, w_down from one torch generator seeded seed*1000003 + 999."""
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(seed * 1000003 + 999)
    H, F, D = shape.hidden, shape.ffn, layer.head_dim
    QD, NQKV = layer.num_q_heads * D, (layer.num_q_heads + 2 * layer.num_kv_heads) * D

    def mat(n, k):
        return (torch.randn((n, k), generator=g, device=dev, dtype=torch.float32) * k ** -0.5).to(torch.bfloat16)

    def gain(n):
        return (1.0 + 0.1 * torch.randn((n,), generator=g, device=dev, dtype=torch.float32)).to(torch.bfloat16)

    return {"norm1": gain(H), "w_qkv": mat(NQKV, H), "w_o": mat(H, QD), "norm2": gain(H), "w_gate": mat(F, H),
            "w_up": mat(F, H), "w_down": mat(H, F)}


def gen_hidden(n_tokens: int, hidden: int, seed: int, device="cpu", scale: float = 1.0):
    """Hidden states x [n_tokens, hidden] ~ N(0, scale^2), bf16."""
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(seed * 1000003 + 555)
    return (torch.randn((n_tokens, hidden), generator=g, device=dev, dtype=torch.float32) * scale).to(torch.bfloat16)
