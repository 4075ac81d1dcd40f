"""fp64 oracle of the dense operators of a transformer layer -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md section 4, "GEMM" (L299-303): "All tokens in the batch, including decode tokens and prefill
chunk tokens, are processed by the same dense operators in each transformer layer, including the
projection matrices in attention (QKV and output projections) and the FFN layers."  The paper names
the operators and nothing else; the layer's shape is BASELINE.json's "Llama-3-8B-shaped layer" and
the models the paper runs use "grouped-query attention and dense feed-forward layers" (L422).

This file is the plain DEFINITION of those operators in float64 (numpy), each written as the
textbook formula with numpy's matmul as the library primitive -- no blocking, no fusion, no
reordering.  Readings (R21-R24), all from BASELINE.json's "Llama-3-8B-shaped",
none from the paper:

* R21  pre-norm decoder layer without biases:
          h  = RMSNorm(x; w_norm1)                 q|k|v = h W_qkv^T   (rows of W_qkv: Hq heads of Q,
          a  = attention(RoPE(q), RoPE(k), v)                            then Hkv heads of K, then V)
          x1 = x + a W_o^T
          h2 = RMSNorm(x1; w_norm2)
          y  = x1 + (SiLU(h2 W_gate^T) * (h2 W_up^T)) W_down^T
* R22  RMSNorm(x; w)_i = x_i / sqrt(mean_j x_j^2 + eps) * w_i, eps inside the square root.
* R23  SiLU(z) = z / (1 + exp(-z)); the gate is the SiLU branch (SwiGLU).
* R24  weights are stored [out_features, in_features] (y = x W^T), no QK-norm, no bias.

Inputs are the bf16 bit patterns the CUDA path receives, widened exactly to float64; nothing is
rounded in between (the CUDA path rounds every tensor it stores to bf16: DESIGN.md derives the
tolerance from that).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It imports nothing of paper_2607_00151_b200; the attention step calls oracle.oracle (same
directory).  Pins: tests/test_layer_oracle_pins.py.
"""
from __future__ import annotations

from typing import Optional

import numpy as np

from . import oracle as _att


def widen(x) -> np.ndarray:
    return _att.widen(x)


def linear(x, w) -> np.ndarray:
    """y[t, n] = sum_k x[t, k] * w[n, k]        (R24)"""
    x = widen(x)
    w = widen(w)
    assert x.ndim == 2 and w.ndim == 2 and x.shape[1] == w.shape[1]
    return x @ w.T


def rmsnorm(x, w, eps: float) -> np.ndarray:
    """R22."""
    x = widen(x)
    w = widen(w)
    ms = np.mean(x * x, axis=-1, keepdims=True)
    return x / np.sqrt(ms + eps) * w


def silu(z) -> np.ndarray:
    """R23."""
    z = np.asarray(z, dtype=np.float64)
    return z / (1.0 + np.exp(-z))


def swiglu_ffn(h, w_gate, w_up, w_down) -> np.ndarray:
    """(SiLU(h W_gate^T) * (h W_up^T)) W_down^T"""
    g = linear(h, w_gate)
    u = linear(h, w_up)
    return linear(silu(g) * u, w_down)


def swiglu_act(h, w_gate, w_up) -> np.ndarray:
    """The FFN's hidden activation SiLU(h W_gate^T) * (h W_up^T)   [T, ffn]"""
    return silu(linear(h, w_gate)) * linear(h, w_up)


def qkv_project(h, w_qkv, Hq: int, Hkv: int, D: int):
    """q [T,Hq,D], k [T,Hkv,D], v [T,Hkv,D] from one projection; rows of w_qkv ordered Q heads, K heads, V heads (R21)."""
    y = linear(h, w_qkv)
    T = y.shape[0]
    assert y.shape[1] == (Hq + 2 * Hkv) * D
    q = y[:, : Hq * D].reshape(T, Hq, D)
    k = y[:, Hq * D: (Hq + Hkv) * D].reshape(T, Hkv, D)
    v = y[:, (Hq + Hkv) * D:].reshape(T, Hkv, D)
    return q, k, v


def qkv_rope(h, w_qkv, Hq: int, Hkv: int, D: int, positions, rope_base: float):
    """Projection followed by RoPE of q and k at the given absolute positions: what the fused
    QKV-projection + RoPE + append call stores (k_rot, v) and hands to attention (q_rot)."""
    q, k, v = qkv_project(h, w_qkv, Hq, Hkv, D)
    pos = np.asarray(positions, dtype=np.int64)
    return _att.rope(q, pos, rope_base), _att.rope(k, pos, rope_base), v


def layer_forward(x, weights: dict, Hq: int, Hkv: int, D: int, eps: float, rope_base: float,
                  k_rot_prefix, v_prefix, P: int, sm_scale: Optional[float] = None) -> dict:
    """One decoder layer (R21) over a segment of T tokens at positions P..P+T-1 whose retained prefix
    (k_rot_prefix [P,Hkv,D] rotated, v_prefix [P,Hkv,D]) is already cached.

    weights: {"norm1" [H], "w_qkv" [(Hq+2Hkv)D, H], "w_o" [H, Hq*D], "norm2" [H], "w_gate" [F, H],
              "w_up" [F, H], "w_down" [H, F]}.  Returns y [T, H] and the intermediates."""
    x = widen(x)
    T = x.shape[0]
    h = rmsnorm(x, weights["norm1"], eps)
    q, k, v = qkv_project(h, weights["w_qkv"], Hq, Hkv, D)
    att = _att.oracle_cached(k_rot_prefix, v_prefix, q, k, v, P, rope_base, sm_scale)
    a = att["o"].reshape(T, Hq * D)
    x1 = x + linear(a, weights["w_o"])
    h2 = rmsnorm(x1, weights["norm2"], eps)
    y = x1 + swiglu_ffn(h2, weights["w_gate"], weights["w_up"], weights["w_down"])
    return {"y": y, "h": h, "q_rot": att["q_rot"], "k_rot": att["k_rot_seg"], "v": v, "attn": att["o"], "x1": x1, "h2": h2}
