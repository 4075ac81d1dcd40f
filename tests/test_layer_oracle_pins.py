"""Pins of oracle/layer_oracle.py (the dense operators of a layer) against things
other than itself: values worked by hand (tests/golden/layer_worked_example.txt), closed forms,
invariants, pure-Python brute force and torch's fp64 library routines.  No GPU."""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import layer_oracle as lo
from oracle import oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden", "layer_worked_example.txt")


def _gold():
    vals = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if not line:
            continue
        key, rest = line.split("=", 1)
        vals[key.strip()] = np.array([float(t) for t in rest.replace(",", " ").split()])
    return vals


# ------------------------------------------------------------------ linear
def test_linear_hand_example():
    g = _gold()
    x = np.array([[1.0, 2.0, 3.0], [0.0, -1.0, 2.0]])
    w = np.array([[1.0, 0.0, 1.0], [2.0, 1.0, 0.0]])       # [out=2, in=3]
    assert np.array_equal(lo.linear(x, w).ravel(), g["linear_y"])


def test_linear_brute_force_nonsquare():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((5, 7))
    w = rng.standard_normal((3, 7))
    ref = [[sum(x[t, k] * w[n, k] for k in range(7)) for n in range(3)] for t in range(5)]
    assert np.allclose(lo.linear(x, w), np.array(ref), rtol=0, atol=1e-13)
    assert lo.linear(x, w).shape == (5, 3)


def test_linear_identity_and_selection():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((4, 6))
    assert np.array_equal(lo.linear(x, np.eye(6)), x)
    sel = np.zeros((2, 6))
    sel[0, 4] = 1.0
    sel[1, 1] = -2.0
    assert np.array_equal(lo.linear(x, sel), np.stack([x[:, 4], -2.0 * x[:, 1]], axis=1))


# ------------------------------------------------------------------ RMSNorm
def test_rmsnorm_hand_and_eps_inside_sqrt():
    g = _gold()
    y = lo.rmsnorm(np.array([[3.0, 4.0]]), np.array([1.0, 2.0]), 0.0)
    assert np.allclose(y.ravel(), g["rmsnorm_34"], rtol=0, atol=1e-15)
    # x = (1,1), eps = 3: 1/sqrt(1+3) = 0.5 (eps added under the root, R22); outside the root it would be 0.25
    assert np.allclose(lo.rmsnorm(np.array([[1.0, 1.0]]), np.ones(2), 3.0), 0.5, rtol=0, atol=1e-15)
    assert np.array_equal(lo.rmsnorm(np.zeros((1, 4)), np.ones(4), 1e-5), np.zeros((1, 4)))


def test_rmsnorm_invariants():
    rng = np.random.default_rng(2)
    x = rng.standard_normal((6, 32))
    w = rng.standard_normal(32)
    y = lo.rmsnorm(x, w, 0.0)
    assert np.allclose(lo.rmsnorm(7.5 * x, w, 0.0), y, rtol=0, atol=1e-13)          # scale invariance
    assert np.allclose(np.mean((y / w) ** 2, axis=-1), 1.0, rtol=0, atol=1e-13)      # unit mean square
    c = lo.rmsnorm(np.full((1, 8), -2.5), np.arange(1.0, 9.0), 0.0)
    assert np.allclose(c, -np.arange(1.0, 9.0), rtol=0, atol=1e-14)                  # constant row -> sign * w
    t = F.rms_norm(torch.from_numpy(x), (32,), torch.from_numpy(w), eps=1e-5).numpy()
    assert np.allclose(lo.rmsnorm(x, w, 1e-5), t, rtol=0, atol=1e-13)


# ------------------------------------------------------------------ SiLU / SwiGLU
def test_silu_closed_forms():
    assert lo.silu(0.0) == 0.0
    assert math.isclose(float(lo.silu(math.log(3.0))), math.log(3.0) * 0.75, rel_tol=1e-15)   # sigma(ln 3) = 3/4
    z = np.linspace(-20, 20, 101)
    assert np.allclose(lo.silu(z) - lo.silu(-z), z, rtol=0, atol=1e-13)               # z (sigma(z) + sigma(-z)) = z
    assert np.allclose(lo.silu(z), F.silu(torch.from_numpy(z)).numpy(), rtol=0, atol=1e-14)
    assert abs(float(lo.silu(40.0)) - 40.0) < 1e-12 and abs(float(lo.silu(-40.0))) < 1e-12


def test_swiglu_gate_is_the_silu_branch():
    g = _gold()
    h = np.array([[1.0]])
    out = lo.swiglu_ffn(h, np.array([[math.log(3.0)]]), np.array([[2.0]]), np.array([[5.0]]))
    # SiLU(ln 3) * 2 * 5 = 7.5 ln 3 ; with gate and up swapped it would be SiLU(2) * ln 3 * 5
    assert math.isclose(float(out[0, 0]), float(g["swiglu_scalar"][0]), rel_tol=1e-12)
    assert math.isclose(float(out[0, 0]), 7.5 * math.log(3.0), rel_tol=1e-15)


def test_swiglu_hidden_permutation_and_library():
    rng = np.random.default_rng(3)
    h = rng.standard_normal((5, 8))
    wg, wu = rng.standard_normal((12, 8)), rng.standard_normal((12, 8))
    wd = rng.standard_normal((8, 12))
    y = lo.swiglu_ffn(h, wg, wu, wd)
    p = rng.permutation(12)
    assert np.allclose(lo.swiglu_ffn(h, wg[p], wu[p], wd[:, p]), y, rtol=0, atol=1e-12)
    th = torch.from_numpy(h)
    t = F.linear(F.silu(F.linear(th, torch.from_numpy(wg))) * F.linear(th, torch.from_numpy(wu)), torch.from_numpy(wd))
    assert np.allclose(y, t.numpy(), rtol=0, atol=1e-12)
    assert np.allclose(lo.linear(lo.swiglu_act(h, wg, wu), wd), y, rtol=0, atol=1e-13)
    assert np.array_equal(lo.swiglu_ffn(h, np.zeros_like(wg), wu, wd), np.zeros((5, 8)))   # SiLU(0) = 0


# ------------------------------------------------------------------ QKV projection
def test_qkv_head_order():
    Hq, Hkv, D, H = 4, 2, 2, 16
    rng = np.random.default_rng(4)
    h = rng.standard_normal((3, H))
    w = np.zeros(((Hq + 2 * Hkv) * D, H))
    for r in range(w.shape[0]):
        w[r, r] = 1.0                      # output feature r = hidden feature r
    q, k, v = lo.qkv_project(h, w, Hq, Hkv, D)
    assert q.shape == (3, Hq, D) and k.shape == (3, Hkv, D) and v.shape == (3, Hkv, D)
    assert np.array_equal(q[:, 2, 1], h[:, 2 * D + 1])
    assert np.array_equal(k[:, 1, 0], h[:, Hq * D + 1 * D + 0])
    assert np.array_equal(v[:, 0, 1], h[:, (Hq + Hkv) * D + 1])


def test_qkv_rope_position_zero_is_projection():
    rng = np.random.default_rng(5)
    h = rng.standard_normal((1, 8))
    w = rng.standard_normal((4 * 4, 8))    # Hq=2, Hkv=1, D=4
    q, k, v = lo.qkv_project(h, w, 2, 1, 4)
    qr, kr, vr = lo.qkv_rope(h, w, 2, 1, 4, [0], 10000.0)
    assert np.array_equal(qr, q) and np.array_equal(kr, k) and np.array_equal(vr, v)
    # position 1, pair (0, D/2) rotates by 1 rad (oracle.rope is pinned in test_oracle_pins.py)
    qr1, _, _ = lo.qkv_rope(h, w, 2, 1, 4, [1], 10000.0)
    assert math.isclose(qr1[0, 0, 0], q[0, 0, 0] * math.cos(1.0) - q[0, 0, 2] * math.sin(1.0), rel_tol=1e-12)


# ------------------------------------------------------------------ the whole layer
def _weights(rng, H, Hq, Hkv, D, Fh, s=0.3):
    return {"norm1": 1.0 + 0.1 * rng.standard_normal(H), "w_qkv": s * rng.standard_normal(((Hq + 2 * Hkv) * D, H)),
            "w_o": s * rng.standard_normal((H, Hq * D)), "norm2": 1.0 + 0.1 * rng.standard_normal(H),
            "w_gate": s * rng.standard_normal((Fh, H)), "w_up": s * rng.standard_normal((Fh, H)),
            "w_down": s * rng.standard_normal((H, Fh))}


def test_layer_residual_structure():
    rng = np.random.default_rng(6)
    H, Hq, Hkv, D, Fh, T = 16, 4, 2, 4, 24, 5
    W = _weights(rng, H, Hq, Hkv, D, Fh)
    x = rng.standard_normal((T, H))
    empty = np.zeros((0, Hkv, D))
    W0 = dict(W, w_o=np.zeros_like(W["w_o"]), w_down=np.zeros_like(W["w_down"]))
    assert np.array_equal(lo.layer_forward(x, W0, Hq, Hkv, D, 1e-5, 1e4, empty, empty, 0)["y"], x)
    # with the FFN off, y - x is linear in W_o
    W1 = dict(W, w_down=np.zeros_like(W["w_down"]))
    W2 = dict(W1, w_o=2.0 * W["w_o"])
    y1 = lo.layer_forward(x, W1, Hq, Hkv, D, 1e-5, 1e4, empty, empty, 0)["y"]
    y2 = lo.layer_forward(x, W2, Hq, Hkv, D, 1e-5, 1e4, empty, empty, 0)["y"]
    assert np.allclose(y2 - x, 2.0 * (y1 - x), rtol=0, atol=1e-12)


def test_layer_against_torch_library_composition():
    """prefix = 0: torch fp64 rms_norm / linear / scaled_dot_product_attention(is_causal) / silu composed by
    hand; RoPE of q and k through oracle.rope (pinned on its own by the closed forms of test_oracle_pins)."""
    rng = np.random.default_rng(7)
    H, Hq, Hkv, D, Fh, T = 32, 4, 2, 8, 40, 9
    W = _weights(rng, H, Hq, Hkv, D, Fh)
    x = rng.standard_normal((T, H))
    empty = np.zeros((0, Hkv, D))
    got = lo.layer_forward(x, W, Hq, Hkv, D, 1e-5, 1e4, empty, empty, 0)

    tx = torch.from_numpy(x)
    tw = {k: torch.from_numpy(v) for k, v in W.items()}
    h = F.rms_norm(tx, (H,), tw["norm1"], eps=1e-5)
    qkv = F.linear(h, tw["w_qkv"])
    q = qkv[:, : Hq * D].reshape(T, Hq, D).numpy()
    k = qkv[:, Hq * D: (Hq + Hkv) * D].reshape(T, Hkv, D).numpy()
    v = qkv[:, (Hq + Hkv) * D:].reshape(T, Hkv, D)
    pos = np.arange(T)
    qr = torch.from_numpy(orc.rope(q, pos, 1e4)).permute(1, 0, 2)                       # [Hq, T, D]
    kr = torch.from_numpy(orc.rope(k, pos, 1e4)).permute(1, 0, 2).repeat_interleave(Hq // Hkv, dim=0)
    vv = v.permute(1, 0, 2).repeat_interleave(Hq // Hkv, dim=0)
    a = F.scaled_dot_product_attention(qr[None], kr[None], vv[None], is_causal=True)[0]  # [Hq, T, D]
    a = a.permute(1, 0, 2).reshape(T, Hq * D)
    x1 = tx + F.linear(a, tw["w_o"])
    h2 = F.rms_norm(x1, (H,), tw["norm2"], eps=1e-5)
    y = x1 + F.linear(F.silu(F.linear(h2, tw["w_gate"])) * F.linear(h2, tw["w_up"]), tw["w_down"])
    assert np.allclose(got["y"], y.numpy(), rtol=0, atol=1e-10)
    assert np.allclose(got["x1"], x1.numpy(), rtol=0, atol=1e-11)


def test_layer_segment_decomposability():
    """prefilling a segment over the cached K', V of the layer's own prefix equals
    rows P.. of the one-shot layer over the whole context (the dense operators act per token)."""
    rng = np.random.default_rng(8)
    H, Hq, Hkv, D, Fh, L, P = 16, 2, 1, 4, 20, 10, 6
    W = _weights(rng, H, Hq, Hkv, D, Fh)
    x = rng.standard_normal((L, H))
    empty = np.zeros((0, Hkv, D))
    full = lo.layer_forward(x, W, Hq, Hkv, D, 1e-5, 1e4, empty, empty, 0)
    seg = lo.layer_forward(x[P:], W, Hq, Hkv, D, 1e-5, 1e4, full["k_rot"][:P], full["v"][:P], P)
    assert np.allclose(seg["y"], full["y"][P:], rtol=0, atol=1e-12)
