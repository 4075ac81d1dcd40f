"""Pins for the fp64 oracle (oracle/): it is checked against things other than itself.

Each test names the pin of SURVEY.md section 8(c) / DESIGN.md it implements and the PAPER.md
passage behind it.  None of these needs a GPU.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand(shape, seed, scale=1.0):
    return np.random.default_rng(seed).standard_normal(shape) * scale


# ---------------------------------------------------------------- brute force (P1)
def _brute_attention(q_rot, k_rot, v, P, scale):
    """Full N x L score matrix with an explicit boolean mask, softmax by numpy; a route that
    shares nothing with the row-by-row C loop."""
    N, Hq, D = q_rot.shape
    L, Hkv, _ = k_rot.shape
    G = Hq // Hkv
    o = np.zeros((N, Hq, D))
    lse = np.zeros((N, Hq))
    allowed = np.arange(L)[None, :] <= (P + np.arange(N))[:, None]
    for h in range(Hq):
        s = scale * (q_rot[:, h, :] @ k_rot[:, h // G, :].T)
        s = np.where(allowed, s, -np.inf)
        m = s.max(axis=1, keepdims=True)
        e = np.exp(s - m)
        z = e.sum(axis=1, keepdims=True)
        o[:, h, :] = (e / z) @ v[:, h // G, :]
        lse[:, h] = (m + np.log(z))[:, 0]
    return o, lse


@pytest.mark.parametrize("D", [8, 64])
@pytest.mark.parametrize("Hq,Hkv", [(1, 1), (4, 1), (4, 4), (8, 2)])
@pytest.mark.parametrize("P,N", [(0, 1), (0, 17), (5, 1), (23, 41), (0, 64)])
def test_p1_brute_force(D, Hq, Hkv, P, N):
    L = P + N
    q = _rand((N, Hq, D), 1)
    k = _rand((L, Hkv, D), 2)
    v = _rand((L, Hkv, D), 3)
    scale = 0.37
    res = orc.attend(q, k, v, P, scale)
    o, lse = _brute_attention(q, k, v, P, scale)
    assert np.abs(res["o"] - o).max() <= 1e-12
    assert np.abs(res["lse"] - lse).max() <= 1e-12


def test_p1_hand_cases():
    # L = 1: the only key gets probability 1, so o = v_0 and lse = s_00.
    q = np.array([[[0.5, -2.0]]])
    k = np.array([[[3.0, 1.0]]])
    v = np.array([[[7.0, -9.0]]])
    r = orc.attend(q, k, v, 0, 1.0)
    assert np.array_equal(r["o"][0, 0], v[0, 0])
    assert abs(r["lse"][0, 0] - (0.5 * 3.0 - 2.0 * 1.0)) <= 1e-15
    # L = 2 with equal scores: row 1 averages v_0 and v_1; row 0 sees only v_0.
    q = np.array([[[1.0, 0.0]], [[1.0, 0.0]]])
    k = np.array([[[2.0, 5.0]], [[2.0, -4.0]]])
    v = np.array([[[1.0, 10.0]], [[3.0, 20.0]]])
    r = orc.attend(q, k, v, 0, 1.0)
    assert np.allclose(r["o"][0, 0], [1.0, 10.0], atol=1e-15)
    assert np.allclose(r["o"][1, 0], [2.0, 15.0], atol=1e-15)
    assert abs(r["lse"][1, 0] - (2.0 + math.log(2.0))) <= 1e-15
    # scores ln 1, ln 3 -> probabilities 1/4, 3/4 (a transposed q/k or a dropped scale fails this)
    q = np.array([[[1.0, 0.0]]])
    k = np.array([[[0.0, 9.0]], [[math.log(3.0) / 0.5, -9.0]]])
    v = np.array([[[4.0, 0.0]], [[8.0, 4.0]]])
    r = orc.attend(q, k, v, 1, 0.5)
    assert np.allclose(r["o"][0, 0], [7.0, 3.0], atol=1e-14)


# ---------------------------------------------------------------- RoPE closed forms (P2a, P2b)
@pytest.mark.parametrize("D,base", [(8, 10000.0), (64, 10000.0), (128, 500000.0)])
def test_p2a_rope_closed_forms(D, base):
    half = D // 2
    x = _rand((5, 3, D), 4)
    # position 0 is the identity, bit for bit
    assert np.array_equal(orc.rope(x, np.zeros(5, dtype=np.int64), base), x)
    # e_0 at p = 1: theta_0 = 1 -> (cos 1, sin 1) in slots 0 and D/2
    e0 = np.zeros((1, 1, D))
    e0[0, 0, 0] = 1.0
    r = orc.rope(e0, [1], base)[0, 0]
    expect = np.zeros(D)
    expect[0], expect[half] = math.cos(1.0), math.sin(1.0)
    assert np.abs(r - expect).max() <= 1e-15
    # e_{m+D/2} at p: -sin in slot m, +cos in slot m+D/2 (sign and pairing)
    for m in (0, 1, half - 1):
        for p in (1, 7, 383, 131071):
            ang = p * base ** (-2.0 * m / D)
            em = np.zeros((1, 1, D))
            em[0, 0, m] = 1.0
            r = orc.rope(em, [p], base)[0, 0]
            expect = np.zeros(D)
            expect[m], expect[m + half] = math.cos(ang), math.sin(ang)
            assert np.abs(r - expect).max() <= 1e-9
            eh = np.zeros((1, 1, D))
            eh[0, 0, m + half] = 1.0
            r = orc.rope(eh, [p], base)[0, 0]
            expect = np.zeros(D)
            expect[m], expect[m + half] = -math.sin(ang), math.cos(ang)
            assert np.abs(r - expect).max() <= 1e-9
    # pairwise norms preserved
    pos = np.array([0, 1, 17, 4096, 131071])
    r = orc.rope(x, pos, base)
    n0 = x[..., :half] ** 2 + x[..., half:] ** 2
    n1 = r[..., :half] ** 2 + r[..., half:] ** 2
    assert np.abs(n0 - n1).max() <= 1e-12


def test_p2a_rope_complex_route():
    # The half-split rotation is multiplication of z_m = x[m] + i x[m+D/2] by exp(i p theta_m).
    D, base = 64, 10000.0
    half = D // 2
    x = _rand((9, 2, D), 5)
    pos = np.array([0, 1, 2, 3, 100, 255, 256, 383, 9999])
    z = x[..., :half] + 1j * x[..., half:]
    theta = base ** (-2.0 * np.arange(half) / D)
    zr = z * np.exp(1j * pos[:, None, None] * theta[None, None, :])
    r = orc.rope(x, pos, base)
    assert np.abs(r[..., :half] - zr.real).max() <= 1e-11
    assert np.abs(r[..., half:] - zr.imag).max() <= 1e-11


def test_p2b_rope_relative_position():
    # <RoPE(q,a), RoPE(k,b)> depends on a-b only: shifting all positions leaves outputs unchanged.
    D, Hq, Hkv, L, base = 64, 4, 2, 40, 10000.0
    q = _rand((L, Hq, D), 6)
    k = _rand((L, Hkv, D), 7)
    v = _rand((L, Hkv, D), 8)
    outs = []
    for shift in (0, 11, 1000):
        pos = np.arange(L) + shift
        r = orc.attend(orc.rope(q, pos, base), orc.rope(k, pos, base), v, 0)
        outs.append(r["o"])
    assert np.abs(outs[0] - outs[1]).max() <= 1e-9
    assert np.abs(outs[0] - outs[2]).max() <= 1e-9


# ---------------------------------------------------------------- closed forms through attention
def test_p2c_uniform_softmax_cumulative_mean():
    # Q = 0 -> row i averages v_0..v_{P+i}; lse_i = ln(P+i+1).  PAPER.md L311: prefix + i + 1 keys.
    D, Hq, Hkv, P, N = 16, 4, 2, 37, 29
    L = P + N
    q = np.zeros((N, Hq, D))
    k = _rand((L, Hkv, D), 9)
    v = _rand((L, Hkv, D), 10)
    r = orc.oracle_cached(orc.rope(k[:P], np.arange(P), 1e4), v[:P], q, k[P:], v[P:], P, 1e4)
    cm = np.cumsum(v, axis=0) / np.arange(1, L + 1)[:, None, None]
    for h in range(Hq):
        assert np.abs(r["o"][:, h] - cm[P:, h // 2]).max() <= 1e-13
    assert np.abs(r["lse"] - np.log(P + 1 + np.arange(N))[:, None]).max() <= 1e-13


def test_p2d_constant_v_and_p3d_rows_sum_to_one():
    D, Hq, Hkv, P, N = 8, 2, 1, 6, 10
    L = P + N
    q = _rand((N, Hq, D), 11, 3.0)
    k = _rand((L, Hkv, D), 12, 3.0)
    c = _rand((D,), 13)
    v = np.broadcast_to(c, (L, Hkv, D)).copy()
    r = orc.attend(q, k, v, P, None, return_probs=True)
    assert np.abs(r["o"] - c).max() <= 1e-13
    assert np.abs(r["probs"].sum(axis=-1) - 1.0).max() <= 1e-12
    # and masked entries are exactly zero
    for i in range(N):
        assert np.all(r["probs"][i, :, P + i + 1:] == 0.0)
        assert np.all(r["probs"][i, :, :P + i + 1] > 0.0)


def test_p2e_spike_no_overflow():
    D, L = 8, 50
    q = np.zeros((1, 1, D))
    q[0, 0, 0] = 1.0
    k = _rand((L, 1, D), 14, 0.01)
    k[17, 0, 0] = 5000.0  # exp(5000) overflows unless the max is subtracted
    v = _rand((L, 1, D), 15)
    r = orc.attend(q, k, v, L - 1, 1.0)
    assert np.all(np.isfinite(r["o"])) and np.isfinite(r["lse"]).all()
    assert np.abs(r["o"][0, 0] - v[17, 0]).max() <= 1e-12


def test_p2f_pair_count_golden():
    # A_j = q*prefix + q(q+1)/2; fixture worked by hand from the closed form.
    rows = [l.split() for l in open(os.path.join(GOLDEN, "pair_counts.txt")) if l.strip() and l[0] != "#"]
    for qs, ps, As in rows:
        qn, P, A = int(qs), int(ps), int(As)
        assert qn * P + qn * (qn + 1) // 2 == A
        if A > 3_000_000:
            continue  # closed form checked above; the oracle visit count on the small ones
        D = 2
        q = np.zeros((qn, 1, D))
        k = np.zeros((P + qn, 1, D))
        r = orc.attend(q, k, k, P)
        assert r["pairs"] == A


# ---------------------------------------------------------------- invariants (P3)
def _ctx(L, Hq, Hkv, D, seed):
    return _rand((L, Hq, D), seed), _rand((L, Hkv, D), seed + 1), _rand((L, Hkv, D), seed + 2)


def test_p3a_segment_decomposability():
    # prefix KV + segment prefill == one-shot prefill of the whole context.
    D, Hq, Hkv, P, N, base = 64, 8, 2, 48, 33, 10000.0
    L = P + N
    q, k, v = _ctx(L, Hq, Hkv, D, 20)
    full = orc.oracle_full(q, k, v, base)
    # the stored prefix is produced by a separate, earlier call that never sees the segment
    k_rot_prefix = orc.rope(k[:P], np.arange(P), base)
    cached = orc.oracle_cached(k_rot_prefix, v[:P], q[P:], k[P:], v[P:], P, base)
    assert np.abs(cached["o"] - full["o"][P:]).max() <= 1e-12
    assert np.abs(cached["lse"] - full["lse"][P:]).max() <= 1e-12
    # chunked (11 tokens at a time, each chunk appended to the stored prefix) == one-shot
    kp, vp = k_rot_prefix, v[:P]
    outs = []
    for s in range(P, L, 11):
        e = min(L, s + 11)
        c = orc.oracle_cached(kp, vp, q[s:e], k[s:e], v[s:e], s, base)
        outs.append(c["o"])
        kp = np.concatenate([kp, c["k_rot_seg"]])
        vp = np.concatenate([vp, v[s:e]])
    assert np.abs(np.concatenate(outs) - full["o"][P:]).max() <= 1e-12
    assert np.abs(kp - full["k_rot"]).max() <= 1e-12


def test_p3b_prefix_independence_and_p3c_causality():
    # "the transformation of each segment is independent of the tokens that follow".
    D, Hq, Hkv, L, base = 32, 4, 4, 30, 10000.0
    q, k, v = _ctx(L, Hq, Hkv, D, 30)
    a = orc.oracle_full(q, k, v, base)
    i = 13
    q2, k2, v2 = q.copy(), k.copy(), v.copy()
    q2[i + 1:] += 5.0
    k2[i + 1:] *= -3.0
    v2[i + 1:] = 1e6
    b = orc.oracle_full(q2, k2, v2, base)
    assert np.array_equal(a["k_rot"][: i + 1], b["k_rot"][: i + 1])  # stored prefix K' unchanged
    assert np.array_equal(a["o"][: i + 1], b["o"][: i + 1])          # rows <= i unchanged, exactly
    assert np.array_equal(a["lse"][: i + 1], b["lse"][: i + 1])
    assert not np.allclose(a["o"][i + 1:], b["o"][i + 1:])


# ---------------------------------------------------------------- GQA (P4)
def test_p4_gqa_special_cases():
    D, Hq, Hkv, P, N = 16, 8, 2, 9, 12
    G = Hq // Hkv
    L = P + N
    q = _rand((N, Hq, D), 40)
    k = _rand((L, Hkv, D), 41)
    v = _rand((L, Hkv, D), 42)
    r = orc.attend(q, k, v, P)
    # replicate each kv head G times and run as plain MHA (G = 1): head h must pick kv head h // G
    r1 = orc.attend(q, np.repeat(k, G, axis=1), np.repeat(v, G, axis=1), P)
    assert np.abs(r["o"] - r1["o"]).max() <= 1e-14
    # equal q heads inside one group give equal outputs; across groups they do not
    q2 = q.copy()
    q2[:, 1] = q2[:, 0]
    q2[:, G] = q2[:, 0]
    r2 = orc.attend(q2, k, v, P)
    assert np.array_equal(r2["o"][:, 0], r2["o"][:, 1])
    assert not np.allclose(r2["o"][:, 0], r2["o"][:, G])


# ---------------------------------------------------------------- library special case (P5)
@pytest.mark.parametrize("P", [0, 19])
def test_p5_torch_sdpa(P):
    D, H, N = 32, 3, 21
    L = P + N
    q = _rand((N, H, D), 50)
    k = _rand((L, H, D), 51)
    v = _rand((L, H, D), 52)
    r = orc.attend(q, k, v, P)  # G = 1, no RoPE: textbook causal attention
    tq = torch.from_numpy(q).permute(1, 0, 2)[None]
    tk = torch.from_numpy(k).permute(1, 0, 2)[None]
    tv = torch.from_numpy(v).permute(1, 0, 2)[None]
    if P == 0:
        ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, is_causal=True)
    else:
        mask = torch.arange(L)[None, :] <= (P + torch.arange(N))[:, None]
        ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, attn_mask=mask)
    ref = ref[0].permute(1, 0, 2).numpy()
    assert np.abs(r["o"] - ref).max() <= 1e-12


def test_sampled_rows_equal_full():
    D, Hq, Hkv, P, N = 16, 4, 2, 7, 20
    L = P + N
    q = _rand((N, Hq, D), 60)
    k = _rand((L, Hkv, D), 61)
    v = _rand((L, Hkv, D), 62)
    full = orc.attend(q, k, v, P)
    rows = np.array([0, 19, 5, 5, 12])
    heads = np.array([0, 3, 1, 2, 0], dtype=np.int32)
    s = orc.attend(q, k, v, P, rows=rows, heads=heads)
    assert np.array_equal(s["o"], full["o"][rows, heads])
    assert np.array_equal(s["lse"], full["lse"][rows, heads])


def test_widen_bf16_is_exact():
    t = torch.randn(64, generator=torch.Generator().manual_seed(0)).to(torch.bfloat16)
    w = orc.widen(t)
    assert w.dtype == np.float64
    assert np.array_equal(w.astype(np.float32), t.float().numpy())


def test_wire_image_is_the_stated_reindexing():
    """N4 hand-over image (PAPER.md L426 / L424): image[c][h][t][d] = (K', V)[c][t][head_begin + h][d].
    Hand-written tiny case, the library transpose, and the head slice of a sharded receiver."""
    # n = 2 tokens, Hkv = 2, D = 2; entries encode (tensor, token, head, dim) so a wrong index order shows
    k = np.array([[[100, 101], [110, 111]], [[200, 201], [210, 211]]], dtype=np.float64)        # [t][h][d]
    v = -k
    img = orc.wire_image(k, v)
    expect_k = [[[100, 101], [200, 201]], [[110, 111], [210, 211]]]                                # [h][t][d]
    assert img.shape == (2, 2, 2, 2)
    assert img[0].tolist() == expect_k and img[1].tolist() == (-np.array(expect_k)).tolist()
    rng = np.random.default_rng(0)
    k, v = rng.standard_normal((7, 4, 6)), rng.standard_normal((7, 4, 6))
    img = orc.wire_image(k, v)
    assert np.array_equal(img[0], np.transpose(k, (1, 0, 2))) and np.array_equal(img[1], np.transpose(v, (1, 0, 2)))
    part = orc.wire_image(k, v, head_begin=1, head_count=2)
    assert np.array_equal(part, img[:, 1:3])
    # concatenating token ranges of images = image of the concatenation (in-order import)
    a, b = orc.wire_image(k[:3], v[:3]), orc.wire_image(k[3:], v[3:])
    assert np.array_equal(np.concatenate([a, b], axis=2), img)
