"""GPU parity of the layer's dense operators through the C ABI
against oracle/layer_oracle.py on the same seeded bf16 inputs.  Run with -m gpu on a B200.

Tolerance: inputs are bf16 and exact in fp64; the tensor cores accumulate in
fp32 (error ~ 2^-24 sqrt(K) |y|, negligible) and every stored tensor is rounded once to bf16
(half an ulp = 2^-9 relative), so an element of a single operator is within 2^-8 |ref| + 1e-3 rms(ref)
of the fp64 definition and the normalised L2 error is ~ 1.7e-3 (gate 4e-3); a whole layer stores h,
q', k', v, a, x1, h2 and the FFN activation in bf16 on the way: gate 1e-2 normalised L2."""
import numpy as np
import pytest
import torch

from oracle import layer_oracle as lo
from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.harness import gather_kv, pool_views
from paper_2607_00151_b200.workloads import Layer, LayerShape, gen_hidden, gen_layer_weights

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
SENT = 0x7FC1


def _rand(shape, seed, scale=1.0):
    g = torch.Generator(device=DEV)
    g.manual_seed(seed)
    return (torch.randn(shape, generator=g, device=DEV, dtype=torch.float32) * scale).to(torch.bfloat16)


def _check_op(got, ref, what, rel_l2=4e-3):
    g = got.detach().double().cpu().numpy()
    assert np.isfinite(g).all(), what
    rms = np.sqrt(np.mean(ref * ref))
    err = np.abs(g - ref)
    bound = 2.0 ** -8 * np.abs(ref) + 1e-3 * rms
    bad = err > bound
    assert not bad.any(), "%s: %d elements off, worst %.3e at %s (ref %.4f)" % (
        what, int(bad.sum()), err.max(), np.unravel_index(np.argmax(err - bound), err.shape), ref.flat[np.argmax(err - bound)])
    l2 = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    assert l2 <= rel_l2, "%s: normalised L2 %.3e" % (what, l2)
    return l2


# ------------------------------------------------------------------ sa_linear
@pytest.mark.parametrize("M,N,K,res", [
    (1, 256, 64, False),          # one row, one tile, one k-step
    (77, 256, 192, True),         # ragged rows
    (128, 512, 4096, False),      # exactly one m-tile, long K (ring wraps 16 times)
    (300, 520, 192, True),        # several tiles in both directions, N ragged (520 = 2*256 + 8)
    (385, 136, 128, False),       # N < one tile
    (2085, 6144, 4096, True),     # QKV-projection shape of the Llama-8B layer, 17 x 24 tiles: persistent loop > 1 tile per CTA
])
def test_linear(M, N, K, res):
    x = _rand((M, K), 1)
    w = _rand((N, K), 2, K ** -0.5)
    r = _rand((M, N), 3) if res else None
    y = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device=DEV)
    sa.sa_linear(x, w, y, r)
    torch.cuda.synchronize()
    ref = lo.linear(x, w)
    if res:
        ref = ref + lo.widen(r)
    _check_op(y, ref, "linear %dx%dx%d" % (M, N, K))


def test_linear_degenerate_and_errors():
    x = _rand((4, 64), 1)
    w = _rand((8, 64), 2)
    y = torch.zeros((4, 8), dtype=torch.bfloat16, device=DEV)
    sa.sa_linear(x, w, y)                       # N = 8: a single 16-byte column group
    torch.cuda.synchronize()
    _check_op(y, lo.linear(x, w), "linear 4x8x64")
    sa.sa_linear(x[:0], w, y[:0])               # M = 0: no-op
    with pytest.raises(sa.SAError) as e:
        sa.sa_linear(_rand((4, 72), 1), _rand((8, 72), 2), y)   # K not a multiple of 64
    assert e.value.status == sa.SA_ERR_UNSUPPORTED
    # y may alias the residual
    r = _rand((4, 8), 5)
    ref = lo.linear(x, w) + lo.widen(r)
    sa.sa_linear(x, w, r, r)
    torch.cuda.synchronize()
    _check_op(r, ref, "linear in-place residual")


def test_linear_untouched_outside():
    """Rows >= M and the bytes after the last row are not written (the tile is 128 x 256, the matrix is not)."""
    M, N, K = 130, 264, 64
    x = _rand((M, K), 1)
    w = _rand((N, K), 2)
    buf = torch.zeros((M + 126) * N + 64, dtype=torch.int16, device=DEV) + 0x7FC1
    y = buf[: M * N].view(torch.bfloat16).view(M, N)
    sa.sa_linear(x, w, y)
    torch.cuda.synchronize()
    assert (buf[M * N:] == 0x7FC1).all()
    _check_op(y, lo.linear(x, w), "linear 130x264x64")


# ------------------------------------------------------------------ split-K (small M: decode batches)
@pytest.mark.parametrize("M,N,K,res", [
    (1, 4096, 4096, True),        # one decode row through the output projection: 16 tiles x 9 k slices
    (64, 4096, 14336, True),      # the down projection of a 64-row decode batch: 224 k-steps cut 9 ways
    (200, 6144, 4096, False),     # two m-tiles x 24 n-tiles = 48 tiles x 3 slices
    (130, 520, 448, True),        # ragged N, 7 k-steps in 3 uneven slices (2 + 2 + 3)
])
def test_linear_split_k(M, N, K, res):
    nb = sa.sa_linear_workspace_bytes(M, N, K)
    assert nb > 0, "this shape is expected to split"
    x = _rand((M, K), 11)
    w = _rand((N, K), 12, K ** -0.5)
    r = _rand((M, N), 13) if res else None
    ws = torch.full((nb,), 0xFF, dtype=torch.uint8, device=DEV)   # NaN bit patterns: a partial read before it is written shows
    ref = lo.linear(x, w)
    if res:
        ref = ref + lo.widen(r)
    ys = []
    for _ in range(2):
        y = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device=DEV)
        sa.sa_linear_ws(x, w, y, ws, r)
        torch.cuda.synchronize()
        _check_op(y, ref, "split-K linear %dx%dx%d" % (M, N, K))
        ys.append(y)
    assert torch.equal(ys[0].view(torch.int16), ys[1].view(torch.int16)), "slices are summed in a fixed order"
    # without scratch the same call runs unsplit and still meets the oracle
    y0 = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device=DEV)
    sa.sa_linear_ws(x, w, y0, None, r)
    torch.cuda.synchronize()
    _check_op(y0, ref, "unsplit fallback")
    # large M never asks for scratch
    assert sa.sa_linear_workspace_bytes(4096, N, K) == 0


def test_swiglu_split_k():
    M, F, K = 16, 4096, 4096      # 32 tiles x 4 slices
    nb = sa.sa_swiglu_workspace_bytes(M, F, K)
    assert nb > 0
    x = _rand((M, K), 14)
    wg = _rand((F, K), 15, 2.0 * K ** -0.5)
    wu = _rand((F, K), 16, K ** -0.5)
    ws = torch.full((nb,), 0xFF, dtype=torch.uint8, device=DEV)
    act = torch.full((M, F), float("nan"), dtype=torch.bfloat16, device=DEV)
    sa.sa_swiglu_ws(x, wg, wu, act, ws)
    torch.cuda.synchronize()
    _check_op(act, lo.swiglu_act(x, wg, wu), "split-K swiglu")


# ------------------------------------------------------------------ sa_swiglu / sa_rmsnorm
@pytest.mark.parametrize("M,F,K", [(5, 128, 64), (200, 328, 256), (1030, 14336, 4096)])
def test_swiglu(M, F, K):
    x = _rand((M, K), 4)
    wg = _rand((F, K), 5, 2.0 * K ** -0.5)     # gate pre-activations ~ N(0, 4): both tails of SiLU
    wu = _rand((F, K), 6, K ** -0.5)
    act = torch.full((M, F), float("nan"), dtype=torch.bfloat16, device=DEV)
    sa.sa_swiglu(x, wg, wu, act)
    torch.cuda.synchronize()
    _check_op(act, lo.swiglu_act(x, wg, wu), "swiglu %dx%dx%d" % (M, F, K))


@pytest.mark.parametrize("M,H", [(1, 64), (9, 4096), (1000, 4096), (33, 520)])
def test_rmsnorm(M, H):
    x = _rand((M, H), 7, 3.0)
    w = (1.0 + 0.1 * _rand((H,), 8).float()).to(torch.bfloat16)
    y = torch.empty_like(x)
    sa.sa_rmsnorm(x, w, 1e-5, y)
    torch.cuda.synchronize()
    _check_op(y, lo.rmsnorm(x, w, 1e-5), "rmsnorm %dx%d" % (M, H))


# ------------------------------------------------------------------ fused QKV projection + RoPE + append
def _pool(layer: Layer, num_pages, max_sessions=8, max_tokens=4096, order_seed=5, sentinel=SENT):
    cfg = sa.PoolConfig(layer.num_q_heads, layer.num_kv_heads, layer.head_dim, layer.page_size, num_pages, max_sessions,
                        max_tokens, layer.rope_base, 0)
    nbytes = sa.sa_kv_pool_storage_bytes(cfg)
    storage = torch.empty(nbytes, dtype=torch.uint8, device=DEV)
    storage.view(torch.int16)[: nbytes // 2].fill_(np.array(sentinel, dtype=np.uint16).view(np.int16).item())
    order = np.random.default_rng(order_seed).permutation(num_pages).astype(np.int32)
    return sa.sa_kv_pool_create(cfg, storage, order)


def test_qkv_rope_append_matches_oracle_and_placement():
    layer = Layer(8, 2, 128, 64, 500000.0)      # N = 12 heads * 128 = 1536 = 6 tiles
    H = 256
    W = gen_layer_weights(layer, LayerShape(H, 512), 21, DEV)
    pool = _pool(layer, 64)
    prefixes, news = [100, 0, 777], [300, 1, 131]          # mid-page starts, a decode row, ragged lengths
    sids = [sa.sa_kv_session_open(pool) for _ in prefixes]
    # retained prefixes through the unfused append (raw k, v)
    kv_prefix = []
    for i, P in enumerate(prefixes):
        k = _rand((P, layer.num_kv_heads, 128), 100 + i)
        v = _rand((P, layer.num_kv_heads, 128), 200 + i)
        kv_prefix.append((k, v))
        if P:
            sa.sa_rope_kv_append(pool, [sids[i]], [0, P], k, v, None)
    torch.cuda.synchronize()
    kp, vp = pool_views(pool)
    before_k, before_v = kp.clone(), vp.clone()

    T = sum(news)
    h = gen_hidden(T, H, 22, DEV)
    indptr = np.concatenate([[0], np.cumsum(news)]).astype(np.int32)
    q_out = torch.full((T, layer.num_q_heads, 128), float("nan"), dtype=torch.bfloat16, device=DEV)
    ws = torch.empty(sa.sa_qkv_rope_append_workspace_bytes(pool, T), dtype=torch.uint8, device=DEV)
    sa.sa_qkv_rope_append(pool, sids, indptr, h, W["w_qkv"], q_out, ws)
    torch.cuda.synchronize()

    touched = torch.zeros(kp.shape[:3], dtype=torch.bool, device=DEV)      # [page, head, slot]
    for i, (P, n) in enumerate(zip(prefixes, news)):
        a, b = int(indptr[i]), int(indptr[i + 1])
        pos = np.arange(P, P + n)
        q_ref, k_ref, v_ref = lo.qkv_rope(h[a:b], W["w_qkv"], layer.num_q_heads, layer.num_kv_heads, 128, pos, layer.rope_base)
        ln, pages = sa.sa_kv_session_query(pool, sids[i])
        assert ln == P + n
        k_gpu, v_gpu = gather_kv(pool, pages, ln)
        _check_op(q_out[a:b], q_ref, "Q' of request %d" % i)
        _check_op(k_gpu[P:], k_ref, "K' of request %d" % i)
        _check_op(v_gpu[P:], v_ref, "V of request %d" % i)
        # the retained prefix keeps its bits (prefix KV independent of what follows)
        if P:
            k0, v0 = gather_kv(pool, pages, P)
            kr = orc.rope(kv_prefix[i][0].cpu(), np.arange(P), layer.rope_base)
            assert np.abs(k0.double().cpu().numpy() - kr).max() <= 2e-2
            assert torch.equal(v0.view(torch.int16), kv_prefix[i][1].view(torch.int16))
        for p_ in pos:
            touched[pages[p_ // 64], :, p_ % 64] = True
    # every slot the fused call did not address keeps its bits
    same_k = (kp.view(torch.int16) == before_k.view(torch.int16)).all(dim=-1)
    same_v = (vp.view(torch.int16) == before_v.view(torch.int16)).all(dim=-1)
    assert same_k[~touched].all() and same_v[~touched].all()


def test_qkv_fused_equals_unfused_within_one_rounding():
    """sa_linear -> sa_rope_kv_append (two roundings of q, k) against the fused call (one): within bf16 rounding,
    V bit-equal (no arithmetic after the projection)."""
    layer = Layer(8, 2, 128, 64, 500000.0)
    H, T, P = 192, 260, 37
    W = gen_layer_weights(layer, LayerShape(H, 256), 31, DEV)
    h = gen_hidden(T, H, 32, DEV)
    outs = []
    for fused in (True, False):
        pool = _pool(layer, 32)
        sid = sa.sa_kv_session_open(pool)
        k0, v0 = _rand((P, 2, 128), 1), _rand((P, 2, 128), 2)
        sa.sa_rope_kv_append(pool, [sid], [0, P], k0, v0, None)
        if fused:
            q = torch.empty((T, 8, 128), dtype=torch.bfloat16, device=DEV)
            ws = torch.empty(sa.sa_qkv_rope_append_workspace_bytes(pool, T), dtype=torch.uint8, device=DEV)
            sa.sa_qkv_rope_append(pool, [sid], [0, T], h, W["w_qkv"], q, ws)
        else:
            qkv = torch.empty((T, 12 * 128), dtype=torch.bfloat16, device=DEV)
            sa.sa_linear(h, W["w_qkv"], qkv)
            q = qkv[:, : 8 * 128].reshape(T, 8, 128).contiguous()
            k = qkv[:, 8 * 128: 10 * 128].reshape(T, 2, 128).contiguous()
            v = qkv[:, 10 * 128:].reshape(T, 2, 128).contiguous()
            sa.sa_rope_kv_append(pool, [sid], [0, T], k, v, q)
        torch.cuda.synchronize()
        ln, pages = sa.sa_kv_session_query(pool, sid)
        kk, vv = gather_kv(pool, pages, ln)
        outs.append((q.float().cpu(), kk.float().cpu(), vv.clone().cpu()))
    (qf, kf, vf), (qu, ku, vu) = outs
    assert torch.equal(vf.view(torch.int16), vu.view(torch.int16))
    for a, b, name in ((qf, qu, "q"), (kf, ku, "k")):
        # the unfused route rounds the pair (x_m, x_{m+64}) to bf16 before rotating it: the difference is bounded
        # by bf16 half-ulps of the pair's norm (which the rotation preserves), not of the element itself
        pair = torch.cat([a[..., 64:], a[..., :64]], dim=-1)
        assert ((a - b).abs() <= 2.0 ** -7 * (a.abs() + pair.abs()) + 1e-6).all(), name
        assert (a - b).abs().max() > 0, name + ": the two routes should differ in rounding somewhere"


def test_qkv_rope_append_out_of_pages_changes_nothing():
    layer = Layer(8, 2, 128, 64, 500000.0)
    pool = _pool(layer, 4)
    sid = sa.sa_kv_session_open(pool)
    W = gen_layer_weights(layer, LayerShape(64, 64), 41, DEV)
    T = 5 * 64
    h = gen_hidden(T, 64, 42, DEV)
    q = torch.empty((T, 8, 128), dtype=torch.bfloat16, device=DEV)
    ws = torch.empty(sa.sa_qkv_rope_append_workspace_bytes(pool, T), dtype=torch.uint8, device=DEV)
    with pytest.raises(sa.SAError) as e:
        sa.sa_qkv_rope_append(pool, [sid], [0, T], h, W["w_qkv"], q, ws)
    assert e.value.status == sa.SA_ERR_OUT_OF_PAGES
    assert sa.sa_kv_session_query(pool, sid) == (0, []) and sa.sa_kv_pool_free_pages(pool) == 4


# ------------------------------------------------------------------ one whole layer
def _layer_case(layer, shape, prefixes, news, seed):
    W = gen_layer_weights(layer, shape, seed, DEV)
    used = sum((p + n + 63) // 64 for p, n in zip(prefixes, news))
    pool = _pool(layer, used * 2 + 4, max_sessions=len(prefixes) + 2, max_tokens=max(p + n for p, n in zip(prefixes, news)) + 64)
    sids = [sa.sa_kv_session_open(pool) for _ in prefixes]
    lw = sa.LayerWeights(W["norm1"], W["w_qkv"], W["w_o"], W["norm2"], W["w_gate"], W["w_up"], W["w_down"], shape.rms_eps)
    # the retained prefixes are built by the layer itself (one earlier forward over the prefix tokens)
    xs = [gen_hidden(p + n, shape.hidden, seed * 100 + i, DEV) for i, (p, n) in enumerate(zip(prefixes, news))]
    live = [i for i, p in enumerate(prefixes) if p > 0]
    if live:
        xp = torch.cat([xs[i][: prefixes[i]] for i in live]).contiguous()
        ip = np.concatenate([[0], np.cumsum([prefixes[i] for i in live])]).astype(np.int32)
        ws = torch.empty(sa.sa_layer_workspace_bytes(pool, lw, [sids[i] for i in live], ip), dtype=torch.uint8, device=DEV)
        sa.sa_layer_forward(pool, lw, [sids[i] for i in live], ip, xp, torch.empty_like(xp), ws)
    x = torch.cat([xs[i][prefixes[i]:] for i in range(len(prefixes))]).contiguous()
    indptr = np.concatenate([[0], np.cumsum(news)]).astype(np.int32)
    ws = torch.empty(sa.sa_layer_workspace_bytes(pool, lw, sids, indptr), dtype=torch.uint8, device=DEV)
    y = torch.full_like(x, float("nan"))
    sa.sa_layer_forward(pool, lw, sids, indptr, x, y, ws)
    torch.cuda.synchronize()
    return W, xs, y, indptr, pool, sids


def test_layer_forward_mixed_batch_vs_oracle():
    layer = Layer(4, 2, 128, 64, 500000.0)
    shape = LayerShape(256, 512)
    prefixes, news = [150, 400, 0], [200, 1, 70]          # prefill chunk on a prefix, decode row, prefill from scratch
    W, xs, y, indptr, pool, sids = _layer_case(layer, shape, prefixes, news, 51)
    empty = np.zeros((0, layer.num_kv_heads, 128))
    for i, (P, n) in enumerate(zip(prefixes, news)):
        full = lo.layer_forward(xs[i], W, layer.num_q_heads, layer.num_kv_heads, 128, shape.rms_eps, layer.rope_base, empty, empty, 0)
        ref = full["y"][P:]
        got = y[int(indptr[i]): int(indptr[i + 1])].double().cpu().numpy()
        assert np.isfinite(got).all()
        l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        assert l2 <= 1e-2, (i, l2)
        assert np.abs(got - ref).max() <= 2.0 ** -6 * np.abs(ref).max() + 1e-2, (i, np.abs(got - ref).max())
        # the cache the layer built: K' of the whole session against the oracle's
        ln, pages = sa.sa_kv_session_query(pool, sids[i])
        k_gpu, v_gpu = gather_kv(pool, pages, ln)
        # (two roundings on the way: h = RMSNorm(x) is stored in bf16 before the projection)
        for g_, r_ in ((k_gpu, full["k_rot"]), (v_gpu, full["v"])):
            g_ = g_.double().cpu().numpy()
            assert np.linalg.norm(g_ - r_) / np.linalg.norm(r_) <= 6e-3
            assert np.abs(g_ - r_).max() <= 2.0 ** -6 * np.abs(r_).max()


def test_layer_forward_llama8b_shape_sampled():
    """BASELINE.json's Llama-3-8B-shaped layer at full width (H 4096, F 14336, 32/8 heads): a 300-token chunk over
    a 500-token prefix.  The oracle runs the whole (small) context in fp64."""
    layer = Layer(32, 8, 128, 64, 500000.0)
    shape = LayerShape(4096, 14336)
    W, xs, y, indptr, pool, sids = _layer_case(layer, shape, [500], [300], 61)
    empty = np.zeros((0, 8, 128))
    full = lo.layer_forward(xs[0], W, 32, 8, 128, shape.rms_eps, layer.rope_base, empty, empty, 0)
    got = y.double().cpu().numpy()
    ref = full["y"][500:]
    l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert np.isfinite(got).all() and l2 <= 1e-2, l2


def test_gemm_table_shape():
    ms = sa.sa_gemm_table(1024, 2048, 8, 2, 128, [1, 64, 512, 2048], warmup=1, iters=3)
    assert ms.shape == (4,) and (ms > 0).all()
    assert ms[3] > ms[0]                      # compute-bound end costs more than the memory-bound end (L303)
