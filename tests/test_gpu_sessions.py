"""GPU tests of the session operations behind the commit splice (PAPER.md L47
"directly replaces the prefix in the working context", L170, L186-187): a lookahead session forked
from the main one shares the retained prefix's pages, rebuilds the transformed segment behind it,
and is committed by a block-table swap.  Everything is compared bit for bit with a session built
from scratch, and the re-prefill itself with the fp64 oracle."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.harness import gather_kv, pool_views
from paper_2607_00151_b200.workloads import Layer

from gpu_util import check_out

pytestmark = pytest.mark.gpu

SENT = 0x7FC1


def _bits(t):
    return t.contiguous().view(torch.int16)


def _mk_pool(L: Layer, num_pages, max_tokens, order, sentinel=SENT):
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, num_pages, 8, max_tokens, L.rope_base, 0)
    nbytes = sa.sa_kv_pool_storage_bytes(cfg)
    storage = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    storage.view(torch.int16)[: nbytes // 2].fill_(np.array(sentinel, dtype=np.uint16).view(np.int16).item())
    return sa.sa_kv_pool_create(cfg, storage, order)


def _rand(n, h, d, gen, scale):
    return (torch.randn((n, h, d), generator=gen, device="cuda", dtype=torch.float32) * scale).to(torch.bfloat16)


def _attend(pool, sid, q_rot):
    n = q_rot.shape[0]
    out = torch.empty_like(q_rot)
    lse = torch.empty((n, q_rot.shape[1]), dtype=torch.float32, device="cuda")
    nb = sa.sa_mixed_attention_workspace_bytes(pool, [sid], [0, n])
    ws = torch.empty(max(nb, 256), dtype=torch.uint8, device="cuda")
    sa.sa_mixed_attention(pool, [sid], [0, n], q_rot, out, lse, 0.0, ws)
    torch.cuda.synchronize()
    return out, lse


@pytest.mark.parametrize("shape", ["llama", "tiny"])
def test_fork_reprefill_commit_bit_equal_to_a_fresh_session(shape):
    if shape == "llama":   # tcgen05 path, page 64; prefix ends inside a page
        L, P, TAIL, SEG, scale = Layer(32, 8, 128, 64, 500000.0), 700, 300, 333, 128 ** -0.5
    else:                  # head_dim 64 path, page 16
        L, P, TAIL, SEG, scale = Layer(8, 2, 64, 16, 10000.0), 41, 30, 50, 1.0
    B = L.page_size
    n_pages = 2 * ((P + TAIL + SEG) // B + 4) + 8
    order = np.random.default_rng(99).permutation(n_pages).astype(np.int32)
    pool = _mk_pool(L, n_pages, 4096, order)
    g = torch.Generator(device="cuda")
    g.manual_seed(1234)
    k_main, v_main = _rand(P + TAIL, L.num_kv_heads, L.head_dim, g, scale), _rand(P + TAIL, L.num_kv_heads, L.head_dim, g, 1.0)
    k_seg, v_seg = _rand(SEG, L.num_kv_heads, L.head_dim, g, scale), _rand(SEG, L.num_kv_heads, L.head_dim, g, 1.0)
    q_seg = _rand(SEG, L.num_q_heads, L.head_dim, g, scale)
    k_dec, v_dec = _rand(1, L.num_kv_heads, L.head_dim, g, scale), _rand(1, L.num_kv_heads, L.head_dim, g, 1.0)
    q_dec = _rand(1, L.num_q_heads, L.head_dim, g, scale)

    # ---- main session: the untransformed context (retained prefix + a tail that the transformation drops)
    main = sa.sa_kv_session_open(pool)
    sa.sa_rope_kv_append(pool, [main], [0, P + TAIL], k_main, v_main, None)
    torch.cuda.synchronize()
    len_main, pg_main = sa.sa_kv_session_query(pool, main)
    km0, vm0 = gather_kv(pool, pg_main, len_main)
    free0 = sa.sa_kv_pool_free_pages(pool)

    # ---- lookahead: fork at the retained prefix, rebuild the transformed segment behind it
    la = sa.sa_kv_session_fork(pool, main, P)
    len_la, pg_la = sa.sa_kv_session_query(pool, la)
    assert len_la == P and pg_la[: P // B] == pg_main[: P // B]
    assert (P % B == 0) or (pg_la[-1] not in pg_main and sa.sa_kv_pool_free_pages(pool) == free0 - 1)
    torch.cuda.synchronize()
    kf, vf = gather_kv(pool, pg_la, P)
    assert torch.equal(_bits(kf), _bits(km0[:P])) and torch.equal(_bits(vf), _bits(vm0[:P]))   # the prefix, bit for bit
    q_la = q_seg.clone()
    sa.sa_rope_kv_append(pool, [la], [0, SEG], k_seg, v_seg, q_la)
    out_la, lse_la = _attend(pool, la, q_la)
    # the main session did not notice: same pages, same bits (prefix independence, L45)
    assert sa.sa_kv_session_query(pool, main) == (len_main, pg_main)
    km1, vm1 = gather_kv(pool, pg_main, len_main)
    assert torch.equal(_bits(km1), _bits(km0)) and torch.equal(_bits(vm1), _bits(vm0))

    # ---- the same transformed context built from scratch in a second pool (another page map)
    order2 = np.random.default_rng(7).permutation(n_pages).astype(np.int32)
    pool2 = _mk_pool(L, n_pages, 4096, order2)
    ref = sa.sa_kv_session_open(pool2)
    sa.sa_rope_kv_append(pool2, [ref], [0, P], k_main[:P].contiguous(), v_main[:P].contiguous(), None)
    q_ref = q_seg.clone()
    sa.sa_rope_kv_append(pool2, [ref], [0, SEG], k_seg, v_seg, q_ref)
    out_ref, lse_ref = _attend(pool2, ref, q_ref)
    assert torch.equal(_bits(q_la), _bits(q_ref))
    assert torch.equal(_bits(out_la), _bits(out_ref)) and torch.equal(lse_la, lse_ref)

    # ---- and against the fp64 oracle (segment decomposability, L105-109)
    kr = orc.rope(k_main[:P].cpu(), np.arange(P), L.rope_base)
    o = orc.oracle_cached(kr, orc.widen(v_main[:P].cpu()), q_seg.cpu(), k_seg.cpu(), v_seg.cpu(), P, L.rope_base)
    check_out(out_la, o["o"], "forked re-prefill (%s)" % shape)

    # ---- commit: the main session now IS the transformed context; a decode step on it matches the fresh one
    sa.sa_kv_session_commit(pool, main, la)
    assert sa.sa_kv_session_query(pool, main) == (P + SEG, sa.sa_kv_session_query(pool, main)[1])
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_query(pool, la)
    used = (P + SEG + B - 1) // B
    assert sa.sa_kv_pool_free_pages(pool) == n_pages - used          # the superseded tail pages are free again
    qd1, qd2 = q_dec.clone(), q_dec.clone()
    sa.sa_rope_kv_append(pool, [main], [0, 1], k_dec, v_dec, qd1)
    sa.sa_rope_kv_append(pool2, [ref], [0, 1], k_dec, v_dec, qd2)
    o1, l1 = _attend(pool, main, qd1)
    o2, l2 = _attend(pool2, ref, qd2)
    assert torch.equal(_bits(o1), _bits(o2)) and torch.equal(l1, l2)
    # every page no session holds still carries the sentinel or stale data, never a fresh write: the pages of
    # pool 2 that were never handed out are untouched
    kp2, _ = pool_views(pool2)
    held = torch.zeros(n_pages, dtype=torch.bool)
    held[torch.as_tensor(sa.sa_kv_session_query(pool2, ref)[1])] = True
    sent = np.array(SENT, dtype=np.uint16).view(np.int16).item()
    assert (_bits(kp2[~held]) == sent).all()
    sa.sa_kv_session_close(pool, main)
    assert sa.sa_kv_pool_free_pages(pool) == n_pages


def test_copy_on_write_keeps_the_other_holder_intact():
    """Truncate into a shared page and append again: the appender moves to a private copy (device
    copy of the page), the fork keeps reading the old bits."""
    L = Layer(8, 2, 64, 16, 10000.0)
    pool = _mk_pool(L, 32, 1024, None)
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    k, v = _rand(64, 2, 64, g, 1.0), _rand(64, 2, 64, g, 1.0)
    k2, v2 = _rand(8, 2, 64, g, 1.0), _rand(8, 2, 64, g, 1.0)
    a = sa.sa_kv_session_open(pool)
    sa.sa_rope_kv_append(pool, [a], [0, 64], k, v, None)
    f = sa.sa_kv_session_fork(pool, a, 64)
    torch.cuda.synchronize()
    _, pg = sa.sa_kv_session_query(pool, a)
    ka, va = gather_kv(pool, pg, 64)
    sa.sa_kv_session_truncate(pool, a, 40)
    sa.sa_rope_kv_append(pool, [a], [0, 8], k2, v2, None)
    torch.cuda.synchronize()
    la, pga = sa.sa_kv_session_query(pool, a)
    assert la == 48 and pga[:2] == pg[:2] and pga[2] != pg[2]
    kf, vf = gather_kv(pool, sa.sa_kv_session_query(pool, f)[1], 64)
    assert torch.equal(_bits(kf), _bits(ka)) and torch.equal(_bits(vf), _bits(va))        # the fork is intact
    kn, vn = gather_kv(pool, pga, 48)
    assert torch.equal(_bits(kn[:40]), _bits(ka[:40])) and torch.equal(_bits(vn[:40]), _bits(va[:40]))   # copied prefix of the page
    assert torch.equal(_bits(vn[40:]), _bits(v2))                                           # new tokens, V is a bit copy
    k2_ref = orc.rope(k2.cpu(), np.arange(40, 48), L.rope_base)
    assert np.abs(kn[40:].double().cpu().numpy() - k2_ref).max() <= 4e-2                      # rotated at positions 40..47
