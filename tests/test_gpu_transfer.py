"""GPU tests of the KV hand-over between pools ("KV transfer" between
prefill and decode instances, L424 tensor parallelism): a session leaves one pool as a wire image
[2][Hkv][n][D] and enters another pool -- with another page size, another page order, or only a
slice of the kv heads -- from it.  The image is compared with the oracle's re-indexing of the
logical cache (V bit for bit, K' within the RoPE gate), and everything downstream bit for bit
with the session it came from."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.harness import gather_kv, pool_views
from paper_2607_00151_b200.workloads import Layer

pytestmark = pytest.mark.gpu

SENT = 0x7FC1


def _bits(t):
    return t.contiguous().view(torch.int16)


def _mk_pool(L: Layer, num_pages, max_tokens, seed, sentinel=SENT):
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, num_pages, 8, max_tokens, L.rope_base, 0)
    nbytes = sa.sa_kv_pool_storage_bytes(cfg)
    storage = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    storage.view(torch.int16)[: nbytes // 2].fill_(np.array(sentinel, dtype=np.uint16).view(np.int16).item())
    order = np.random.default_rng(seed).permutation(num_pages).astype(np.int32)
    return sa.sa_kv_pool_create(cfg, storage, order)


def _rand(n, h, d, gen, scale):
    return (torch.randn((n, h, d), generator=gen, device="cuda", dtype=torch.float32) * scale).to(torch.bfloat16)


def _attend(pool, sid, q_rot):
    n = q_rot.shape[0]
    out = torch.empty_like(q_rot)
    lse = torch.empty((n, q_rot.shape[1]), dtype=torch.float32, device="cuda")
    ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(pool, [sid], [0, n]), 256), dtype=torch.uint8, device="cuda")
    sa.sa_mixed_attention(pool, [sid], [0, n], q_rot, out, lse, 0.0, ws)
    torch.cuda.synchronize()
    return out, lse


def _source(L: Layer, n, seed, scale):
    """A pool with one session of n cached tokens; returns (pool, sid, k_raw, v_raw)."""
    gen = torch.Generator(device="cuda")
    gen.manual_seed(seed)
    pages = (n + L.page_size - 1) // L.page_size + 3
    pool = _mk_pool(L, pages, n + 2 * L.page_size, seed + 1)
    sid = sa.sa_kv_session_open(pool)
    k, v = _rand(n, L.num_kv_heads, L.head_dim, gen, scale), _rand(n, L.num_kv_heads, L.head_dim, gen, scale)
    sa.sa_rope_kv_append(pool, [sid], [0, n], k, v, None)
    torch.cuda.synchronize()
    return pool, sid, k, v


def _export(pool, sid, t0, n):
    L = pool.cfg
    img = torch.full((2, L.num_kv_heads, n, L.head_dim), float("nan"), dtype=torch.bfloat16, device="cuda")
    assert sa.sa_kv_wire_bytes(pool, n) == img.numel() * 2
    sa.sa_kv_session_export(pool, sid, t0, n, img)
    torch.cuda.synchronize()
    return img


@pytest.mark.parametrize("shape", ["llama", "tiny"])
def test_export_image_matches_the_oracle_reindexing(shape):
    L, n, scale = (Layer(32, 8, 128, 64, 500000.0), 333, 128 ** -0.5) if shape == "llama" else (Layer(8, 2, 64, 16, 10000.0), 77, 1.0)
    pool, sid, k, v = _source(L, n, 11, scale)
    t0, m = 5, n - 9  # a range that starts and ends inside pages
    img = _export(pool, sid, t0, m)
    k_rot = orc.rope(k.cpu(), np.arange(n), L.rope_base)       # fp64 K' of the logical cache
    ref = orc.wire_image(k_rot[t0:t0 + m], orc.widen(v.cpu())[t0:t0 + m])
    got = img.double().cpu().numpy()
    assert np.array_equal(got[1], ref[1]), "V part of the image must be a bit copy"
    # RoPE gate of BASELINE.json (1e-2) where a correctly rounded bf16 can meet it, one bf16 ulp elsewhere (DESIGN.md T-B)
    assert (np.abs(got[0] - ref[0]) <= np.maximum(1e-2, 2.0 ** -7 * np.abs(ref[0]))).all()
    # and the K' part is exactly what the pool stores (the hand-over rounds nothing again)
    length, page_ids = sa.sa_kv_session_query(pool, sid)
    ks, vs = gather_kv(pool, list(page_ids), length)
    assert torch.equal(_bits(img[0]), _bits(ks[t0:t0 + m].permute(1, 0, 2)))
    assert torch.equal(_bits(img[1]), _bits(vs[t0:t0 + m].permute(1, 0, 2)))
    sa.sa_kv_pool_destroy(pool)


def test_roundtrip_into_other_page_size_and_order_is_bit_exact():
    L = Layer(32, 8, 128, 64, 500000.0)
    n = 700
    pool, sid, k, v = _source(L, n, 21, 128 ** -0.5)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(5)
    q = _rand(200, L.num_q_heads, L.head_dim, gen, 128 ** -0.5)
    # the last 200 cached tokens double as the queries' own positions: a re-prefill chunk over the handed-over cache
    o_src, lse_src = _attend(pool, sid, q)
    for B2, seed in ((64, 3), (16, 4)):
        L2 = Layer(L.num_q_heads, L.num_kv_heads, L.head_dim, B2, L.rope_base)
        dst = _mk_pool(L2, (n + B2 - 1) // B2 + 5, n + 128, seed)
        sid2 = sa.sa_kv_session_open(dst)
        free0 = sa.sa_kv_pool_free_pages(dst)
        # in order, in three uneven pieces that do not end on page boundaries
        for t0, m in ((0, 100), (100, 233), (333, n - 333)):
            sa.sa_kv_session_import(dst, sid2, m, _export(pool, sid, t0, m), L.num_kv_heads, 0)
        torch.cuda.synchronize()
        length, page_ids = sa.sa_kv_session_query(dst, sid2)
        assert length == n and sa.sa_kv_pool_free_pages(dst) == free0 - (n + B2 - 1) // B2
        k2, v2 = gather_kv(dst, list(page_ids), n)
        ls, ps = sa.sa_kv_session_query(pool, sid)
        k1, v1 = gather_kv(pool, list(ps), n)
        assert torch.equal(_bits(k1), _bits(k2)) and torch.equal(_bits(v1), _bits(v2))
        # slots the session does not own keep the sentinel (last page's tail and every unused page)
        kp, vp = pool_views(dst)
        used = set(int(p) for p in page_ids)
        for pg in range(dst.cfg.num_pages):
            lo = 0 if pg not in used else (n % B2 if pg == int(page_ids[-1]) and n % B2 else B2)
            if lo < B2:
                assert (_bits(kp[pg, :, lo:, :]) == np.array(SENT, dtype=np.uint16).view(np.int16).item()).all()
                assert (_bits(vp[pg, :, lo:, :]) == np.array(SENT, dtype=np.uint16).view(np.int16).item()).all()
        o2, lse2 = _attend(dst, sid2, q)
        if B2 == L.page_size:
            assert torch.equal(_bits(o_src), _bits(o2)) and torch.equal(lse_src, lse2)
        else:  # another page size: same logical tiles, the bits still agree (tiles are 128 logical keys)
            assert torch.equal(_bits(o_src), _bits(o2))
        sa.sa_kv_pool_destroy(dst)
    sa.sa_kv_pool_destroy(pool)


def test_head_sharded_receivers_reproduce_the_unsharded_attention():
    """Tensor-parallel receivers: rank r of 2 holds kv heads [4r, 4r+4) and q heads [16r, 16r+16)."""
    L = Layer(32, 8, 128, 64, 500000.0)
    n = 515
    pool, sid, k, v = _source(L, n, 31, 128 ** -0.5)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(6)
    q = _rand(130, L.num_q_heads, L.head_dim, gen, 128 ** -0.5)
    o_full, lse_full = _attend(pool, sid, q)
    img = _export(pool, sid, 0, n)
    world = 2
    Ls = Layer(L.num_q_heads // world, L.num_kv_heads // world, L.head_dim, L.page_size, L.rope_base)
    outs, lses = [], []
    for r in range(world):
        shard = _mk_pool(Ls, n // 64 + 4, n + 64, 40 + r)
        s2 = sa.sa_kv_session_open(shard)
        sa.sa_kv_session_import(shard, s2, n, img, L.num_kv_heads, r * Ls.num_kv_heads)
        qs = q[:, r * Ls.num_q_heads:(r + 1) * Ls.num_q_heads].contiguous()
        o, l = _attend(shard, s2, qs)
        outs.append(o)
        lses.append(l)
        # the oracle's head slice of the image is what this rank stored
        length, page_ids = sa.sa_kv_session_query(shard, s2)
        ks, vs = gather_kv(shard, list(page_ids), n)
        ref_v = orc.wire_image(orc.widen(k.cpu()), orc.widen(v.cpu()), r * Ls.num_kv_heads, Ls.num_kv_heads)[1]
        assert np.array_equal(vs.permute(1, 0, 2).double().cpu().numpy(), ref_v)
        sa.sa_kv_pool_destroy(shard)
    assert torch.equal(_bits(torch.cat(outs, dim=1)), _bits(o_full))
    assert torch.equal(torch.cat(lses, dim=1), lse_full)
    sa.sa_kv_pool_destroy(pool)


def test_errors_change_nothing():
    L = Layer(8, 2, 64, 16, 10000.0)
    pool, sid, k, v = _source(L, 40, 51, 1.0)
    img = torch.zeros((2, 2, 40, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_export(pool, sid, 10, 31, img)               # range leaves the session
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_export(pool, sid, 0, 40, img.view(-1)[: 2 * 2 * 39 * 64])  # image too small
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_export(pool, sid, 0, 8, img.view(-1)[4:])    # not 16-byte aligned
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_import(pool, sid, 8, img, 2, 1)              # head slice leaves the image
    free0 = sa.sa_kv_pool_free_pages(pool)
    big = torch.zeros((2, 2, 16 * (free0 + 2), 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(sa.SAError) as ei:
        sa.sa_kv_session_import(pool, sid, big.shape[2], big, 2, 0)
    assert ei.value.status in (sa.SA_ERR_OUT_OF_PAGES, sa.SA_ERR_INVALID_ARG)
    assert sa.sa_kv_pool_free_pages(pool) == free0 and sa.sa_kv_session_query(pool, sid)[0] == 40
    sa.sa_kv_session_export(pool, sid, 0, 0, img)                     # empty range: legal, no launch
    sa.sa_kv_session_import(pool, sid, 0, img, 2, 0)
    assert sa.sa_kv_session_query(pool, sid)[0] == 40
    sa.sa_kv_pool_destroy(pool)


@pytest.mark.parametrize("n_sessions", [5, 70])
def test_many_sessions_in_one_call_equal_one_call_per_session(n_sessions):
    """sa_kv_sessions_export / sa_kv_sessions_import (one launch for every session of a batch; 5 sessions ride in the kernel
    parameters, 70 go through the metadata slab) against the per-session calls: images and imported pages bit for bit,
    ragged lengths incl. an empty range, two ranges of one session, sentinel slots untouched, all-or-nothing page demand."""
    L = Layer(32, 8, 128, 64, 500000.0)
    rng = np.random.default_rng(100 + n_sessions)
    lens = [int(x) for x in rng.integers(1, 400, size=n_sessions)]
    lens[1] = 64      # ends on a page boundary
    gen = torch.Generator(device="cuda")
    gen.manual_seed(7)
    pages = sum((n + 63) // 64 for n in lens) + 8
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, pages, n_sessions + 2, 1024, L.rope_base, 0)

    def mk(seed):
        nbytes = sa.sa_kv_pool_storage_bytes(cfg)
        storage = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        storage.view(torch.int16)[: nbytes // 2].fill_(np.array(SENT, dtype=np.uint16).view(np.int16).item())
        return sa.sa_kv_pool_create(cfg, storage, np.random.default_rng(seed).permutation(pages).astype(np.int32))
    src = mk(1)
    sids = [sa.sa_kv_session_open(src) for _ in lens]
    for sid, n in zip(sids, lens):
        sa.sa_rope_kv_append(src, [sid], [0, n], _rand(n, 8, 128, gen, 0.1), _rand(n, 8, 128, gen, 0.1), None)
    # ranges: every session whole, except session 0 in two pieces and session 2 as an empty range plus the whole
    ranges = [(sids[0], 0, lens[0] // 2), (sids[0], lens[0] // 2, lens[0] - lens[0] // 2), (sids[2], 3 if lens[2] > 3 else 0, 0)]
    ranges += [(sid, 0, n) for sid, n in zip(sids[1:], lens[1:])]
    new_img = lambda n: torch.full((2, 8, n, 128), float("nan"), dtype=torch.bfloat16, device="cuda")
    one = [new_img(n) for _, _, n in ranges]
    for (sid, t0, n), im in zip(ranges, one):
        sa.sa_kv_session_export(src, sid, t0, n, im)
    many = [new_img(n) for _, _, n in ranges]
    sa.sa_kv_sessions_export(src, [r[0] for r in ranges], [r[1] for r in ranges], [r[2] for r in ranges], many)
    assert sa.sa_last_launch_count(src) == (1 if len(ranges) <= 64 else 2)
    torch.cuda.synchronize()
    for a, b in zip(one, many):
        assert torch.equal(_bits(a), _bits(b))
    # import: whole sessions (session 0 from its two pieces joined along tokens), one call vs one call per session
    whole = [torch.cat([many[0], many[1]], dim=2).contiguous()] + many[3:]
    assert [w_.shape[2] for w_ in whole] == lens
    dst_a, dst_b = mk(2), mk(2)
    sa_ids = [sa.sa_kv_session_open(dst_a) for _ in lens]
    sb_ids = [sa.sa_kv_session_open(dst_b) for _ in lens]
    for sid, n, im in zip(sa_ids, lens, whole):
        sa.sa_kv_session_import(dst_a, sid, n, im, 8, 0)
    # the joint call first fails for want of pages without touching anything ...
    free0 = sa.sa_kv_pool_free_pages(dst_b)
    hog = sa.sa_kv_session_open(dst_b)
    sa.sa_rope_kv_append(dst_b, [hog], [0, 9 * 64], _rand(9 * 64, 8, 128, gen, 0.1), _rand(9 * 64, 8, 128, gen, 0.1), None)
    with pytest.raises(sa.SAError) as e:
        sa.sa_kv_sessions_import(dst_b, sb_ids, lens, whole, 8, 0)
    assert e.value.status == sa.SA_ERR_OUT_OF_PAGES and all(sa.sa_kv_session_query(dst_b, s)[0] == 0 for s in sb_ids)
    hog_pages = set(int(x) for x in sa.sa_kv_session_query(dst_b, hog)[1])   # these lose their sentinel to the hog's own data
    sa.sa_kv_session_close(dst_b, hog)
    assert sa.sa_kv_pool_free_pages(dst_b) == free0
    # ... and then does everything in one launch (plus the metadata uploads of a batch too large for the kernel parameters)
    sa.sa_kv_sessions_import(dst_b, sb_ids, lens, whole, 8, 0)
    assert sa.sa_last_launch_count(dst_b) <= (1 if n_sessions <= 64 else 4)
    torch.cuda.synchronize()
    for s_a, s_b, n in zip(sa_ids, sb_ids, lens):
        la, pa = sa.sa_kv_session_query(dst_a, s_a)
        lb, pb = sa.sa_kv_session_query(dst_b, s_b)
        assert la == lb == n
        ka, va = gather_kv(dst_a, list(pa), n)
        kb, vb = gather_kv(dst_b, list(pb), n)
        assert torch.equal(_bits(ka), _bits(kb)) and torch.equal(_bits(va), _bits(vb))
    # sentinel: every slot no session owns is untouched in the jointly imported pool
    kp, vp = pool_views(dst_b)
    owned = {}
    for s_b, n in zip(sb_ids, lens):
        pg = sa.sa_kv_session_query(dst_b, s_b)[1]
        for i, p_ in enumerate(pg):
            owned[int(p_)] = min(64, n - 64 * i)
    sent = np.array(SENT, dtype=np.uint16).view(np.int16).item()
    for pg in range(pages):
        lo = owned.get(pg, 0)
        if lo < 64 and pg not in hog_pages:
            assert (_bits(kp[pg, :, lo:, :]) == sent).all() and (_bits(vp[pg, :, lo:, :]) == sent).all()
    for p_ in (src, dst_a, dst_b):
        sa.sa_kv_pool_destroy(p_)


def test_export_at_the_range_limit_of_a_pool_whose_slabs_are_smaller_than_it():
    """4 x max_sessions ranges in one sa_kv_sessions_export on a pool with many sessions and few pages: its metadata slab
    (64 (max_sessions + 8) + 4 num_pages + 64 KiB + 64 bytes = 198 208 here) holds 6194 ranges of 32 bytes, the documented
    limit is 8192.  The list must go out in slab-sized pieces, never past a slab's end (that used to overwrite the next
    slab of the ring): every image equals the same tokens cut from a whole-session export made through the
    kernel-parameter path, the bytes between and after the images keep their sentinel, and one range more is refused."""
    L = Layer(8, 2, 64, 16, 10000.0)
    max_sessions, pages = 2048, 256
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, pages, max_sessions, 256, L.rope_base, 0)
    nbytes = sa.sa_kv_pool_storage_bytes(cfg)
    storage = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    pool = sa.sa_kv_pool_create(cfg, storage, np.random.default_rng(5).permutation(pages).astype(np.int32))
    rng = np.random.default_rng(6)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(8)
    lens = [int(x) for x in rng.integers(60, 200, size=16)]
    sids = [sa.sa_kv_session_open(pool) for _ in lens]
    whole = []
    for sid, n in zip(sids, lens):
        sa.sa_rope_kv_append(pool, [sid], [0, n], _rand(n, 2, 64, gen, 1.0), _rand(n, 2, 64, gen, 1.0), None)
        im = torch.empty((2, 2, n, 64), dtype=torch.bfloat16, device="cuda")
        sa.sa_kv_session_export(pool, sid, 0, n, im)
        whole.append(im)
    n_ranges = 4 * max_sessions
    which = rng.integers(0, len(sids), size=n_ranges)
    n_tok = rng.integers(0, 5, size=n_ranges)
    n_tok[:3] = 0                      # the list starts with empty ranges
    n_tok[6190:6200] = [0, 3, 0, 0, 4, 1, 0, 0, 2, 0]   # and has some around the cut
    t0 = np.array([rng.integers(0, lens[w] - n + 1) for w, n in zip(which, n_tok)])
    per_tok = 2 * 2 * 64               # bf16 elements of one token in an image
    offs = np.concatenate([[0], np.cumsum(n_tok * per_tok + 8)])   # 16 sentinel bytes after every image
    flat = torch.full((int(offs[-1]),), SENT, dtype=torch.int16, device="cuda")
    images = [flat[int(o): int(o) + int(n) * per_tok].view(torch.bfloat16).view(2, 2, int(n), 64) for o, n in zip(offs[:-1], n_tok)]
    sa.sa_kv_sessions_export(pool, [sids[w] for w in which], t0, n_tok, images)
    assert sa.sa_last_launch_count(pool) == 4          # two pieces, each a metadata upload and a gather
    torch.cuda.synchronize()
    for i in range(n_ranges):
        want = whole[which[i]][:, :, int(t0[i]): int(t0[i]) + int(n_tok[i]), :]
        assert torch.equal(_bits(images[i]), _bits(want)), "range %d" % i
    gaps = torch.cat([flat[int(o) - 8: int(o)] for o in offs[1:]])
    assert (gaps == np.array(SENT, dtype=np.uint16).view(np.int16).item()).all()
    with pytest.raises(sa.SAError) as e:
        sa.sa_kv_sessions_export(pool, [sids[0]] * (n_ranges + 1), [0] * (n_ranges + 1), [0] * (n_ranges + 1),
                                 [images[0]] * (n_ranges + 1))
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    # the pool still works: a later attention-free call on it reads the same cache
    again = torch.empty_like(whole[3])
    sa.sa_kv_session_export(pool, sids[3], 0, lens[3], again)
    torch.cuda.synchronize()
    assert torch.equal(_bits(again), _bits(whole[3]))
    sa.sa_kv_pool_destroy(pool)
