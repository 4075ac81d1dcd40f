"""Host logic of the page pool, block tables, sessions and the batch planner, on a HOST-ONLY pool
(no GPU): SURVEY 8(a) steps a1 and a3."""
import numpy as np
import pytest

from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.build import build


@pytest.fixture(scope="module", autouse=True)
def _built():
    build()


def _pool(num_pages=64, page_size=16, max_sessions=4, max_tokens=1024, order=None, Hq=8, Hkv=2, D=64):
    cfg = sa.PoolConfig(Hq, Hkv, D, page_size, num_pages, max_sessions, max_tokens, 1e4)
    return sa.sa_kv_pool_create(cfg, free_page_order=order, host_only=True)


def test_pages_handed_out_in_given_order():
    order = np.random.default_rng(0).permutation(64).astype(np.int32)
    p = _pool(order=order)
    s0, s1 = sa.sa_kv_session_open(p), sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [s0, s1], [0, 40, 57], None, None)  # 40 tokens -> 3 pages, 17 -> 2 pages
    l0, pg0 = sa.sa_kv_session_query(p, s0)
    l1, pg1 = sa.sa_kv_session_query(p, s1)
    assert (l0, l1) == (40, 17)
    assert pg0 == order[:3].tolist() and pg1 == order[3:5].tolist()
    assert sa.sa_kv_pool_free_pages(p) == 59
    # growing inside the last page takes no page; crossing it takes the next of the order
    sa.sa_rope_kv_append(p, [s0], [0, 8], None, None)
    assert sa.sa_kv_session_query(p, s0) == (48, order[:3].tolist())
    sa.sa_rope_kv_append(p, [s0], [0, 1], None, None)
    assert sa.sa_kv_session_query(p, s0) == (49, order[:3].tolist() + [int(order[5])])


def test_truncate_keeps_prefix_pages_and_recycles_tail():
    p = _pool()
    s = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [s], [0, 100], None, None)  # 7 pages
    _, pages = sa.sa_kv_session_query(p, s)
    sa.sa_kv_session_truncate(p, s, 33)  # keeps ceil(33/16) = 3 pages
    ln, kept = sa.sa_kv_session_query(p, s)
    assert ln == 33 and kept == pages[:3]
    assert sa.sa_kv_pool_free_pages(p) == 61
    # most recently freed page is reused first
    sa.sa_rope_kv_append(p, [s], [0, 16], None, None)
    assert sa.sa_kv_session_query(p, s)[1] == pages[:4]
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_truncate(p, s, 1000)
    sa.sa_kv_session_close(p, s)
    assert sa.sa_kv_pool_free_pages(p) == 64
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_query(p, s)


def test_out_of_pages_is_all_or_nothing():
    p = _pool(num_pages=4)
    s0, s1 = sa.sa_kv_session_open(p), sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [s0], [0, 20], None, None)  # 2 pages
    with pytest.raises(sa.SAError) as e:
        sa.sa_rope_kv_append(p, [s0, s1], [0, 10, 60], None, None)  # needs 0 + 4 > 2 free
    assert e.value.status == sa.SA_ERR_OUT_OF_PAGES
    assert sa.sa_kv_session_query(p, s0)[0] == 20 and sa.sa_kv_session_query(p, s1) == (0, [])
    assert sa.sa_kv_pool_free_pages(p) == 2


def test_argument_validation():
    p = _pool(max_sessions=2, max_tokens=64)
    s0 = sa.sa_kv_session_open(p)
    s1 = sa.sa_kv_session_open(p)
    with pytest.raises(sa.SAError) as e:
        sa.sa_kv_session_open(p)
    assert e.value.status == sa.SA_ERR_OUT_OF_SESSIONS
    for sids, indptr in (([s0, s0], [0, 1, 2]), ([s0], [1, 2]), ([s0], [0, -1]), ([7], [0, 1]), ([s0], [0, 65])):
        with pytest.raises(sa.SAError) as e:
            sa.sa_rope_kv_append(p, sids, indptr, None, None)
        assert e.value.status == sa.SA_ERR_INVALID_ARG
    assert sa.sa_kv_session_query(p, s0) == (0, []) and sa.sa_kv_session_query(p, s1) == (0, [])
    # permutation check
    with pytest.raises(sa.SAError):
        _pool(num_pages=4, order=np.array([0, 1, 1, 3], dtype=np.int32))
    # attention on a host-only pool has no fallback
    sa.sa_rope_kv_append(p, [s0], [0, 4], None, None)
    with pytest.raises(sa.SAError) as e:
        sa.sa_mixed_attention(p, [s0], [0, 1], 0, 0)
    assert e.value.status == sa.SA_ERR_CUDA


def test_planner_classes_and_sums():
    # Llama-3-8B-shaped layer: G = 4 -> up to 4 query tokens are "decode-like"
    p = _pool(num_pages=4096, page_size=64, max_sessions=8, max_tokens=65536, Hq=32, Hkv=8, D=128)
    sids = [sa.sa_kv_session_open(p) for _ in range(4)]
    lens = [20480, 3000, 8192 + 2048, 5]
    sa.sa_rope_kv_append(p, sids, np.concatenate([[0], np.cumsum(lens)]), None, None)
    # decode row on 20480, 3 rows on 3000, a 2048-chunk on an 8192 prefix, an empty request
    st = sa.sa_mixed_attention_plan(p, sids, [0, 1, 4, 4 + 2048, 4 + 2048])
    assert st["decode_requests"] == 2 and st["prefill_requests"] == 1
    assert st["decode_ctas"] == 8 * (20 + 3)                 # Hkv x ceil(kv/1024) splits
    assert st["partial_rows"] == 20 * 1 * 32 + 3 * 3 * 32    # [split][token][head]
    assert st["sum_decode_kv"] == 20480 * 1 + 3000 * 3
    assert st["sum_prefill_A"] == 2048 * 8192 + 2048 * 2049 // 2
    assert st["tcgen05"] == 1   # every supported shape has a tcgen05 instantiation
    parts, sm = sa.sa_mixed_attention_schedule(p, sids, [0, 1, 4, 4 + 2048, 4 + 2048])
    assert st["prefill_ctas"] == sm["parts"] == len(parts) >= 8 * (2048 * 4 // 256)
    # a request cannot have more query rows than cached tokens (append first, then attend)
    with pytest.raises(sa.SAError):
        sa.sa_mixed_attention_plan(p, [sids[3]], [0, 6])
    assert sa.sa_mixed_attention_workspace_bytes(p, sids, [0, 1, 4, 4 + 2048, 4 + 2048]) >= st["partial_rows"] * (128 + 1) * 4


def _check_schedule(p, sids, lens_prefix, lens_new, G=4, Hkv=8):
    """Every item (request, kv head, 256-row tile) is covered exactly once, in KV order, by its parts."""
    indptr = np.concatenate([[0], np.cumsum(lens_new)]).astype(np.int32)
    parts, sm = sa.sa_mixed_attention_schedule(p, sids, indptr)
    assert sm["parts"] == len(parts) and sm["ctas"] >= 1
    # parts are grouped by CTA in execution order
    assert (np.diff(parts[:, 0]) >= 0).all()
    items = {}
    for cta, r, g, tile, u0, u1, n_kv, slot in parts.tolist():
        assert 0 <= u0 < u1 <= n_kv
        items.setdefault((r, g, tile), []).append((u0, u1, n_kv, slot, cta))
    n_items, total, n_split, slots = 0, 0, 0, []
    for r, (P, n) in enumerate(zip(lens_prefix, lens_new)):
        if n * G <= 16:
            continue
        for g in range(Hkv):
            for tile in range((n * G + 255) // 256):
                tok_max = min(n - 1, (tile * 256 + 255) // G)
                n_kv = (P + tok_max + 1 + 127) // 128           # keys 0 .. prefix + tok_max
                ps = sorted(items.pop((r, g, tile)))
                assert ps[0][0] == 0 and ps[-1][1] == n_kv and all(a[1] == b[0] for a, b in zip(ps, ps[1:]))
                assert all(x[2] == n_kv for x in ps)
                if len(ps) == 1:
                    assert ps[0][3] == -1
                else:
                    assert [x[3] for x in ps] == list(range(ps[0][3], ps[0][3] + len(ps)))   # consecutive slots, KV order
                    assert len(set(x[4] for x in ps)) == len(ps)                          # on different CTAs
                    n_split += 1
                    slots += [x[3] for x in ps]
                n_items += 1
                total += n_kv
    assert not items, "schedule has parts of items that do not exist"
    assert sorted(slots) == list(range(sm["slots"])) and n_split == sm["split_items"] and total == sm["total_units"]
    load = np.zeros(sm["ctas"], dtype=np.int64)
    for cta, r, g, tile, u0, u1, n_kv, slot in parts.tolist():
        load[cta] += u1 - u0 + 3
    assert load.max() == sm["makespan"]
    return parts, sm, n_items, load


def test_tc5_schedule_covers_items_and_balances():
    p = _pool(num_pages=20000, page_size=64, max_sessions=24, max_tokens=65536, Hq=32, Hkv=8, D=128)
    cases = [
        ([24576], [2048]),                       # config 2's chunk: 256 equal items on 148 CTAs
        ([20480], [512]),                        # a small lookahead chunk: 64 items, fewer than the SMs
        ([0], [100]),                            # one short request without a prefix
        ([8192, 16384, 24576, 32768, 20000, 77], [2048, 2048, 2048, 2048, 1, 3]),   # config 4 shaped, with decode rows
        (list(range(1000, 17000, 1000)), [512 + 211 * i for i in range(16)]),       # ragged like config 3
        ([5, 130, 0, 17], [7, 40, 300, 5]),      # tiny ragged requests
    ]
    for prefix, new in cases:
        sids = [sa.sa_kv_session_open(p) for _ in prefix]
        sa.sa_rope_kv_append(p, sids, np.concatenate([[0], np.cumsum([a + b for a, b in zip(prefix, new)])]), None, None)
        parts, sm, n_items, load = _check_schedule(p, sids, prefix, new)
        ideal = (sm["total_units"] + 3 * n_items) / sm["ctas"]
        # balanced: the makespan is within a few tiles (fixed costs of the extra parts, minimum part) of the ideal
        assert sm["makespan"] <= ideal + 3 * 2 + 4 + 1, (prefix, new, sm, ideal)
        if n_items >= 64 and sm["total_units"] >= 16 * sm["ctas"]:
            assert (load > 0).sum() == sm["ctas"], "a balanced schedule of a large batch uses every CTA"
            assert sm["slots"] <= 2 * sm["ctas"] + n_items // 4
        for sid in sids:
            sa.sa_kv_session_close(p, sid)


# ---- session operations of the commit splice -------------
def test_fork_shares_whole_pages_and_copies_the_partial_one():
    p = _pool(num_pages=32, page_size=16, max_sessions=4)
    src = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [src], [0, 100], None, None)          # 7 pages: 6 full + 4 tokens
    _, pg = sa.sa_kv_session_query(p, src)
    # fork at a page boundary: shares pages, takes none
    f0 = sa.sa_kv_session_fork(p, src, 64)
    assert sa.sa_kv_session_query(p, f0) == (64, pg[:4]) and sa.sa_kv_pool_free_pages(p) == 25
    assert [sa.sa_kv_page_refcount(p, x) for x in pg] == [2, 2, 2, 2, 1, 1, 1]
    # fork inside a page: shares the whole pages below, owns a copy of the page the prefix ends in
    f1 = sa.sa_kv_session_fork(p, src, 70)
    l1, pg1 = sa.sa_kv_session_query(p, f1)
    assert l1 == 70 and pg1[:4] == pg[:4] and pg1[4] not in pg and len(pg1) == 5
    assert sa.sa_kv_pool_free_pages(p) == 24
    assert [sa.sa_kv_page_refcount(p, x) for x in pg[:5]] == [3, 3, 3, 3, 1] and sa.sa_kv_page_refcount(p, pg1[4]) == 1
    # the fork appends on its own pages; the source is untouched
    sa.sa_rope_kv_append(p, [f1], [0, 30], None, None)
    assert sa.sa_kv_session_query(p, src) == (100, pg)
    l1, pg1b = sa.sa_kv_session_query(p, f1)
    assert l1 == 100 and pg1b[:5] == pg1 and not set(pg1b[4:]) & set(pg)
    # closing a holder only frees pages nobody else holds
    sa.sa_kv_session_close(p, src)
    assert [sa.sa_kv_page_refcount(p, x) for x in pg] == [2, 2, 2, 2, 0, 0, 0]
    sa.sa_kv_session_close(p, f0)
    sa.sa_kv_session_close(p, f1)
    assert sa.sa_kv_pool_free_pages(p) == 32 and all(sa.sa_kv_page_refcount(p, x) == 0 for x in range(32))
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_fork(p, src, 0)                            # closed source


def test_append_copies_a_shared_partial_page_on_write():
    p = _pool(num_pages=16, page_size=16, max_sessions=4)
    src = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [src], [0, 64], None, None)           # 4 full pages
    f = sa.sa_kv_session_fork(p, src, 64)
    _, pg = sa.sa_kv_session_query(p, src)
    # truncating the source into a shared page and appending again must not write that page
    sa.sa_kv_session_truncate(p, src, 40)                          # keeps pages 0..2, page 2 is now partly valid
    assert [sa.sa_kv_page_refcount(p, x) for x in pg] == [2, 2, 2, 1]
    free0 = sa.sa_kv_pool_free_pages(p)
    sa.sa_rope_kv_append(p, [src], [0, 4], None, None)
    l, pg2 = sa.sa_kv_session_query(p, src)
    assert l == 44 and pg2[:2] == pg[:2] and pg2[2] != pg[2] and len(pg2) == 3
    assert sa.sa_kv_page_refcount(p, pg[2]) == 1 and sa.sa_kv_page_refcount(p, pg2[2]) == 1
    assert sa.sa_kv_pool_free_pages(p) == free0 - 1
    assert sa.sa_kv_session_query(p, f) == (64, pg)               # the fork still sees the old pages
    # a second append into the now private page takes nothing
    sa.sa_rope_kv_append(p, [src], [0, 2], None, None)
    assert sa.sa_kv_session_query(p, src)[1] == pg2 and sa.sa_kv_pool_free_pages(p) == free0 - 1
    # out of pages: a copy-on-write needs a page like any other growth, and a failed call changes nothing
    q = _pool(num_pages=4, page_size=16, max_sessions=4)
    a = sa.sa_kv_session_open(q)
    sa.sa_rope_kv_append(q, [a], [0, 64], None, None)
    b = sa.sa_kv_session_fork(q, a, 64)
    sa.sa_kv_session_truncate(q, a, 50)
    with pytest.raises(sa.SAError) as e:
        sa.sa_rope_kv_append(q, [a], [0, 1], None, None)
    assert e.value.status == sa.SA_ERR_OUT_OF_PAGES and sa.sa_kv_session_query(q, a)[0] == 50
    with pytest.raises(sa.SAError) as e:
        sa.sa_kv_session_fork(q, a, 50)                            # would need a page for the partial copy
    assert e.value.status == sa.SA_ERR_OUT_OF_PAGES


def test_commit_swaps_block_tables_and_releases_superseded_pages():
    p = _pool(num_pages=32, page_size=16, max_sessions=4)
    main = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [main], [0, 200], None, None)         # 13 pages
    _, pg_main = sa.sa_kv_session_query(p, main)
    # lookahead: keep 3 pages' worth of prefix, rebuild a shorter (transformed) context behind it
    la = sa.sa_kv_session_fork(p, main, 48)
    sa.sa_rope_kv_append(p, [la], [0, 40], None, None)
    l_la, pg_la = sa.sa_kv_session_query(p, la)
    assert l_la == 88 and pg_la[:3] == pg_main[:3]
    sa.sa_kv_session_commit(p, main, la)
    assert sa.sa_kv_session_query(p, main) == (88, pg_la)
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_query(p, la)                              # the lookahead session is gone
    # the 10 superseded pages are free again, the shared prefix pages have one holder
    assert sa.sa_kv_pool_free_pages(p) == 32 - len(pg_la)
    assert [sa.sa_kv_page_refcount(p, x) for x in pg_la] == [1] * len(pg_la)
    assert all(sa.sa_kv_page_refcount(p, x) == 0 for x in pg_main[3:])
    with pytest.raises(sa.SAError):
        sa.sa_kv_session_commit(p, main, main)


def test_import_books_pages_like_an_append_and_validates_the_head_slice():
    """N4 (PAPER.md L426 KV transfer, L424 head sharding): the host half of sa_kv_session_import on a
    host-only pool: same page arithmetic as an append, copy-on-write of a shared partial page, all-or-nothing."""
    order = np.random.default_rng(1).permutation(32).astype(np.int32)
    p = _pool(num_pages=32, order=order, Hkv=2)
    assert sa.sa_kv_wire_bytes(p, 10) == 2 * 2 * 10 * 64 * 2 and sa.sa_kv_wire_bytes(p, 0) == 0
    s = sa.sa_kv_session_open(p)
    sa.sa_kv_session_import(p, s, 40, None, 8, 6)          # heads [6, 8) of an 8-head image: legal
    assert sa.sa_kv_session_query(p, s) == (40, order[:3].tolist())
    sa.sa_kv_session_import(p, s, 9, None, 2, 0)           # crosses into a 4th page
    assert sa.sa_kv_session_query(p, s) == (49, order[:4].tolist())
    for src_heads, head_begin in ((8, 7), (1, 0), (2, -1), (0, 0)):
        with pytest.raises(sa.SAError) as ei:
            sa.sa_kv_session_import(p, s, 4, None, src_heads, head_begin)
        assert ei.value.status == sa.SA_ERR_INVALID_ARG
    free0 = sa.sa_kv_pool_free_pages(p)
    with pytest.raises(sa.SAError) as ei:
        sa.sa_kv_session_import(p, s, 16 * free0 + 16, None, 2, 0)
    assert ei.value.status in (sa.SA_ERR_OUT_OF_PAGES, sa.SA_ERR_INVALID_ARG)
    assert sa.sa_kv_pool_free_pages(p) == free0 and sa.sa_kv_session_query(p, s)[0] == 49
    # a fork holds its own copy of the partial 4th page: importing into the fork leaves the source session's page alone
    f = sa.sa_kv_session_fork(p, s, 49)
    shared = sa.sa_kv_session_query(p, s)[1][3]
    sa.sa_kv_session_import(p, f, 3, None, 2, 0)
    assert sa.sa_kv_session_query(p, f)[0] == 52 and sa.sa_kv_session_query(p, s)[1][3] == shared
    # export on a host-only pool: argument checks run, the copy itself needs a device
    with pytest.raises(sa.SAError) as ei:
        sa.sa_kv_session_export(p, s, 40, 10, None)
    assert ei.value.status == sa.SA_ERR_INVALID_ARG


def test_two_appenders_of_one_shared_partial_page_need_one_copy():
    """Two sessions that share a partly filled last page (forked at a page boundary, then both truncated into the shared
    page) append in ONE call: the page is copied for the first appender only -- the second is then its last holder -- so the
    call needs one free page, not two (the demand is min(appenders, holders - 1) per shared page)."""
    p = _pool(num_pages=4, max_sessions=4)
    a = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [a], [0, 40], None, None)          # 3 pages
    b = sa.sa_kv_session_fork(p, a, 32)                        # shares pages 0 and 1, nothing copied
    sa.sa_kv_session_truncate(p, a, 20)                        # page 2 back to the pool; page 1 now partial in both
    sa.sa_kv_session_truncate(p, b, 20)
    c = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [c], [0, 1], None, None)           # takes one of the two free pages
    assert sa.sa_kv_pool_free_pages(p) == 1
    shared = sa.sa_kv_session_query(p, a)[1][1]
    assert sa.sa_kv_session_query(p, b)[1][1] == shared and sa.sa_kv_page_refcount(p, shared) == 2
    sa.sa_rope_kv_append(p, [a, b], [0, 4, 8], None, None)     # both fit in their partial page: one copy-on-write in all
    pa, pb = sa.sa_kv_session_query(p, a)[1], sa.sa_kv_session_query(p, b)[1]
    assert sa.sa_kv_session_query(p, a)[0] == 24 and sa.sa_kv_session_query(p, b)[0] == 24
    assert pa[0] == pb[0] and pa[1] != pb[1] and pb[1] == shared
    assert sa.sa_kv_page_refcount(p, pa[1]) == 1 and sa.sa_kv_page_refcount(p, pb[1]) == 1
    assert sa.sa_kv_pool_free_pages(p) == 0
    # and with no free page left the same situation is refused without touching anything
    sa.sa_kv_session_truncate(p, a, 16)                        # a's private copy back to the pool (1 free page)
    d = sa.sa_kv_session_fork(p, b, 16)                        # shares page 0 only
    sa.sa_rope_kv_append(p, [d], [0, 1], None, None)           # takes the free page
    assert sa.sa_kv_pool_free_pages(p) == 0
    sa.sa_kv_session_truncate(p, a, 8)
    sa.sa_kv_session_truncate(p, d, 8)                         # d's page freed; a, b, d all hold page 0; a and d partial in it
    assert sa.sa_kv_pool_free_pages(p) == 1
    with pytest.raises(sa.SAError):
        sa.sa_rope_kv_append(p, [a, d], [0, 1, 2], None, None)  # holders 3 (b keeps it), appenders 2: two copies, one page
    assert sa.sa_kv_session_query(p, a)[0] == 8 and sa.sa_kv_session_query(p, d)[0] == 8 and sa.sa_kv_pool_free_pages(p) == 1


def test_latency_table_workspace_is_sized_on_a_host_only_twin():
    """sa_latency_table_workspace_bytes replays the run's sessions on a host-only twin of the pool: it needs no device, and
    the figure grows with the decode batch (split partials) on top of the fixed buffers (sources, queries, L2 flush)."""
    p = _pool(num_pages=4096, page_size=64, max_sessions=40, max_tokens=8192, Hq=32, Hkv=8, D=128)
    a = sa.sa_latency_table_workspace_bytes(p, [0, 512], [1], 1024, 512, 2048, 3)
    b = sa.sa_latency_table_workspace_bytes(p, [0, 512], [1, 32], 1024, 512, 2048, 3)
    assert (256 << 20) < a < b < (300 << 20)
    with pytest.raises(sa.SAError) as e:
        sa.sa_latency_table_workspace_bytes(p, [0], [64], 1024, 512, 2048, 3)   # more scratch sessions than the pool has
    assert e.value.status == sa.SA_ERR_OUT_OF_SESSIONS
    assert sa.sa_kv_pool_free_pages(p) == 4096


def test_cached_plan_is_dropped_when_the_batch_or_a_session_changes():
    """The planner keeps the plan of the last batch (sa_mixed_attention_workspace_bytes followed by sa_mixed_attention
    plans once); a different batch, or the same batch after a session grew or shrank, must be planned afresh."""
    p = _pool(num_pages=512, max_tokens=4096)
    a, b = sa.sa_kv_session_open(p), sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [a, b], [0, 1500, 1800], None, None)
    s1 = sa.sa_mixed_attention_plan(p, [a, b], [0, 1, 301])          # a: decode row over 1500, b: 300-token chunk over 300
    assert s1 == sa.sa_mixed_attention_plan(p, [a, b], [0, 1, 301])  # the cached plan answers the same
    ws1 = sa.sa_mixed_attention_workspace_bytes(p, [a, b], [0, 1, 301])
    assert s1["sum_decode_kv"] == 1500 and s1["sum_prefill_A"] == 300 * 301 // 2
    sa.sa_rope_kv_append(p, [a], [0, 700], None, None)               # a grows past another 1024-key split
    s2 = sa.sa_mixed_attention_plan(p, [a, b], [0, 1, 301])
    assert s2["sum_decode_kv"] == 2200 and s2["decode_ctas"] == 3 * 2 and s1["decode_ctas"] == 2 * 2       # decode CTAs = Hkv x splits
    assert sa.sa_mixed_attention_workspace_bytes(p, [a, b], [0, 1, 301]) > ws1
    s3 = sa.sa_mixed_attention_plan(p, [b, a], [0, 300, 301])        # same sessions, other order
    assert s3["sum_decode_kv"] == 2200 and s3["sum_prefill_A"] == s1["sum_prefill_A"]
    s4 = sa.sa_mixed_attention_plan(p, [a, b], [0, 1, 201])          # same sessions, other chunk length
    assert s4["sum_prefill_A"] == 200 * 100 + 200 * 201 // 2
    sa.sa_kv_session_truncate(p, a, 1500)
    assert sa.sa_mixed_attention_plan(p, [a, b], [0, 1, 301]) == s1
