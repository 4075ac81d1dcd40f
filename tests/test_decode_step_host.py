"""Host half of the capturable decode iteration (sa_decode_step_prepare) on a HOST-ONLY pool: the page taken when a
session's last page is full, the growth by one token, the split plan of each row (1024-key splits: the
row attends to its whole cache), and the all-or-nothing error behaviour."""
import numpy as np
import pytest

from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.build import build


@pytest.fixture(scope="module", autouse=True)
def _built():
    build()


def _pool(num_pages=256, page_size=16, max_sessions=8, max_tokens=4096, order=None, Hq=8, Hkv=2, D=64):
    cfg = sa.PoolConfig(Hq, Hkv, D, page_size, num_pages, max_sessions, max_tokens, 1e4)
    return sa.sa_kv_pool_create(cfg, free_page_order=order, host_only=True)


def test_prepare_grows_each_session_by_one_and_takes_pages_on_page_boundaries():
    order = np.random.default_rng(1).permutation(256).astype(np.int32)
    p = _pool(order=order)
    a, b, c = (sa.sa_kv_session_open(p) for _ in range(3))
    sa.sa_rope_kv_append(p, [a, b, c], [0, 16, 16 + 1023, 16 + 1023 + 1024], None, None)  # 16 / 1023 / 1024 tokens
    free0 = sa.sa_kv_pool_free_pages(p)
    pages = {s: sa.sa_kv_session_query(p, s)[1] for s in (a, b, c)}
    step = sa.sa_decode_step_create(p, 4, 4096)
    sa.sa_decode_step_prepare(step, [a, b, c])
    # a: page full -> new page; b: slot 15 of its 64th page is free; c: page full -> new page
    la, pa = sa.sa_kv_session_query(p, a)
    lb, pb = sa.sa_kv_session_query(p, b)
    lc, pc = sa.sa_kv_session_query(p, c)
    assert (la, lb, lc) == (17, 1024, 1025)
    assert pa[:-1] == pages[a] and pb == pages[b] and pc[:-1] == pages[c]
    assert sa.sa_kv_pool_free_pages(p) == free0 - 2
    nxt = order[256 - free0:]  # pages are handed out in the pool's order
    assert pa[-1] == int(nxt[0]) and pc[-1] == int(nxt[1])
    st = sa.sa_decode_step_stats(step)
    # splits of 1024 keys over the cache INCLUDING the new token: 17 -> 1, 1024 -> 1, 1025 -> 2; Hkv = 2 items per split
    assert st["requests"] == 3 and st["items"] == 2 * (1 + 1 + 2) and st["capacity"] == 4
    assert st["max_part_rows"] == 4 * 8 * 4
    # a second step on a subset
    sa.sa_decode_step_prepare(step, [c])
    assert sa.sa_kv_session_query(p, c)[0] == 1026 and sa.sa_kv_session_query(p, a)[0] == 17
    assert sa.sa_decode_step_stats(step)["items"] == 4
    sa.sa_decode_step_prepare(step, [])
    assert sa.sa_decode_step_stats(step)["requests"] == 0 and sa.sa_decode_step_stats(step)["items"] == 0


def test_prepare_errors_change_nothing():
    p = _pool(num_pages=5, max_tokens=64)
    a, b = sa.sa_kv_session_open(p), sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [a, b], [0, 32, 64], None, None)   # 2 + 2 pages, both on a page boundary; 1 page left
    step = sa.sa_decode_step_create(p, 2, 33)
    sa.sa_decode_step_prepare(step, [a])                       # fine: takes the last page, a now holds 33 tokens
    state = [sa.sa_kv_session_query(p, s) for s in (a, b)], sa.sa_kv_pool_free_pages(p), sa.sa_decode_step_stats(step)

    def unchanged():
        assert ([sa.sa_kv_session_query(p, s) for s in (a, b)], sa.sa_kv_pool_free_pages(p), sa.sa_decode_step_stats(step)) == state
    for bad, status in (([b], sa.SA_ERR_OUT_OF_PAGES), ([a, a], sa.SA_ERR_INVALID_ARG), ([7], sa.SA_ERR_INVALID_ARG),
                        ([a, b, a], sa.SA_ERR_INVALID_ARG)):
        with pytest.raises(sa.SAError) as e:
            sa.sa_decode_step_prepare(step, bad)
        assert e.value.status == status
        unchanged()
    # the step's own limit on the cache length (33 tokens, own token included)
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_prepare(step, [a])
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    unchanged()
    # enqueue has no device to run on
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_enqueue(step, 1, 1, 1, 1, None, 0.0, 0)
    assert e.value.status == sa.SA_ERR_CUDA


def test_shared_partial_last_page_is_refused():
    p = _pool()
    a = sa.sa_kv_session_open(p)
    sa.sa_rope_kv_append(p, [a], [0, 40], None, None)
    f = sa.sa_kv_session_fork(p, a, 40)        # whole pages shared, the partial one copied
    sa.sa_kv_session_truncate(p, f, 20)        # now ends inside a page it shares with `a`
    step = sa.sa_decode_step_create(p, 2, 128)
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_prepare(step, [f])
    assert e.value.status == sa.SA_ERR_UNSUPPORTED and sa.sa_kv_session_query(p, f)[0] == 20
    sa.sa_decode_step_prepare(step, [a])       # a's own partial page is private
    assert sa.sa_kv_session_query(p, a)[0] == 41


def test_create_arguments():
    p = _pool(max_sessions=4, max_tokens=512)
    for cap, mk in ((0, 64), (5, 64), (2, 0), (2, 513)):
        with pytest.raises(sa.SAError):
            sa.sa_decode_step_create(p, cap, mk)
    assert sa.sa_decode_step_device_bytes(p, 4, 512) > 4 * 8 * 64 * 4


def test_cancel_undoes_the_last_prepare_and_only_that():
    """sa_decode_step_cancel (a prepared step that will not run): lengths back, pages back so that they are handed out in
    the same order again, the step empty; refused when there is nothing to undo or a session moved since."""
    order = np.random.default_rng(2).permutation(256).astype(np.int32)
    p = _pool(order=order)
    a, b, c = (sa.sa_kv_session_open(p) for _ in range(3))
    sa.sa_rope_kv_append(p, [a, b, c], [0, 16, 16 + 20, 16 + 20 + 32], None, None)   # a, c end on a page boundary, b inside one
    step = sa.sa_decode_step_create(p, 4, 4096)
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_cancel(step)                       # nothing prepared yet
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    before = [sa.sa_kv_session_query(p, s) for s in (a, b, c)], sa.sa_kv_pool_free_pages(p)
    sa.sa_decode_step_prepare(step, [a, b, c])
    after = [sa.sa_kv_session_query(p, s) for s in (a, b, c)], sa.sa_kv_pool_free_pages(p)
    assert after[1] == before[1] - 2 and [x[0] for x in after[0]] == [17, 21, 33]
    sa.sa_decode_step_cancel(step)
    assert ([sa.sa_kv_session_query(p, s) for s in (a, b, c)], sa.sa_kv_pool_free_pages(p)) == before
    st = sa.sa_decode_step_stats(step)
    assert st["requests"] == 0 and st["items"] == 0
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_cancel(step)                       # already undone
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    # the same prepare again takes the same pages for the same sessions
    sa.sa_decode_step_prepare(step, [a, b, c])
    assert ([sa.sa_kv_session_query(p, s) for s in (a, b, c)], sa.sa_kv_pool_free_pages(p)) == after
    # a session that moved since the prepare: nothing is undone
    sa.sa_kv_session_truncate(p, b, 5)
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_cancel(step)
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    assert sa.sa_kv_session_query(p, a) == after[0][0] and sa.sa_kv_session_query(p, c) == after[0][2]
    assert sa.sa_kv_session_query(p, b)[0] == 5
    # a failed prepare does not disturb what can be cancelled: the last SUCCESSFUL prepare stays the one that is undone
    sa.sa_decode_step_prepare(step, [a])
    with pytest.raises(sa.SAError):
        sa.sa_decode_step_prepare(step, [a, a])
    sa.sa_decode_step_cancel(step)
    assert sa.sa_kv_session_query(p, a) == after[0][0]


def test_step_may_be_destroyed_after_its_pool():
    """sa_decode_step_destroy reads nothing of the pool (garbage collection may run it after sa_kv_pool_destroy)."""
    p = _pool()
    step = sa.sa_decode_step_create(p, 2, 64)
    sa.sa_kv_pool_destroy(p)
    sa.sa_decode_step_destroy(step)
