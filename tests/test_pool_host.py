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
    tile = 256 if st["tcgen05"] else 64
    assert st["prefill_ctas"] == 8 * (2048 * 4 // tile)
    # a request cannot have more query rows than cached tokens (append first, then attend)
    with pytest.raises(sa.SAError):
        sa.sa_mixed_attention_plan(p, [sids[3]], [0, 6])
    assert sa.sa_mixed_attention_workspace_bytes(p, sids, [0, 1, 4, 4 + 2048, 4 + 2048]) >= st["partial_rows"] * (128 + 1) * 4
