"""The capturable decode iteration (sa_decode_step_prepare + sa_decode_step_enqueue, the TBT path):
bit-equal to sa_rope_kv_append + sa_mixed_attention on a twin pool, eagerly and as ONE captured CUDA graph replayed over
iterations whose batch changes (sessions join and leave, caches cross page and 1024-key split boundaries), and within
the gates of the fp64 oracle."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from gpu_util import check_derived

pytestmark = pytest.mark.gpu


def _bits(t):
    return t.view(torch.int16)


def _twin_pools(Hq, Hkv, D, page, pages, max_sessions, max_tokens, base, seed):
    order = np.random.default_rng(seed).permutation(pages).astype(np.int32)
    cfg = sa.PoolConfig(Hq, Hkv, D, page, pages, max_sessions, max_tokens, base, 0)
    return sa.sa_kv_pool_create(cfg, free_page_order=order), sa.sa_kv_pool_create(cfg, free_page_order=order), cfg


@pytest.mark.parametrize("shape", [(32, 8, 128, 64, 500000.0), (8, 2, 64, 16, 1e4)])
def test_decode_step_graph_replay_equals_eager_calls_bitwise(shape):
    Hq, Hkv, D, page, base = shape
    # caches that sit on and around a page end, a split end (1024 keys) and the empty session
    lens0 = [1023, 1024, 63, 2500, 5000, 0, 64, 2047]
    n = len(lens0)
    iters = 5
    pages = sum((L + iters + page - 1) // page + 1 for L in lens0) + 8
    eager, stepped, cfg = _twin_pools(Hq, Hkv, D, page, pages, n + 1, 8192, base, 5)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1234)
    rnd = lambda t, h: (torch.randn((t, h, D), generator=gen, device="cuda") * 0.7).to(torch.bfloat16)
    hist_k, hist_v = [rnd(L, Hkv) for L in lens0], [rnd(L, Hkv) for L in lens0]
    sids_e = [sa.sa_kv_session_open(eager) for _ in range(n)]
    sids_s = [sa.sa_kv_session_open(stepped) for _ in range(n)]
    live = [i for i in range(n) if lens0[i] > 0]
    indptr = np.concatenate([[0], np.cumsum([lens0[i] for i in live])]).astype(np.int32)
    kk, vv = torch.cat([hist_k[i] for i in live]), torch.cat([hist_v[i] for i in live])
    for pool, sids in ((eager, sids_e), (stepped, sids_s)):
        sa.sa_rope_kv_append(pool, [sids[i] for i in live], indptr, kk, vv, None)
    step = sa.sa_decode_step_create(stepped, n, 8192)
    # static buffers of the captured graph
    k_in, v_in = torch.zeros((n, Hkv, D), dtype=torch.bfloat16, device="cuda"), torch.zeros((n, Hkv, D), dtype=torch.bfloat16, device="cuda")
    q_in, out = torch.zeros((n, Hq, D), dtype=torch.bfloat16, device="cuda"), torch.full((n, Hq, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((n, Hq), float("nan"), dtype=torch.float32, device="cuda")
    graph = None
    batches = [list(range(n)), [0, 3, 5], [1], list(range(n - 1, -1, -1)), [2, 4, 6, 7, 0]]
    for it, batch in enumerate(batches):
        b = len(batch)
        k1, v1, q1 = rnd(b, Hkv), rnd(b, Hkv), rnd(b, Hq)
        # ---- eager reference path on the twin pool
        qe = q1.clone()
        ip = np.arange(b + 1, dtype=np.int32)
        se = [sids_e[i] for i in batch]
        sa.sa_rope_kv_append(eager, se, ip, k1, v1, qe)
        oe, le = torch.empty_like(qe), torch.empty((b, Hq), dtype=torch.float32, device="cuda")
        ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(eager, se, ip), 256), dtype=torch.uint8, device="cuda")
        sa.sa_mixed_attention(eager, se, ip, qe, oe, le, 0.0, ws)
        # ---- the step: host half, then the device half (captured on the first iteration, replayed afterwards)
        torch.cuda.synchronize()                      # the previous replay has consumed the slab
        sa.sa_decode_step_prepare(step, [sids_s[i] for i in batch])
        k_in[:b], v_in[:b], q_in[:b] = k1, v1, q1
        out.fill_(float("nan"))
        lse.fill_(float("nan"))
        if it == 0:
            sa.sa_decode_step_enqueue(step, k_in, v_in, q_in, out, lse)      # eager enqueue of the same two launches
            torch.cuda.synchronize()
            assert sa.sa_decode_step_stats(step)["launches"] == 2
            assert torch.equal(_bits(out[:b]), _bits(oe)) and torch.equal(lse[:b], le) and torch.equal(_bits(q_in[:b]), _bits(qe))
            # enqueue is idempotent for a prepared step; capture it (nothing runs during capture)
            q_in[:b] = q1
            out.fill_(float("nan"))
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                sa.sa_decode_step_enqueue(step, k_in, v_in, q_in, out, lse)
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(_bits(out[:b]), _bits(oe)), "iteration %d: output bits differ from the eager calls" % it
        assert torch.equal(lse[:b], le)
        assert torch.equal(_bits(q_in[:b]), _bits(qe)), "rotated q differs"
        assert torch.isnan(out[b:].float()).all() and torch.isnan(lse[b:]).all(), "rows beyond the step's batch were written"
        for j, i in enumerate(batch):
            hist_k[i] = torch.cat([hist_k[i], k1[j:j + 1]])
            hist_v[i] = torch.cat([hist_v[i], v1[j:j + 1]])
        if it == len(batches) - 1:
            # the oracle on the last iteration's rows (definition: PAPER.md L305, one query over the whole cache)
            for j, i in enumerate(batch):
                L = hist_k[i].shape[0]
                kr = orc.rope(hist_k[i][:L - 1].cpu(), np.arange(L - 1), base)
                ref = orc.oracle_cached(kr, orc.widen(hist_v[i][:L - 1].cpu()), q1[j:j + 1].cpu(), hist_k[i][L - 1:].cpu(),
                                        hist_v[i][L - 1:].cpu(), L - 1, base)
                # gates of DESIGN.md 3a for these inputs: scores of std sm_scale * 0.7 * 0.7 * sqrt(D) = 0.49, V of std 0.7
                check_derived(out[j:j + 1], lse[j:j + 1], ref, 0.49, 0.7, "step row s%d" % i)
    # ---- the caches of the two pools hold the same bits
    for i in range(n):
        Le, Ls = sa.sa_kv_session_query(eager, sids_e[i])[0], sa.sa_kv_session_query(stepped, sids_s[i])[0]
        assert Le == Ls == hist_k[i].shape[0]
        ie = torch.empty((2, Hkv, Le, D), dtype=torch.bfloat16, device="cuda")
        is_ = torch.empty_like(ie)
        sa.sa_kv_session_export(eager, sids_e[i], 0, Le, ie)
        sa.sa_kv_session_export(stepped, sids_s[i], 0, Ls, is_)
        torch.cuda.synchronize()
        assert torch.equal(_bits(ie), _bits(is_)), "session %d: stored K'/V differ" % i
    assert sa.sa_kv_pool_free_pages(eager) == sa.sa_kv_pool_free_pages(stepped)


def test_decode_step_at_config4_scale_equals_the_eager_call_bitwise():
    """64 decode rows on 8 K - 32 K contexts (BASELINE.json config 4's decode set, lengths from the same seed): the
    captured step strides 2368 CTAs over ~11 000 items where the eager call launches one CTA per item; every output
    bit and lse must agree, over two replays, and sampled rows must meet the oracle."""
    Hq, Hkv, D, page, base = 32, 8, 128, 64, 500000.0
    rng = np.random.default_rng(4)
    lens = [int(x) for x in rng.integers(8192, 32768, size=64)]
    n = len(lens)
    pages = sum(L // page + 2 for L in lens) + 8
    eager, stepped, cfg = _twin_pools(Hq, Hkv, D, page, pages, n + 1, 32768 + 64, base, 9)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(4321)
    rnd = lambda t, h: (torch.randn((t, h, D), generator=gen, device="cuda") * D ** -0.5).to(torch.bfloat16)
    src_k, src_v = rnd(32768, Hkv), rnd(32768, Hkv)
    sids_e = [sa.sa_kv_session_open(eager) for _ in range(n)]
    sids_s = [sa.sa_kv_session_open(stepped) for _ in range(n)]
    offs = [int(x) for x in rng.integers(0, 32768 - max(lens), size=n)] if max(lens) < 32768 else [0] * n
    for i, L in enumerate(lens):   # every session a different window of the source
        for pool, sids in ((eager, sids_e), (stepped, sids_s)):
            sa.sa_rope_kv_append(pool, [sids[i]], [0, L], src_k[offs[i]:offs[i] + L], src_v[offs[i]:offs[i] + L], None)
    step = sa.sa_decode_step_create(stepped, n, 32768 + 64)
    k_in, v_in, q_in = rnd(n, Hkv), rnd(n, Hkv), rnd(n, Hq)
    out = torch.empty((n, Hq, D), dtype=torch.bfloat16, device="cuda")
    lse = torch.empty((n, Hq), dtype=torch.float32, device="cuda")
    ip = np.arange(n + 1, dtype=np.int32)
    graph = None
    for it in range(2):
        k1, v1, q1 = rnd(n, Hkv), rnd(n, Hkv), rnd(n, Hq)
        qe = q1.clone()
        sa.sa_rope_kv_append(eager, sids_e, ip, k1, v1, qe)
        oe, le = torch.empty_like(qe), torch.empty((n, Hq), dtype=torch.float32, device="cuda")
        ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(eager, sids_e, ip), 256), dtype=torch.uint8, device="cuda")
        sa.sa_mixed_attention(eager, sids_e, ip, qe, oe, le, 0.0, ws)
        torch.cuda.synchronize()
        sa.sa_decode_step_prepare(step, sids_s)
        k_in.copy_(k1), v_in.copy_(v1), q_in.copy_(q1)
        if graph is None:
            sa.sa_decode_step_enqueue(step, k_in, v_in, q_in, out, lse)
            torch.cuda.synchronize()
            assert torch.equal(_bits(out), _bits(oe)) and torch.equal(lse, le)
            q_in.copy_(q1)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                sa.sa_decode_step_enqueue(step, k_in, v_in, q_in, out, lse)
        out.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        st = sa.sa_decode_step_stats(step)
        assert st["items"] == sum(Hkv * ((L + it + 1 + 1023) // 1024) for L in lens) and st["grid_ctas"] == 16 * torch.cuda.get_device_properties(0).multi_processor_count
        assert torch.equal(_bits(out), _bits(oe)), "replay %d differs from the eager call" % it
        assert torch.equal(lse, le)
        if it == 1:
            for i in (0, 17, 63):   # the oracle on three rows of the last iteration
                L = lens[i] + 2
                kk = torch.cat([src_k[offs[i]:offs[i] + lens[i]], kprev[i:i + 1], k1[i:i + 1]]).cpu()
                vv = torch.cat([src_v[offs[i]:offs[i] + lens[i]], vprev[i:i + 1], v1[i:i + 1]]).cpu()
                kr = orc.rope(kk[:L - 1], np.arange(L - 1), base)
                ref = orc.oracle_cached(kr, orc.widen(vv[:L - 1]), q1[i:i + 1].cpu(), kk[L - 1:], vv[L - 1:], L - 1, base)
                # BASELINE.json's distribution (values N(0,1)/sqrt(128)): its own gates apply (derived terms are far below)
                check_derived(out[i:i + 1], lse[i:i + 1], ref, 128 ** -0.5, 128 ** -0.5, "cfg4-scale step row %d" % i)
        kprev, vprev = k1, v1


def test_decode_step_errors_on_a_device_pool_change_nothing():
    """Error behaviour of the pair on a device pool (include/smoothagent.h): enqueue before any prepare is refused; a
    failed prepare leaves sessions, pages and the step's prepared batch as they were, and a replay after it still
    recomputes the last prepared batch bit for bit."""
    Hq, Hkv, D, page, base = 8, 2, 64, 16, 1e4
    cfg = sa.PoolConfig(Hq, Hkv, D, page, 6, 3, 64, base, 0)
    pool = sa.sa_kv_pool_create(cfg)
    a, b = sa.sa_kv_session_open(pool), sa.sa_kv_session_open(pool)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(5)
    rnd = lambda t, h: torch.randn((t, h, D), generator=gen, device="cuda").to(torch.bfloat16)
    sa.sa_rope_kv_append(pool, [a, b], [0, 32, 64], rnd(64, Hkv), rnd(64, Hkv), None)   # 2 + 2 pages, 2 left
    step = sa.sa_decode_step_create(pool, 2, 40)
    k, v, q = rnd(2, Hkv), rnd(2, Hkv), rnd(2, Hq)
    out = torch.full((2, Hq, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((2, Hq), float("nan"), dtype=torch.float32, device="cuda")
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_enqueue(step, k, v, q, out, lse)
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    sa.sa_decode_step_prepare(step, [a, b])            # takes the two free pages
    q0 = q.clone()
    sa.sa_decode_step_enqueue(step, k, v, q, out, lse)
    torch.cuda.synchronize()
    first = out.clone(), lse.clone()
    assert torch.isfinite(out.float()).all() and sa.sa_kv_pool_free_pages(pool) == 0
    state = [sa.sa_kv_session_query(pool, s) for s in (a, b)], sa.sa_decode_step_stats(step)["items"]
    c = sa.sa_kv_session_open(pool)
    for bad, status in (([c], sa.SA_ERR_OUT_OF_PAGES), ([a, a], sa.SA_ERR_INVALID_ARG), ([a, b, c], sa.SA_ERR_INVALID_ARG)):
        with pytest.raises(sa.SAError) as e:
            sa.sa_decode_step_prepare(step, bad)
        assert e.value.status == status
        assert ([sa.sa_kv_session_query(pool, s) for s in (a, b)], sa.sa_decode_step_stats(step)["items"]) == state
    # the step still holds its last prepared batch: enqueue again re-places the same tokens and recomputes the same rows
    q.copy_(q0)
    out.fill_(float("nan"))
    sa.sa_decode_step_enqueue(step, k, v, q, out, lse)
    torch.cuda.synchronize()
    assert torch.equal(_bits(out), _bits(first[0])) and torch.equal(lse, first[1])
    # a cache longer than the step was created for
    for _ in range(7):                                # one prepare, one execution (include/smoothagent.h)
        sa.sa_decode_step_prepare(step, [a])
        q.copy_(q0)
        sa.sa_decode_step_enqueue(step, k, v, q, out, lse)
    assert sa.sa_kv_session_query(pool, a)[0] == 40
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_prepare(step, [a])
    assert e.value.status == sa.SA_ERR_INVALID_ARG and sa.sa_kv_session_query(pool, a)[0] == 40


def test_cancelled_prepare_leaves_no_trace_on_the_device_path():
    """sa_decode_step_cancel on a device pool: a prepared batch that is dropped instead of executed.  A replay of the
    captured graph after the cancel touches nothing, and the next prepared batch (other sessions, the pages the dropped
    one had taken handed out again) equals the eager calls on a twin pool that never saw the dropped batch, bit for bit."""
    Hq, Hkv, D, page, base = 8, 2, 64, 16, 1e4
    lens0 = [15, 37, 1023, 47]                       # after iteration 0 sessions 0, 2, 3 end on a page boundary
    n = len(lens0)
    eager, stepped, cfg = _twin_pools(Hq, Hkv, D, page, 96, n + 1, 2048, base, 11)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(99)
    rnd = lambda t, h: (torch.randn((t, h, D), generator=gen, device="cuda") * 0.7).to(torch.bfloat16)
    sids_e = [sa.sa_kv_session_open(eager) for _ in range(n)]
    sids_s = [sa.sa_kv_session_open(stepped) for _ in range(n)]
    indptr = np.concatenate([[0], np.cumsum(lens0)]).astype(np.int32)
    kk, vv = rnd(int(indptr[-1]), Hkv), rnd(int(indptr[-1]), Hkv)
    for pool, sids in ((eager, sids_e), (stepped, sids_s)):
        sa.sa_rope_kv_append(pool, sids, indptr, kk, vv, None)
    step = sa.sa_decode_step_create(stepped, n, 2048)
    k_in, v_in, q_in = rnd(n, Hkv), rnd(n, Hkv), rnd(n, Hq)
    out = torch.full((n, Hq, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((n, Hq), float("nan"), dtype=torch.float32, device="cuda")

    def eager_step(batch, k1, v1, q1):
        b = len(batch)
        qe, ip, se = q1.clone(), np.arange(b + 1, dtype=np.int32), [sids_e[i] for i in batch]
        sa.sa_rope_kv_append(eager, se, ip, k1, v1, qe)
        oe, le = torch.empty_like(qe), torch.empty((b, Hq), dtype=torch.float32, device="cuda")
        ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(eager, se, ip), 256), dtype=torch.uint8, device="cuda")
        sa.sa_mixed_attention(eager, se, ip, qe, oe, le, 0.0, ws)
        torch.cuda.synchronize()
        return oe, le

    # iteration 0 on both pools, captured
    k1, v1, q1 = k_in.clone(), v_in.clone(), q_in.clone()
    oe, le = eager_step(list(range(n)), k1, v1, q1)
    sa.sa_decode_step_prepare(step, sids_s)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        sa.sa_decode_step_enqueue(step, k_in, v_in, q_in, out, lse)
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(_bits(out), _bits(oe)) and torch.equal(lse, le)
    # a batch is prepared (sessions 2 and 0 each take a page for it) and dropped
    state = [sa.sa_kv_session_query(stepped, s) for s in sids_s], sa.sa_kv_pool_free_pages(stepped)
    pool_bits = stepped.storage.clone()
    sa.sa_decode_step_prepare(step, [sids_s[1], sids_s[2], sids_s[0]])
    assert sa.sa_kv_pool_free_pages(stepped) == state[1] - 2
    sa.sa_decode_step_cancel(step)
    assert ([sa.sa_kv_session_query(stepped, s) for s in sids_s], sa.sa_kv_pool_free_pages(stepped)) == state
    with pytest.raises(sa.SAError) as e:
        sa.sa_decode_step_enqueue(step, k_in, v_in, q_in, out, lse)      # the step holds no batch
    assert e.value.status == sa.SA_ERR_INVALID_ARG
    out.fill_(float("nan"))
    lse.fill_(float("nan"))
    q_keep = q_in.clone()
    graph.replay()                                                       # an empty step: nothing is placed, no row is written
    torch.cuda.synchronize()
    assert torch.isnan(out.float()).all() and torch.isnan(lse).all() and torch.equal(_bits(q_in), _bits(q_keep))
    kv_bytes = 2 * 96 * Hkv * page * D * 2                               # the K and V pages lead the pool's storage
    assert torch.equal(stepped.storage[:kv_bytes], pool_bits[:kv_bytes]), "a cancelled step wrote into the cache"
    # the next real batch: the twin pool never heard of the dropped one
    batch = [3, 0, 2]
    k1, v1, q1 = rnd(3, Hkv), rnd(3, Hkv), rnd(3, Hq)
    oe, le = eager_step(batch, k1, v1, q1)
    sa.sa_decode_step_prepare(step, [sids_s[i] for i in batch])
    k_in[:3], v_in[:3], q_in[:3] = k1, v1, q1
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(_bits(out[:3]), _bits(oe)) and torch.equal(lse[:3], le)
    for i in range(n):
        assert sa.sa_kv_session_query(eager, sids_e[i]) == sa.sa_kv_session_query(stepped, sids_s[i])
