"""The closed loop of Algorithm 2 on the kernels: a lookahead re-prefill is streamed
chunk by chunk into a forked session WHILE decode iterations run, each hybrid batch built by the scheduler core under the
latency bound delta with a latency model fitted on this device, and committed at the end.

Per iteration: the latency-critical decode rows are admitted first, sa_dynamic_chunk sizes the best-effort chunk that
still fits under delta (Eq. 1 with the coefficients sa_latency_fit gives for an sa_latency_table of this pool),
sa_schedule_hybrid must admit exactly that batch, and the batch then RUNS: one sa_rope_kv_append and one
sa_mixed_attention over the decode rows and the chunk together.

What is checked (nothing of it is a timing: the measured times against delta are printed and are bench.py's business):
  * every executed batch was admitted with an estimate <= delta, chunks are multiples of the granularity except the last,
    and they add up to the segment;
  * the decode rows of every iteration are bit-equal to the same rows run alone on a twin pool (their bits do not depend
    on the chunk they are co-batched with);
  * the committed session's cache is bit-equal to the one a one-shot re-prefill builds on the twin pool (another page map),
    whatever the chunking was, and a decode step on it afterwards is bit-equal too;
  * sampled rows of the streamed segment's outputs meet the fp64 oracle of the one-shot re-prefill within BASELINE.json's
    gates (segment decomposability, L105-109: chunked = one-shot);
  * pages: the lookahead's pages replace the dropped tail's, nothing leaks.
Synthetic lengths and values only (BASELINE.json's distribution: N(0,1)/sqrt(128))."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.workloads import Layer

from gpu_util import check_lse, check_out

pytestmark = pytest.mark.gpu


def _bits(t):
    return t.contiguous().view(torch.int16)


def _pool(L, pages, max_sessions, max_tokens, seed):
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, pages, max_sessions, max_tokens, L.rope_base, 0)
    return sa.sa_kv_pool_create(cfg, free_page_order=np.random.default_rng(seed).permutation(pages).astype(np.int32))


def _attend(pool, sids, indptr, q_rot):
    out = torch.empty_like(q_rot)
    lse = torch.empty((q_rot.shape[0], q_rot.shape[1]), dtype=torch.float32, device="cuda")
    ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(pool, sids, indptr), 256), dtype=torch.uint8, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sa.sa_mixed_attention(pool, sids, indptr, q_rot, out, lse, 0.0, ws)
    e1.record()
    torch.cuda.synchronize()
    return out, lse, e0.elapsed_time(e1)


def test_lookahead_segment_streamed_under_delta_while_decoding_then_committed():
    L = Layer(32, 8, 128, 64, 500000.0)
    Hq, Hkv, D, B = L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size
    P, TAIL, SEG, n_dec, GRAN, MAXC = 3000, 1500, 2600, 8, 128, 2048
    rng = np.random.default_rng(31)
    dec_len0 = [int(x) for x in rng.integers(1500, 5000, size=n_dec)]
    pages = 4096
    loop = _pool(L, pages, 32, 16384, 1)
    twin = _pool(L, pages, 32, 16384, 2)
    g = torch.Generator(device="cuda")
    g.manual_seed(77)
    rnd = lambda n, h: (torch.randn((n, h, D), generator=g, device="cuda") * D ** -0.5).to(torch.bfloat16)

    # ---- the device's latency model: a small profiled table of this pool, fitted (Eq. 1; this path has no GEMMs)
    pt, db = [0, 512, 1024, 2048], [0, n_dec]
    ms, sums = sa.sa_latency_table(loop, pt, db, P + SEG // 2, 1500, 5000, seed=3, warmup=2, iters=5)
    keep = [(a, b) for a in range(len(pt)) for b in range(len(db)) if pt[a] + db[b] > 0]
    model, fit_err = sa.sa_latency_fit([ms[a, b] for a, b in keep], [sums[a, b] for a, b in keep], True)
    assert model.alpha_d_ms > 0 and model.alpha_p_ms > 0
    assert sa.sa_kv_pool_free_pages(loop) == pages                      # the table closed its scratch sessions

    # ---- sessions: the main agent's context (retained prefix + a tail the transformation drops), decode requests
    k_main, v_main = rnd(P + TAIL, Hkv), rnd(P + TAIL, Hkv)
    main = sa.sa_kv_session_open(loop)
    sa.sa_rope_kv_append(loop, [main], [0, P + TAIL], k_main, v_main, None)
    dec_loop = [sa.sa_kv_session_open(loop) for _ in dec_len0]
    dec_twin = [sa.sa_kv_session_open(twin) for _ in dec_len0]
    for i, n in enumerate(dec_len0):
        k, v = rnd(n, Hkv), rnd(n, Hkv)
        sa.sa_rope_kv_append(loop, [dec_loop[i]], [0, n], k, v, None)
        sa.sa_rope_kv_append(twin, [dec_twin[i]], [0, n], k, v, None)
    k_seg, v_seg, q_seg = rnd(SEG, Hkv), rnd(SEG, Hkv), rnd(SEG, Hq)
    free_before = sa.sa_kv_pool_free_pages(loop)

    # delta: what the decode rows alone are estimated to cost at the end of the run plus room for a 512-token chunk at the
    # deepest prefix -- every iteration can then admit at least one granule and none can admit the whole segment
    dec_end = [n + 64 for n in dec_len0]
    delta = sa.sa_est_batch_latency(model, dec_end, [(512, P + SEG)])
    assert sa.sa_est_batch_latency(model, dec_end, [(SEG, P)]) > delta

    # ---- the loop
    look = sa.sa_kv_session_fork(loop, main, P)
    out_seg = torch.empty((SEG, Hq, D), dtype=torch.bfloat16, device="cuda")
    lse_seg = torch.empty((SEG, Hq), dtype=torch.float32, device="cuda")
    done, chunks, report = 0, [], []
    dec_lens = list(dec_len0)
    while done < SEG:
        decode_L = [n + 1 for n in dec_lens]                            # a decode row attends to its cache incl. its own token
        c = sa.sa_dynamic_chunk(model, decode_L, [], P + done, SEG - done, MAXC, GRAN, delta)
        assert c > 0, "delta leaves no room for a lookahead granule"
        assert c == SEG - done or c % GRAN == 0
        n_d, n_lc, n_be, est = sa.sa_schedule_hybrid(model, decode_L, [], [(c, P + done)], delta)
        assert (n_d, n_lc, n_be) == (n_dec, 0, 1) and est <= delta      # Alg. 2 admits exactly the batch that is about to run
        if c < SEG - done:                                              # and would not have admitted a granule more
            assert sa.sa_est_batch_latency(model, decode_L, [(c + GRAN, P + done)]) > delta or c == MAXC
        kd, vd, qd = rnd(n_dec, Hkv), rnd(n_dec, Hkv), rnd(n_dec, Hq)
        sids = dec_loop + [look]
        indptr = np.concatenate([np.arange(n_dec + 1), [n_dec + c]]).astype(np.int32)
        k = torch.cat([kd, k_seg[done:done + c]])
        v = torch.cat([vd, v_seg[done:done + c]])
        q = torch.cat([qd, q_seg[done:done + c]])
        sa.sa_rope_kv_append(loop, sids, indptr, k, v, q)
        out, lse, t_ms = _attend(loop, sids, indptr, q)
        out_seg[done:done + c], lse_seg[done:done + c] = out[n_dec:], lse[n_dec:]
        # the same decode rows alone on the twin pool
        q2 = qd.clone()
        ip = np.arange(n_dec + 1, dtype=np.int32)
        sa.sa_rope_kv_append(twin, dec_twin, ip, kd, vd, q2)
        o2, l2, _ = _attend(twin, dec_twin, ip, q2)
        assert torch.equal(_bits(out[:n_dec]), _bits(o2)) and torch.equal(lse[:n_dec], l2), "decode rows depend on the co-batched chunk"
        report.append((c, est, t_ms))
        chunks.append(c)
        done += c
        dec_lens = [n + 1 for n in dec_lens]
    assert sum(chunks) == SEG and len(chunks) >= 2
    print("delta %.3f ms, fit error %.1f %%; (chunk, estimate ms, measured ms of the attention call, first run, cold): %s"
          % (delta, 100 * fit_err, ", ".join("(%d, %.3f, %.3f)" % r for r in report)))

    # ---- commit: the working context IS the transformed one now; the dropped tail's pages are free again
    sa.sa_kv_session_commit(loop, main, look)
    n_main, pg_main = sa.sa_kv_session_query(loop, main)
    assert n_main == P + SEG and len(pg_main) == (P + SEG + B - 1) // B
    grown = sum((n + len(chunks) + B - 1) // B - (n + B - 1) // B for n in dec_len0)
    assert sa.sa_kv_pool_free_pages(loop) == free_before + (P + TAIL + B - 1) // B - len(pg_main) - grown

    # ---- one-shot re-prefill of the same transformed context on the twin pool: same cache bits, whatever the chunking
    ref = sa.sa_kv_session_open(twin)
    sa.sa_rope_kv_append(twin, [ref], [0, P], k_main[:P].contiguous(), v_main[:P].contiguous(), None)
    sa.sa_rope_kv_append(twin, [ref], [0, SEG], k_seg, v_seg, q_seg.clone())
    img_a = torch.empty((2, Hkv, P + SEG, D), dtype=torch.bfloat16, device="cuda")
    img_b = torch.empty_like(img_a)
    sa.sa_kv_session_export(loop, main, 0, P + SEG, img_a)
    sa.sa_kv_session_export(twin, ref, 0, P + SEG, img_b)
    torch.cuda.synchronize()
    assert torch.equal(_bits(img_a), _bits(img_b)), "the streamed cache differs from the one-shot cache"
    kd, vd, qd = rnd(1, Hkv), rnd(1, Hkv), rnd(1, Hq)
    qa, qb = qd.clone(), qd.clone()
    sa.sa_rope_kv_append(loop, [main], [0, 1], kd, vd, qa)
    sa.sa_rope_kv_append(twin, [ref], [0, 1], kd, vd, qb)
    oa, la, _ = _attend(loop, [main], [0, 1], qa)
    ob, lb, _ = _attend(twin, [ref], [0, 1], qb)
    assert torch.equal(_bits(oa), _bits(ob)) and torch.equal(la, lb)

    # ---- the streamed outputs against the fp64 oracle of the one-shot re-prefill (chunk ends and random rows)
    ends = np.cumsum(chunks)
    rows = np.concatenate([[0], ends - 1, ends[:-1], rng.integers(0, SEG, size=48)]).astype(np.int64)
    heads = rng.integers(0, Hq, size=rows.shape[0]).astype(np.int32)
    kr = orc.rope(k_main[:P].cpu(), np.arange(P), L.rope_base)
    o = orc.oracle_cached(kr, orc.widen(v_main[:P].cpu()), q_seg.cpu(), k_seg.cpu(), v_seg.cpu(), P, L.rope_base, rows=rows, heads=heads)
    ri, hi = torch.as_tensor(rows), torch.as_tensor(heads.astype(np.int64))
    check_out(out_seg[ri, hi], o["o"], "streamed lookahead segment")
    check_lse(lse_seg[ri, hi], o["lse"], 1e-3, "streamed lookahead segment")
    for s in dec_loop + [main]:
        sa.sa_kv_session_close(loop, s)
    assert sa.sa_kv_pool_free_pages(loop) == pages
    sa.sa_kv_pool_destroy(loop)
    sa.sa_kv_pool_destroy(twin)
