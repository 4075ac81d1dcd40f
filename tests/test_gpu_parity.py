"""GPU parity tests: the CUDA path (through the C-ABI) against the fp64 oracle on the same seeded
inputs, plus the bit-exact invariants of BASELINE.json's north_star.  Run with -m gpu on a B200."""
import copy

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200 import workloads as wl
from paper_2607_00151_b200.harness import Runner, gather_kv, make_pool, pool_views
from paper_2607_00151_b200.workloads import Layer, SessionSpec, Workload, gen_session

from gpu_util import (bf16_rne, check_derived, check_lse, check_out, check_rope_k, oracle_session, oracle_session_stored,
                      run_workload)

pytestmark = pytest.mark.gpu

SENT = 0x7FC1  # a bf16 NaN pattern used as "untouched slot" sentinel


def _bits(t):
    return t.contiguous().view(torch.int16)


def _small_l8b(sessions, seed=11, pages=None, scale=128 ** -0.5, B=64, D=128, Hq=32, Hkv=8):
    used = sum((s.total + B - 1) // B for s in sessions)
    return Workload("small", Layer(Hq, Hkv, D, B, 500000.0), sessions, num_pages=pages or (used * 2 + 8),
                    value_scale=scale, seed=seed)


# ------------------------------------------------------------------ config 1: append
def test_cfg1_append_placement_and_rope():
    w = wl.config1()
    s = w.sessions[0]
    pool, r, data = run_workload(w, "random", sentinel=SENT)
    k_raw, v_raw, q_raw = data[0]
    ln, pages = sa.sa_kv_session_query(pool, r.sids[0])
    assert ln == s.total and len(pages) == (s.total + 15) // 16
    assert pages == w.page_order()[: len(pages)].tolist()
    k_gpu, v_gpu = r.gather_kv(0)
    # V: a bit copy
    assert torch.equal(_bits(v_gpu), _bits(v_raw))
    # K': RoPE at absolute positions 0..383 (gate 1e-2 with reading T-B)
    k_ref = orc.rope(k_raw.cpu(), np.arange(s.total), w.layer.rope_base)
    err, n_unattainable = check_rope_k(k_gpu, k_ref, "cfg1 K'")
    assert n_unattainable < 50
    # and much tighter in the bulk: at most 1 bf16 ulp from the correctly rounded value
    rne = bf16_rne(k_ref)
    g = k_gpu.double().cpu().numpy()
    ulp = 2.0 ** (np.floor(np.log2(np.maximum(np.abs(rne), 1e-30))) - 7)
    assert (np.abs(g - rne) <= ulp + 1e-30).all()
    assert (g == rne).mean() > 0.99
    # Q' rotated in place at positions prefix..prefix+N-1
    q_ref = orc.rope(q_raw.cpu(), np.arange(s.prefix, s.total), w.layer.rope_base)
    check_rope_k(r.outputs()[0][2], q_ref, "cfg1 Q'")
    # every slot the calls did not address keeps its sentinel bits
    kp, vp = pool_views(pool)
    used = torch.zeros(w.num_pages, dtype=torch.bool)
    used[torch.as_tensor(pages)] = True
    sent = np.array(SENT, dtype=np.uint16).view(np.int16).item()
    assert (_bits(kp[~used]) == sent).all() and (_bits(vp[~used]) == sent).all()
    # identity page map gives the same K' bits (placement does not touch the arithmetic)
    pool2, r2, _ = run_workload(w, "identity", sentinel=SENT, data=data)
    assert sa.sa_kv_session_query(pool2, r2.sids[0])[1] == list(range(len(pages)))
    k2, v2 = r2.gather_kv(0)
    assert torch.equal(_bits(k2), _bits(k_gpu)) and torch.equal(_bits(v2), _bits(v_gpu))


def test_partial_page_untouched_slots_and_prefix_independence():
    # prefix 21 tokens (page of 16: second page partly filled), segment 10 tokens starting mid-page
    w = Workload("pp", Layer(8, 2, 64, 16, 10000.0), [SessionSpec(21, 10)], num_pages=8, value_scale=1.0, seed=5)
    pool = make_pool(w, 0, "random", sentinel=SENT)
    data = {0: gen_session(w, 0, "cuda")}
    r = Runner(w, pool, data)
    r.fill_prefixes()
    torch.cuda.synchronize()
    kp, vp = pool_views(pool)
    _, pages = sa.sa_kv_session_query(pool, r.sids[0])
    sent = np.array(SENT, dtype=np.uint16).view(np.int16).item()
    # slots 5..15 of the second page are still sentinel after the prefix append
    assert (_bits(kp[pages[1], :, 5:]) == sent).all() and (_bits(vp[pages[1], :, 5:]) == sent).all()
    before_k, before_v = kp[pages[:2]].clone(), vp[pages[:2]].clone()
    r.step()
    torch.cuda.synchronize()
    _, pages2 = sa.sa_kv_session_query(pool, r.sids[0])
    assert pages2 == pages  # 31 tokens still fit the two pages
    # P3b: the stored prefix is untouched by the segment append, bit for bit
    assert torch.equal(_bits(kp[pages[0]]), _bits(before_k[0])) and torch.equal(_bits(vp[pages[0]]), _bits(before_v[0]))
    assert torch.equal(_bits(kp[pages[1], :, :5]), _bits(before_k[1][:, :5]))
    # slots 31-16 = 15 is the only untouched slot of page 1 now
    assert (_bits(kp[pages[1], :, 15:]) == sent).all()
    k_gpu, v_gpu = r.gather_kv(0)
    assert torch.equal(_bits(v_gpu), _bits(data[0][1]))


# ------------------------------------------------------------------ config 1: attention
def test_cfg1_attention_parity_and_decomposability():
    w = wl.config1()
    pool, r, data = run_workload(w)
    ref = oracle_session(w, 0, data)
    out, lse, _ = r.outputs()[0]
    check_out(out, ref["o"], "cfg1 cached")
    check_lse(lse, ref["lse"], 1e-2, "cfg1 cached")
    # head_dim 64 / page 16 runs on the tcgen05 kernel too (one 64-dim half per tile), not on an mma.sync fallback
    assert sa.sa_mixed_attention_plan(pool, r.rounds[0].sids, r.rounds[0].indptr)["tcgen05"] == 1
    # P3a on the GPU: one-shot prefill of the whole 384-token context gives the same rows
    w_full = copy.deepcopy(w)
    w_full.sessions = [SessionSpec(0, 384)]
    k, v, q = data[0]
    g = torch.Generator(device="cuda").manual_seed(99)
    q_all = torch.cat([torch.randn((256, 8, 64), generator=g, device="cuda").to(torch.bfloat16), q])
    pool_f, r_f, _ = run_workload(w_full, data={0: (k, v, q_all)})
    out_f = r_f.outputs()[0][0]
    full = orc.oracle_full(q_all.cpu(), k.cpu(), v.cpu(), w.layer.rope_base)
    check_out(out_f, full["o"], "cfg1 one-shot")
    check_out(out_f[256:], ref["o"], "cfg1 one-shot vs cached oracle")
    # chunked by 32 == one shot within tolerance
    w_ch = copy.deepcopy(w)
    w_ch.sessions = [SessionSpec(256, 128, chunk=32)]
    pool_c, r_c, _ = run_workload(w_ch, data=data)
    assert len(r_c.rounds) == 4
    check_out(r_c.outputs()[0][0], ref["o"], "cfg1 chunked")
    # stored K' of the chunked run equals the one-shot run bit for bit
    assert torch.equal(_bits(r_c.gather_kv(0)[0]), _bits(r.gather_kv(0)[0]))


@pytest.mark.parametrize("sigma_logit", [2.0, 4.0])
def test_cfg1_sharp_values(sigma_logit):
    """Config 1 itself is reading T-A's "sharp" case (N(0,1) values: scores of std 1); here Q, K ~ N(0, sigma^2) with
    sigma^2 = 2 and 4 ("peaked": a handful of keys carry each row): running max and O rescale paths.  Against the unrounded oracle the gates are derived_gates' (the bf16
    storage of K', Q' moves every score by ~2.4e-3 sigma_logit: DESIGN.md 3a); against the oracle evaluated on q', k'
    rounded to bf16 -- what the cache holds -- the same kernel output meets the tighter stored-operand gates."""
    w = wl.config1()
    pool, r, data = run_workload(w, scale=sigma_logit ** 0.5)
    out, lse, _ = r.outputs()[0]
    e = check_derived(out, lse, oracle_session(w, 0, data), sigma_logit, 1.0, "cfg1 sigma %g" % sigma_logit)
    e2 = check_derived(out, lse, oracle_session_stored(w, 0, data), sigma_logit, 1.0, "cfg1 sigma %g, stored operands" % sigma_logit,
                       stored_rounded=True)
    print("cfg1 sigma_logit %g: vs oracle %s; vs oracle on bf16 q', k' %s" % (sigma_logit, e, e2))


def test_cfg1_page_permutation_and_nan_slots_bit_exact():
    w = wl.config1()
    pool_a, r_a, data = run_workload(w, "random", sentinel=0)
    out_a = r_a.outputs()[0][0].clone()
    lse_a = r_a.outputs()[0][1].clone()
    other = np.random.default_rng(12345).permutation(w.num_pages).astype(np.int32)
    pool_b, r_b, _ = run_workload(w, other, sentinel=SENT, data=data)
    assert sa.sa_kv_session_query(pool_a, r_a.sids[0])[1] != sa.sa_kv_session_query(pool_b, r_b.sids[0])[1]
    out_b, lse_b, _ = r_b.outputs()[0]
    assert torch.isfinite(out_b.float()).all()
    assert torch.equal(_bits(out_a), _bits(out_b))
    assert torch.equal(lse_a, lse_b)


def test_nan_in_unused_slots_of_last_page_ragged():
    # lengths that leave the last page partly filled, NaN everywhere else; decode + prefill rows
    sessions = [SessionSpec(100, 37), SessionSpec(70, 1), SessionSpec(0, 50), SessionSpec(1029, 1)]
    w = _small_l8b(sessions)
    pool_a, r_a, data = run_workload(w, "random", sentinel=0)
    pool_b, r_b, _ = run_workload(w, "random", sentinel=SENT, data=data)
    for i in range(len(sessions)):
        oa, ob = r_a.outputs()[i][0], r_b.outputs()[i][0]
        assert torch.isfinite(ob.float()).all()
        assert torch.equal(_bits(oa), _bits(ob))
        ref = oracle_session(w, i, data)
        check_out(ob, ref["o"], "ragged nan s%d" % i)
        check_lse(r_b.outputs()[i][1], ref["lse"], 1e-3, "ragged nan s%d" % i)


def test_causality_bit_exact():
    # P3c: perturbing tokens after position i leaves output rows <= i unchanged, bit for bit
    w = _small_l8b([SessionSpec(90, 200)], scale=1.0)
    pool, r, data = run_workload(w)
    out0 = r.outputs()[0][0].clone()
    k, v, q = (t.clone() for t in data[0])
    cut = 117  # segment row index
    k[90 + cut + 1:] *= -3.0
    v[90 + cut + 1:] += 7.0
    q[cut + 1:] *= 0.5
    pool2, r2, _ = run_workload(w, data={0: (k, v, q)})
    out1 = r2.outputs()[0][0]
    assert torch.equal(_bits(out0[: cut + 1]), _bits(out1[: cut + 1]))
    assert not torch.equal(_bits(out0[cut + 1:]), _bits(out1[cut + 1:]))


def test_uniform_softmax_cumulative_mean_and_constant_v():
    # P2c: Q = 0 -> row i is the mean of v_0..v_{P+i}, lse = ln(P+i+1): every row has a different
    # right answer, so any mask / offset / page slip shows.  P2d: constant V -> o = c.
    sessions = [SessionSpec(333, 300), SessionSpec(2100, 1), SessionSpec(64, 64), SessionSpec(0, 5)]
    w = _small_l8b(sessions)  # v ~ N(0,1)/sqrt(128), x8 below -> std 0.7: the 2e-2 gate binds
    data = {}
    for i in range(len(sessions)):
        k, v, q = gen_session(w, i, "cuda")
        data[i] = (k, v * 8.0, torch.zeros_like(q))
    pool, r, _ = run_workload(w, data=data)
    for i, s in enumerate(sessions):
        v64 = data[i][1].double().cpu().numpy()
        cm = np.cumsum(v64, axis=0) / np.arange(1, s.total + 1)[:, None, None]
        ref = np.repeat(cm[s.prefix:], 4, axis=1)  # q head h reads kv head h // 4
        out, lse, _ = r.outputs()[i]
        g = out.double().cpu().numpy()
        assert np.abs(g - ref).max() <= 2e-2
        assert np.linalg.norm(g - ref) / np.linalg.norm(ref) <= 1e-2
        assert np.abs(lse.double().cpu().numpy() - np.log(s.prefix + 1 + np.arange(s.new))[:, None]).max() <= 1e-4
    c = torch.linspace(-2, 2, 128, device="cuda").to(torch.bfloat16)
    data2 = {i: (data[i][0], c.expand_as(data[i][1]).contiguous(), gen_session(w, i, "cuda")[2]) for i in data}
    pool2, r2, _ = run_workload(w, data=data2)
    for i in data2:
        assert (r2.outputs()[i][0].float() - c.float()).abs().max() <= 2e-2


def test_degenerate_sizes():
    L = Layer(32, 8, 128, 64, 500000.0)
    w = Workload("deg", L, [SessionSpec(0, 1), SessionSpec(0, 3), SessionSpec(5, 0), SessionSpec(0, 129), SessionSpec(63, 1)],
                 num_pages=32, value_scale=1.0, seed=21)
    pool, r, data = run_workload(w)
    for i, s in enumerate(w.sessions):
        if s.new == 0:
            continue
        ref = oracle_session(w, i, data)   # N(0,1) values: scores of std 1, |o| up to |v|max ~ 4.5 (one-key rows)
        check_derived(r.outputs()[i][0], r.outputs()[i][1], ref, 1.0, 1.0, "deg s%d" % i)
    # kv = 1: the row attends only itself, o = v_0 exactly (probability 1)
    assert torch.equal(_bits(r.outputs()[0][0][0]), _bits(data[0][1][0].repeat_interleave(4, dim=0)))
    # n_req = 0 and an all-empty batch are no-ops
    sa.sa_rope_kv_append(pool, [], [0], None, None)
    sa.sa_mixed_attention(pool, [], [0], None, None)
    q = torch.zeros((1, 32, 128), dtype=torch.bfloat16, device="cuda")
    sa.sa_mixed_attention(pool, [r.sids[2]], [0, 0], q, q)
    assert sa.sa_last_launch_count(pool) == 0
    # workspace too small is reported, not overrun
    with pytest.raises(sa.SAError) as e:
        sa.sa_mixed_attention(pool, [r.sids[4]], [0, 1], q, q, None, 0.0, torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.status == sa.SA_ERR_WORKSPACE_TOO_SMALL


def test_mixed_batch_equals_separate_calls_bitwise():
    # co-batching must not change a row's bits: mixed == prefill-only == decode-only
    sessions = [SessionSpec(700, 300), SessionSpec(130, 90), SessionSpec(2500, 1), SessionSpec(1024, 1), SessionSpec(4999, 1)]
    w = _small_l8b(sessions)
    pool, r, data = run_workload(w)
    mixed = {i: (r.outputs()[i][0].clone(), r.outputs()[i][1].clone()) for i in range(len(sessions))}
    rd = r.rounds[0]
    for group in ([0, 1], [2, 3, 4], [4, 0], [1]):
        sids = [rd.sids[j] for j in group]
        qs = [rd.q[int(rd.indptr[j]): int(rd.indptr[j + 1])] for j in group]
        indptr = np.concatenate([[0], np.cumsum([t.shape[0] for t in qs])]).astype(np.int32)
        q = torch.cat(qs).contiguous()
        out = torch.empty_like(q)
        lse = torch.empty((q.shape[0], 32), dtype=torch.float32, device="cuda")
        ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(pool, sids, indptr), 256), dtype=torch.uint8, device="cuda")
        sa.sa_mixed_attention(pool, sids, indptr, q, out, lse, 0.0, ws)
        torch.cuda.synchronize()
        for n, j in enumerate(group):
            a, b = int(indptr[n]), int(indptr[n + 1])
            assert torch.equal(_bits(out[a:b]), _bits(mixed[j][0])), "session %d differs when batched as %r" % (j, group)
            assert torch.equal(lse[a:b], mixed[j][1])
    for i in range(len(sessions)):
        ref = oracle_session(w, i, data)
        check_out(mixed[i][0], ref["o"], "mixed s%d" % i)
        check_lse(mixed[i][1], ref["lse"], 1e-3, "mixed s%d" % i)


def test_decode_row_bits_do_not_depend_on_the_batch_size():
    """Splits depend on the request alone (R17), so a decode row's bits must be the same alone, in a
    40-row batch and in a 140-row batch, whatever launch shape the planner picks, and must meet the oracle
    (PAPER.md L305).  140 forks of one 8000-token session share its pages."""
    L = Layer(32, 8, 128, 64, 500000.0)
    ctx, n_rows = 8000, 140                      # 8 splits per (row, head), the last one ragged
    pages = ctx // 64 + 2 + n_rows + 4           # the forks share the whole pages and own a copy of the partial one
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, pages, n_rows + 2, ctx + 64, L.rope_base, 0)
    storage = torch.empty(sa.sa_kv_pool_storage_bytes(cfg), dtype=torch.uint8, device="cuda")
    pool = sa.sa_kv_pool_create(cfg, storage, np.random.default_rng(3).permutation(pages).astype(np.int32))
    gen = torch.Generator(device="cuda")
    gen.manual_seed(77)
    rnd = lambda n, h: (torch.randn((n, h, 128), generator=gen, device="cuda") * 128 ** -0.5).to(torch.bfloat16)
    k, v, q = rnd(ctx, 8), rnd(ctx, 8), rnd(n_rows, 32)
    base = sa.sa_kv_session_open(pool)
    sa.sa_rope_kv_append(pool, [base], [0, ctx], k, v, None)
    sids = [base] + [sa.sa_kv_session_fork(pool, base, ctx) for _ in range(n_rows - 1)]

    def run(rows):
        ss = [sids[i] for i in rows]
        ip = np.arange(len(rows) + 1, dtype=np.int32)
        qq = q[rows].contiguous()
        out = torch.empty_like(qq)
        lse = torch.empty((len(rows), 32), dtype=torch.float32, device="cuda")
        ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(pool, ss, ip), 256), dtype=torch.uint8, device="cuda")
        sa.sa_mixed_attention(pool, ss, ip, qq, out, lse, 0.0, ws)
        torch.cuda.synchronize()
        return out, lse

    o140, l140 = run(list(range(140)))           # 140 x 8 x 8 = 8960 decode CTAs
    o40, l40 = run(list(range(100, 140)))        # 2560
    assert torch.equal(_bits(o40), _bits(o140[100:])) and torch.equal(l40, l140[100:])
    for i in (0, 57, 139):                       # 64
        o1, l1 = run([i])
        assert torch.equal(_bits(o1[0]), _bits(o140[i])) and torch.equal(l1[0], l140[i])
    # the oracle: every session holds the same 8000 cached tokens; row i queries with q[i] (already rotated) at position 7999
    k_rot = orc.rope(k.cpu(), np.arange(ctx), L.rope_base)
    for i in (0, 139):
        ref = orc.attend(orc.widen(q[i:i + 1].cpu()), k_rot, orc.widen(v.cpu()), ctx - 1)
        check_out(o140[i:i + 1], ref["o"], "decode row %d" % i)
    sa.sa_kv_pool_destroy(pool)


@pytest.mark.parametrize("Hq,Hkv,D,B", [(8, 8, 128, 64), (16, 2, 128, 16), (64, 8, 128, 64), (4, 2, 64, 64), (16, 1, 64, 16)])
def test_shapes_gqa_pages(Hq, Hkv, D, B):
    sessions = [SessionSpec(150, 77), SessionSpec(1100, 1), SessionSpec(0, 200), SessionSpec(40, 2)]
    w = _small_l8b(sessions, seed=31, scale=D ** -0.25, B=B, D=D, Hq=Hq, Hkv=Hkv)
    pool, r, data = run_workload(w, sentinel=SENT)
    for i in range(len(sessions)):
        ref = oracle_session(w, i, data)   # q, k, v ~ N(0, D^-1/2): scores of std D^-1/2
        check_derived(r.outputs()[i][0], r.outputs()[i][1], ref, D ** -0.5, D ** -0.25, "shape s%d" % i)


def test_truncate_then_reprefill_reuses_pages_and_matches():
    # the step is repeatable: truncate to the retained prefix, re-append, re-attend -> same bits
    w = _small_l8b([SessionSpec(300, 200), SessionSpec(500, 1)])
    pool, r, data = run_workload(w)
    a = {i: r.outputs()[i][0].clone() for i in range(2)}
    pages_a = [sa.sa_kv_session_query(pool, s)[1] for s in r.sids]
    r.step()
    torch.cuda.synchronize()
    assert [sa.sa_kv_session_query(pool, s)[1] for s in r.sids] != [] and sa.sa_kv_session_query(pool, r.sids[0])[0] == 500
    for i in range(2):
        assert torch.equal(_bits(a[i]), _bits(r.outputs()[i][0]))
    assert sorted(sum(pages_a, [])) == sorted(sum([sa.sa_kv_session_query(pool, s)[1] for s in r.sids], []))


@pytest.mark.parametrize("B,G", [(16, 4), (64, 2)])
def test_head_dim_64_long_context_stream_k_parts_and_merge(B, G):
    # head_dim 64 on the tcgen05 kernel (DH = 1) at a size where items are cut along KV and merged: a 1500-row chunk on a
    # 9000-token prefix, a second ragged session and a decode row, NaN in every unused slot; sampled rows against the oracle
    sessions = [SessionSpec(9000, 1500), SessionSpec(3001, 700), SessionSpec(5000, 1)]
    w = _small_l8b(sessions, seed=64, scale=64 ** -0.25, B=B, D=64, Hq=4 * G, Hkv=4)
    pool, r, data = run_workload(w, sentinel=0x7FC1)
    st = sa.sa_mixed_attention_plan(pool, r.rounds[0].sids, r.rounds[0].indptr)
    assert st["tcgen05"] == 1 and st["prefill_requests"] == 2 and st["decode_requests"] == 1
    parts, sm = sa.sa_mixed_attention_schedule(pool, r.rounds[0].sids, r.rounds[0].indptr)
    assert sm["split_items"] > 0   # some items are split, so tc5_merge_kernel<1> runs
    rng = np.random.default_rng(640)
    for i, s in enumerate(sessions):
        if s.new == 1:
            rows, heads = np.zeros(4 * G, dtype=np.int64), np.arange(4 * G, dtype=np.int32)
        else:
            rows = np.concatenate([[0, s.new - 1], rng.integers(0, s.new, size=62)])
            heads = rng.integers(0, 4 * G, size=64).astype(np.int32)
        ref = oracle_session(w, i, data, rows=rows, heads=heads)
        out, lse, _ = r.outputs()[i]
        idx = (torch.as_tensor(rows), torch.as_tensor(heads.astype(np.int64)))
        check_derived(out[idx], lse[idx], ref, 64 ** -0.5, 64 ** -0.25, "D64 B%d s%d" % (B, i))
