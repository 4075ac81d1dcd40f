"""The pins of SURVEY 8(c) that have a GPU side and that test_gpu_parity.py does not run:

  P2a  position 0 is the identity of RoPE: K' and Q' of a token at position 0 keep their input bits;
  P2b  <RoPE(q, a), RoPE(k, b)> depends on a - b only: the same tokens placed a constant number of positions
       later give the same attention (shown through a closed form, see the test);
  P2e  a key whose score dominates ("spike") -- early, late, inside a later stream-K part, inside a later
       decode split, on the diagonal -- gives o = v_spike with no overflow: drives the running max, the lazy
       O rescale (threshold 2^8) and the clamped cubic exp2 of the tcgen05 kernel far past moderate logits.

PAPER.md L311-313 fixes the mask these checks protect; L305 the decode row.  Everything goes through the C ABI.
"""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.harness import gather_kv
from paper_2607_00151_b200.workloads import Layer

from gpu_util import U_BF16, bf16_rne, check_lse, check_out, check_rope_k, derived_gates

pytestmark = pytest.mark.gpu


def _bits(t):
    return t.contiguous().view(torch.int16)


def _pool(L, pages, sessions, max_tokens, seed=1, host_only=False):
    cfg = sa.PoolConfig(L.num_q_heads, L.num_kv_heads, L.head_dim, L.page_size, pages, sessions, max_tokens, L.rope_base, 0)
    order = np.random.default_rng(seed).permutation(pages).astype(np.int32)
    return sa.sa_kv_pool_create(cfg, None, order, host_only=host_only)


def _randn(gen, shape, std):
    return (torch.randn(shape, generator=gen, device="cuda", dtype=torch.float32) * std).to(torch.bfloat16)


def _attend(pool, sids, indptr, q, want_lse=True):
    indptr = np.asarray(indptr, dtype=np.int32)
    out = torch.empty_like(q)
    lse = torch.empty((q.shape[0], q.shape[1]), dtype=torch.float32, device="cuda") if want_lse else None
    ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(pool, sids, indptr), 256), dtype=torch.uint8, device="cuda")
    sa.sa_mixed_attention(pool, sids, indptr, q, out, lse, 0.0, ws)
    torch.cuda.synchronize()
    return out, lse


# ------------------------------------------------------------------------------------------- P2a
@pytest.mark.parametrize("Hq,Hkv,D,B,base,n_sessions", [(8, 2, 64, 16, 1e4, 3), (32, 8, 128, 64, 5e5, 3), (32, 8, 128, 64, 5e5, 70)])
def test_position0_is_a_bit_exact_identity(Hq, Hkv, D, B, base, n_sessions):
    """cos 0 = 1, sin 0 = 0: the first token of a fresh session must come out of sa_rope_kv_append with the bits it
    went in with, K' in the page and Q' in place.  70 sessions take the metadata-slab path of the append, 3 the
    path that carries the metadata in the kernel parameters."""
    L = Layer(Hq, Hkv, D, B, base)
    lens = [1 + 7 * (i % 5) for i in range(n_sessions)]          # 1, 8, 15, ... tokens; token 0 is at position 0
    pool = _pool(L, sum((n + B - 1) // B for n in lens) + 4, n_sessions + 1, 64)
    gen = torch.Generator(device="cuda").manual_seed(100 + n_sessions)
    T = sum(lens)
    k, v, q = _randn(gen, (T, Hkv, D), 1.0), _randn(gen, (T, Hkv, D), 1.0), _randn(gen, (T, Hq, D), 1.0)
    q_in = q.clone()
    sids = [sa.sa_kv_session_open(pool) for _ in lens]
    indptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    sa.sa_rope_kv_append(pool, sids, indptr, k, v, q)
    torch.cuda.synchronize()
    for j, sid in enumerate(sids):
        a = int(indptr[j])
        ln, pages = sa.sa_kv_session_query(pool, sid)
        ks, vs = gather_kv(pool, pages, ln)
        assert torch.equal(_bits(ks[0]), _bits(k[a])), "K' at position 0 is not the input (session %d)" % j
        assert torch.equal(_bits(q[a]), _bits(q_in[a])), "Q' at position 0 is not the input (session %d)" % j
        assert torch.equal(_bits(vs), _bits(v[a: a + ln]))
        if ln > 1:   # and the next position IS rotated
            assert not torch.equal(_bits(ks[1]), _bits(k[a + 1]))
    sa.sa_kv_pool_destroy(pool)


# ------------------------------------------------------------------------------------------- P2b
def test_constant_position_shift_leaves_attention_unchanged():
    """The same P + N real tokens are appended after `shift` dummy tokens whose K and V are zero.  RoPE of a zero key
    is zero at any position, so every dummy key scores exactly 0 and carries no value: with Z0 = exp(lse0) the
    softmax mass of the real keys at shift 0,
        o_shift = o_0 * Z0 / (Z0 + shift),        lse_shift = ln(Z0 + shift)
    hold EXACTLY iff the scores between real tokens depend on their position difference only (pin P2b).  o_0, lse_0
    come from the fp64 oracle at shift 0.  shift = 120000 also puts the real tokens at positions ~2^17 where the
    angle p * theta needs the split-precision product of reading R9: the stored K' is checked there against the
    oracle's RoPE, dimension pair by dimension pair."""
    L = Layer(8, 2, 128, 64, 500000.0)
    P, N = 333, 200
    sig = 3.0 ** 0.5                                  # sigma_q = sigma_k: logits of std 3 (sm_scale * sigma^2 * sqrt(D))
    gen = torch.Generator(device="cuda").manual_seed(2024)
    k = _randn(gen, (P + N, 2, 128), sig)
    v = _randn(gen, (P + N, 2, 128), 1.0)
    q = _randn(gen, (N, 8, 128), sig)
    k_rot0 = orc.rope(k.cpu(), np.arange(P + N), L.rope_base)
    ref0 = orc.oracle_cached(k_rot0[:P], orc.widen(v[:P]), q.cpu(), k[P:].cpu(), v[P:].cpu(), P, L.rope_base)
    Z0 = np.exp(ref0["lse"])
    mx, mn, rl, lt = derived_gates(3.0, float(np.abs(ref0["o"]).max()), 1.0)
    shifts = (0, 4133, 120000)
    pool = _pool(L, (max(shifts) + P + N) // 64 + 8, 2, max(shifts) + P + N + 64)
    outs = {}
    for shift in shifts:
        sid = sa.sa_kv_session_open(pool)
        if shift:
            z = torch.zeros((shift, 2, 128), dtype=torch.bfloat16, device="cuda")
            sa.sa_rope_kv_append(pool, [sid], [0, shift], z, z, None)
        sa.sa_rope_kv_append(pool, [sid], [0, P], k[:P].contiguous(), v[:P].contiguous(), None)
        qq = q.clone()
        sa.sa_rope_kv_append(pool, [sid], [0, N], k[P:].contiguous(), v[P:].contiguous(), qq)
        out, lse = _attend(pool, [sid], [0, N], qq)
        o_exp = ref0["o"] * (Z0 / (Z0 + shift))[:, :, None]
        l_exp = np.log(Z0 + shift)
        g = out.double().cpu().numpy()
        rel = np.linalg.norm(g - o_exp) / np.linalg.norm(o_exp)
        assert np.isfinite(g).all() and rel <= rl, "shift %d: rel-L2 %.3e > %.3e" % (shift, rel, rl)
        # absolute gates scaled by the known shrink factor of this row (the bf16 grid of o shrinks with it)
        shrink = (Z0 / (Z0 + shift))[:, :, None]
        assert (np.abs(g - o_exp) <= mx * np.maximum(shrink, 2.0 ** -7)).all(), "shift %d: max-abs" % shift
        check_lse(lse, l_exp, lt, "shift %d" % shift)
        outs[shift] = (g, lse.double().cpu().numpy())
        # stored K' of the real tokens at their shifted positions against the oracle's RoPE (reading T-B gate) ...
        ln, pages = sa.sa_kv_session_query(pool, sid)
        assert ln == shift + P + N
        ks, vs = gather_kv(pool, pages, ln)
        k_ref = orc.rope(k.cpu(), np.arange(shift, shift + P + N), L.rope_base)
        check_rope_k(ks[shift:], k_ref, "K' at shift %d" % shift)
        # ... and, much tighter, bit-equal to the correctly rounded value in >= 97 % of the elements of EVERY dimension
        # pair, the fastest-rotating ones (m = 0..3: an fp32 product p * theta would be off by ~7e-3 rad there) included
        same = (ks[shift:].double().cpu().numpy() == bf16_rne(k_ref))
        per_dim = same.reshape(-1, 128).mean(axis=0)
        assert per_dim.min() >= 0.97, "shift %d: dim %d only %.3f bit-equal to RNE" % (shift, per_dim.argmin(), per_dim.min())
        assert torch.equal(_bits(vs[shift:]), _bits(v))
        if shift:
            assert not ks[:shift].any() and not vs[:shift].any()      # RoPE(0) = 0 exactly
        sa.sa_kv_session_close(pool, sid)
    # GPU against GPU: undo the closed-form factor and the three runs agree with each other as well
    for shift in shifts[1:]:
        back = outs[shift][0] * ((Z0 + shift) / Z0)[:, :, None]
        rel = np.linalg.norm(back - outs[0][0]) / np.linalg.norm(outs[0][0])
        assert rel <= 1.5 * rl, "shift %d vs shift 0 on the GPU: %.3e" % (shift, rel)
    sa.sa_kv_pool_destroy(pool)


# ------------------------------------------------------------------------------------------- P2e
SP = [60, 61, 62, 63]            # spike dimensions: theta_m * 20000 < 0.1 rad at base 5e5, so RoPE barely turns them
QMAG = 24.0                      # q carries QMAG in each spike dimension; a key with k = x gets logit 4 * 24 * x / sqrt(128)


def _spike_mag(logit):
    return logit * (128 ** 0.5) / (len(SP) * QMAG)


def _make_session(gen, total, new, spikes):
    """k, v [total, 8, 128], q [new, 32, 128]; spikes = {key position: target logit}.  Keys that are no spike are zero
    in the spike dimensions (and their RoPE partners), so q's spike dimensions meet spike keys only."""
    sig = 1.0                             # sigma_q = sigma_k = 1 on the 120 regular dimensions -> logit std ~ 0.97
    k = _randn(gen, (total, 8, 128), sig)
    v = _randn(gen, (total, 8, 128), 0.5)
    q = _randn(gen, (new, 32, 128), sig)
    part = [d + 64 for d in SP]
    k[:, :, SP] = 0
    k[:, :, part] = 0
    q[:, :, part] = 0
    q[:, :, SP] = QMAG
    for pos, logit in spikes.items():
        k[pos][:, SP] = torch.tensor(_spike_mag(logit), dtype=torch.bfloat16, device="cuda")
    return k, v, q


def test_spike_keys_early_late_and_across_splits():
    """One mixed call: three 2048-token chunks on a 20,000-token prefix and three decode rows, Llama-3-8B-shaped.
      A  a +200 spike at key 5 (first KV tile: every later tile only adds exp(-200)-sized terms)
      B  spikes arriving LATE and growing: +60 at key 70, +120 inside the SECOND stream-K part of a split item,
         +200 at key prefix-3 (last prefix tile): three O rescales by 2^-86 and below, the last across a merge
      C  a +200 spike INSIDE the chunk (key prefix+1000): rows before it never see it, row 1000 sees it on its diagonal
      D, E, F  decode rows: spike in the first split, in the last split, and +60 early then +200 in a middle split
    Rows that see a spike must return v_spike (the others weigh exp(-60) or less), finite, and match the oracle."""
    L = Layer(32, 8, 128, 64, 500000.0)
    P, N = 20000, 2048
    # where does the schedule cut B's items?  (host-only twin pool with the same lengths: the schedule depends on lengths only)
    twin = _pool(L, 4096, 8, 32768, host_only=True)
    tw = [sa.sa_kv_session_open(twin) for _ in range(6)]
    lens = [P + N, P + N, P + N, 20001, 20001, 20001]
    for sid, n in zip(tw, lens):
        sa.sa_rope_kv_append(twin, [sid], [0, n], None, None, None)
    indptr = np.array([0, N, 2 * N, 3 * N, 3 * N + 1, 3 * N + 2, 3 * N + 3], dtype=np.int32)
    parts, summ = sa.sa_mixed_attention_schedule(twin, tw, indptr)
    assert summ["split_items"] > 0
    later = [p for p in parts if p[1] == 2 and p[7] >= 0 and p[4] > 0 and p[4] * 128 + 7 < P - 200 and p[5] - p[4] >= 2]
    assert later, "the schedule has no later part of a split item of the third request"
    cta, _, g_cut, tile_cut, u0, u1, n_kv, slot = (int(x) for x in later[0])
    mid_key = u0 * 128 + 128 + 7        # second KV tile of that part
    sa.sa_kv_pool_destroy(twin)

    gen = torch.Generator(device="cuda").manual_seed(777)
    # request order A, C, B: the schedule cuts the items it deals last, i.e. those of the third request
    spikes = [{5: 200.0}, {P + 1000: 200.0}, {70: 60.0, mid_key: 120.0, P - 3: 200.0},
              {5: 200.0}, {19990: 200.0}, {100: 60.0, 10300: 200.0}]
    data = [_make_session(gen, n, N if i < 3 else 1, spikes[i]) for i, n in enumerate(lens)]
    pool = _pool(L, sum((n + 63) // 64 for n in lens) + 16, 8, 32768, seed=5)
    sids = [sa.sa_kv_session_open(pool) for _ in lens]
    pre = [n - (N if i < 3 else 1) for i, n in enumerate(lens)]
    p_ind = np.concatenate([[0], np.cumsum(pre)]).astype(np.int32)
    sa.sa_rope_kv_append(pool, sids, p_ind, torch.cat([d[0][:p] for d, p in zip(data, pre)]).contiguous(),
                         torch.cat([d[1][:p] for d, p in zip(data, pre)]).contiguous(), None)
    q = torch.cat([d[2] for d in data]).contiguous()
    sa.sa_rope_kv_append(pool, sids, indptr, torch.cat([d[0][p:] for d, p in zip(data, pre)]).contiguous(),
                         torch.cat([d[1][p:] for d, p in zip(data, pre)]).contiguous(), q)
    parts2, _ = sa.sa_mixed_attention_schedule(pool, sids, indptr)
    assert np.array_equal(parts2, parts)                          # the real pool cuts where the twin said
    out, lse = _attend(pool, sids, indptr, q)
    assert torch.isfinite(out.float()).all() and torch.isfinite(lse).all()

    rng = np.random.default_rng(31)
    for i, n in enumerate(lens):
        k_, v_, q_ = (t.cpu() for t in data[i])
        p_ = pre[i]
        new = n - p_
        a = int(indptr[i])
        if new == 1:
            rows, heads = np.zeros(32, dtype=np.int64), np.arange(32, dtype=np.int32)
        else:
            rows = np.concatenate([[0, new - 1], rng.integers(0, new, size=94)])
            heads = rng.integers(0, 32, size=96).astype(np.int32)
            if i == 2:    # rows of the item whose later part holds the +120 spike: tokens tile*64 .. +63, the 4 heads of kv head g_cut
                toks = np.arange(tile_cut * 64, min(tile_cut * 64 + 64, new), 9)
                rows = np.concatenate([rows, np.repeat(toks, 4)])
                heads = np.concatenate([heads, np.tile(np.arange(g_cut * 4, g_cut * 4 + 4), len(toks))]).astype(np.int32)
            if i == 1:    # around the in-chunk spike
                rows = np.concatenate([rows, [998, 999, 1000, 1001, 1002, 1000, 1000]])
                heads = np.concatenate([heads, [0, 5, 9, 17, 31, 30, 2]]).astype(np.int32)
        k_rot = orc.rope(k_[:p_], np.arange(p_), L.rope_base)
        ref = orc.oracle_cached(k_rot, orc.widen(v_[:p_]), q_, k_[p_:], v_[p_:], p_, L.rope_base, rows=rows, heads=heads)
        ri, hi = torch.as_tensor(rows) + a, torch.as_tensor(heads.astype(np.int64))
        g_o, g_l = out[ri, hi], lse[ri, hi]
        what = "spike session %d" % i
        mx, mn, rl, lt = derived_gates(1.0, float(np.abs(ref["o"]).max()), 0.5)
        check_out(g_o, ref["o"], what, max_abs=mx, mean_abs=mn, rel_l2=rl)
        # a logit of size |s| carried by bf16 operands is off by up to 2 u |s| (both factors rounded); lse follows the top logit
        tol = lt + 2.0 * U_BF16 * np.abs(ref["lse"])
        err = np.abs(g_l.double().cpu().numpy() - ref["lse"])
        assert (err <= tol).all(), "%s: lse error %.3e" % (what, (err - tol).max())
        # rows that see a +200 spike return its value
        top = max(spikes[i], key=lambda kk: spikes[i][kk])
        sees = (p_ + rows) >= top
        assert sees.any()
        if i == 1:
            assert (~sees).any() and np.abs(ref["lse"][~sees]).max() < 30 and ref["lse"][sees].min() > 150
        v_top = v_[top].double().numpy()                       # [8, 128]
        want = v_top[heads[sees] // 4]
        assert np.abs(g_o.double().cpu().numpy()[sees] - want).max() <= 2e-2, what
        assert np.abs(ref["o"][sees] - want).max() <= 1e-9     # (the oracle agrees that nothing else weighs in)
    sa.sa_kv_pool_destroy(pool)
