"""Parity at BASELINE.json's full sizes (configs 2-4; config 5 in test_gpu_config5.py), in the launch
configuration bench.py times: sampled output rows the oracle computes one by one, plus properties
that hold at any size (page-permutation bit-equality, chunked == one-shot within tolerance)."""
import copy

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200 import workloads as wl
from paper_2607_00151_b200.workloads import SessionSpec

from gpu_util import check_lse, check_out, derived_gates, oracle_session, run_workload

V_RMS = 128 ** -0.5   # V of every BASELINE.json config 2-5 workload

pytestmark = pytest.mark.gpu


def _bits(t):
    return t.contiguous().view(torch.int16)


def _sample_check(w, r, data, sessions, n_pairs, seed, lse_tol=1e-3, what="", sigma_logit=None):
    """sigma_logit None: BASELINE.json's distribution and gates (2e-2 / 2e-3, normalised 1e-2, lse 1e-3).  Otherwise the
    "sharp" re-run of reading T-A with scores of that standard deviation: gates from derived_gates."""
    rng = np.random.default_rng(seed)
    worst = (0.0, 0.0, 0.0)
    for i in sessions:
        s = w.sessions[i]
        if s.new == 1:
            rows = np.zeros(w.layer.num_q_heads, dtype=np.int64)
            heads = np.arange(w.layer.num_q_heads, dtype=np.int32)  # decode rows: every head
        else:
            rows = np.concatenate([[0, s.new - 1], rng.integers(0, s.new, size=n_pairs - 2)])
            heads = rng.integers(0, w.layer.num_q_heads, size=n_pairs).astype(np.int32)
        ref = oracle_session(w, i, data, rows=rows, heads=heads)
        out, lse, _ = r.outputs()[i]
        g = out[torch.as_tensor(rows), torch.as_tensor(heads.astype(np.int64))]
        gl = lse[torch.as_tensor(rows), torch.as_tensor(heads.astype(np.int64))]
        if sigma_logit is None:
            e = check_out(g, ref["o"], "%s s%d" % (what, i))
            check_lse(gl, ref["lse"], lse_tol, "%s s%d" % (what, i))
        else:
            mx, mn, rl, lt = derived_gates(sigma_logit, float(np.abs(ref["o"]).max()), V_RMS)
            e = check_out(g, ref["o"], "%s s%d" % (what, i), max_abs=mx, mean_abs=mn, rel_l2=rl)
            check_lse(gl, ref["lse"], lt, "%s s%d" % (what, i))
        worst = tuple(max(a, b) for a, b in zip(worst, e))
    return worst


def test_config2_chunked_reprefill_sampled():
    w = wl.config2()
    pool, r, data = run_workload(w)
    assert len(r.rounds) == 4 and r.rounds[0].q.shape[0] == 2048
    worst = _sample_check(w, r, data, [0], 192, seed=2, what="cfg2")
    print("cfg2 worst (max-abs, mean-abs, rel-L2):", worst)
    # the plan the bench times
    st = sa.sa_mixed_attention_plan(pool, r.rounds[3].sids, r.rounds[3].indptr)
    assert st["sum_prefill_A"] == 2048 * 30720 + 2048 * 2049 // 2 and st["decode_requests"] == 0
    # a different physical page map gives bit-identical outputs
    other = np.random.default_rng(777).permutation(w.num_pages).astype(np.int32)
    pool2, r2, _ = run_workload(w, other, data=data)
    assert torch.equal(_bits(r.outputs()[0][0]), _bits(r2.outputs()[0][0]))
    assert torch.equal(r.outputs()[0][1], r2.outputs()[0][1])
    # chunked (4 x 2048) == one-shot (8192 rows) within tolerance
    w1 = copy.deepcopy(w)
    w1.sessions = [SessionSpec(24576, 8192)]
    pool3, r3, _ = run_workload(w1, data=data)
    a = r.outputs()[0][0].double()
    b = r3.outputs()[0][0].double()
    assert ((a - b).norm() / b.norm()).item() <= 1e-2 and (a - b).abs().max().item() <= 2e-2


@pytest.mark.parametrize("sigma_logit", [1.0, 4.0])
def test_config2_sharp_values_sampled(sigma_logit):
    """Reading T-A: BASELINE.json's distribution gives scores of std 0.008 (a near-uniform softmax), so every config is
    run again with Q, K ~ N(0, sigma^2) unscaled: scores of std sigma_q * sigma_k = 1 ("sharp": the running max moves, the O
    rescale fires) and, here, 4 ("peaked": a handful of keys carry each row)."""
    w = wl.config2()
    pool, r, data = run_workload(w, scale=sigma_logit ** 0.5)
    worst = _sample_check(w, r, data, [0], 96, seed=22, what="cfg2 sharp %g" % sigma_logit, sigma_logit=sigma_logit)
    print("cfg2 sigma_logit %g worst:" % sigma_logit, worst)


def test_config3_sharp_values_sampled():
    w = wl.config3()
    pool, r, data = run_workload(w, scale=1.0, sentinel=0x7FC1)
    worst = _sample_check(w, r, data, range(16), 24, seed=33, what="cfg3 sharp", sigma_logit=1.0)
    print("cfg3 sharp worst:", worst)


def test_config4_sharp_values_sampled():
    w = wl.config4()
    pool, r, data = run_workload(w, scale=1.0, sentinel=0x7FC1)
    worst = _sample_check(w, r, data, list(range(68)), 48, seed=44, what="cfg4 sharp", sigma_logit=1.0)
    print("cfg4 sharp worst:", worst)


def test_config3_ragged_batch_sampled():
    w = wl.config3()
    assert len(w.sessions) == 16 and all(1024 <= s.prefix <= 16384 and 512 <= s.new <= 4096 for s in w.sessions)
    pool, r, data = run_workload(w, sentinel=0x7FC1)   # NaN in every unused slot (R11)
    assert len(r.rounds) == 1 and len(r.rounds[0].sids) == 16
    worst = _sample_check(w, r, data, range(16), 24, seed=3, what="cfg3")
    print("cfg3 worst:", worst)


def test_config4_mixed_lookahead_batch_sampled():
    w = wl.config4()
    pool, r, data = run_workload(w, sentinel=0x7FC1)
    assert len(r.rounds) == 1 and len(r.rounds[0].sids) == 68
    st = sa.sa_mixed_attention_plan(pool, r.rounds[0].sids, r.rounds[0].indptr)
    assert st["prefill_requests"] == 4 and st["decode_requests"] == 64
    assert st["sum_prefill_A"] == w.pair_count() and st["sum_decode_kv"] == w.decode_kv_tokens()
    dec = list(range(4, 68))   # every decode row, every head ("decode rows checked individually")
    worst = _sample_check(w, r, data, [0, 1, 2, 3] + dec, 48, seed=4, what="cfg4")
    print("cfg4 worst:", worst)
    # co-batching must not change a row's bits: decode-only and prefill-only calls on the same rows
    rd = r.rounds[0]
    for group in (list(range(4)), list(range(4, 68))):
        sids = [rd.sids[j] for j in group]
        qs = [rd.q[int(rd.indptr[j]): int(rd.indptr[j + 1])] for j in group]
        indptr = np.concatenate([[0], np.cumsum([t.shape[0] for t in qs])]).astype(np.int32)
        q = torch.cat(qs).contiguous()
        out = torch.empty_like(q)
        ws = torch.empty(max(sa.sa_mixed_attention_workspace_bytes(pool, sids, indptr), 256), dtype=torch.uint8, device="cuda")
        sa.sa_mixed_attention(pool, sids, indptr, q, out, None, 0.0, ws)
        torch.cuda.synchronize()
        ref = torch.cat([rd.out[int(rd.indptr[j]): int(rd.indptr[j + 1])] for j in group])
        assert torch.equal(_bits(out), _bits(ref))
