"""Oracle of the lookahead-aware scheduler core -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain Python, written step by step in the order and notation of PAPER.md section 4
("Lookahead-aware request scheduler", L283-404): the latency model of Eq. 1, Algorithm 1
(slack-aware prefill batching, PD disaggregated) and Algorithm 2 (TBT-bounded hybrid batching, PD
co-located).  Every estimate is re-evaluated from scratch over the whole candidate batch, exactly
as the pseudo-code writes it (``EstBatchLatency(B + {c})``): no running sums, no early exits
beyond the ``break`` the algorithms state.  Nothing here imports or calls the product.

A prefill chunk is a pair (q, prefix): q query tokens over prefix cached tokens (L311); a decode
request is its cache length L (L305).  A model is a dict
``{"c0": ms, "alpha_d": ms per KV token, "alpha_p": ms per causal pair, "gemm": [(M, ms), ...]}``.

Readings (R19 and R25-R28, in this order):
* Algorithm 1, lines 15-17 lost their text in the PDF extraction: on budget overflow the loop
  BREAKS (as Algorithm 2 does at L374-384, and as the in-order lookahead queue of L168 requires).
* ``EstPrefillLatency(r)`` (Alg. 1 line 6) = Eq. 1 of the batch holding r's remaining prefill alone.
* ``T_GEMM(M)`` (L299-303 "offline-profiled lookup table with interpolation"): piecewise linear
  through the table points, constant below the first ("near-constant latency" for small M), the
  last segment's slope beyond the last ("scales approximately linearly"); no table: 0.
* ``c0`` is an intercept the paper's Eq. 1 does not have (fixed cost of launching the attention
  kernels); c0 = 0 gives Eq. 1 literally.

Pins: tests/test_sched_oracle_pins.py (hand-worked examples in tests/golden/sched_worked_example.txt,
closed forms, brute force).
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

import numpy as np

Chunk = Tuple[int, int]  # (q, prefix)


def pairs(q: int, prefix: int) -> int:
    """A_j = sum_{i<q} (prefix + 1 + i)  (L311-313), summed term by term."""
    return sum(prefix + 1 + i for i in range(q))


def t_gemm(model: dict, M: int) -> float:
    tab = model.get("gemm") or []
    if not tab:
        return 0.0
    if len(tab) == 1 or M <= tab[0][0]:
        return float(tab[0][1])
    for (x0, y0), (x1, y1) in zip(tab, tab[1:]):
        if M <= x1:
            return y0 + (M - x0) / (x1 - x0) * (y1 - y0)
    (x0, y0), (x1, y1) = tab[-2], tab[-1]
    return y1 + (M - x1) / (x1 - x0) * (y1 - y0)


def est_batch_latency(model: dict, decode_L: Sequence[int], chunks: Sequence[Chunk]) -> float:
    """Eq. 1 (L349-353): T_GEMM(M) + alpha_d * sum_j L_j + alpha_p * sum_j A_j  (+ c0)."""
    M = len(decode_L) + sum(q for q, _ in chunks)                    # L301
    if M == 0:
        return 0.0
    sum_L = sum(int(L) for L in decode_L)                            # L305-309
    sum_A = sum(pairs(int(q), int(p)) for q, p in chunks)            # L311-319
    return model.get("c0", 0.0) + t_gemm(model, M) + model["alpha_d"] * sum_L + model["alpha_p"] * sum_A


def schedule_hybrid(model: dict, q_dec: Sequence[int], q_lc: Sequence[Chunk], q_be: Sequence[Chunk], delta: float):
    """Algorithm 2 (L363-388).  Returns (admitted decode, LC chunks, BE chunks, estimate of the batch)."""
    B_dec: List[int] = []
    B_pre: List[Chunk] = []
    for r in q_dec:                                                   # line 3
        if est_batch_latency(model, B_dec + [r], B_pre) > delta:      # line 4
            break
        B_dec.append(r)                                               # line 5
    n_lc = 0
    for c in q_lc:                                                    # line 8
        if est_batch_latency(model, B_dec, B_pre + [c]) > delta:      # line 9
            break
        B_pre.append(c)                                               # line 10
        n_lc += 1
    n_be = 0
    for c in q_be:                                                    # line 13
        if est_batch_latency(model, B_dec, B_pre + [c]) > delta:      # line 14
            break
        B_pre.append(c)                                               # line 15
        n_be += 1
    return len(B_dec), n_lc, n_be, est_batch_latency(model, B_dec, B_pre)


def schedule_prefill_slack(model: dict, q_lc: Sequence[Tuple[float, float, int, int]], t_now: float,
                           lc_chunks: Sequence[Chunk], q_be: Sequence[Chunk]):
    """Algorithm 1 (L321-347).  q_lc: (t_arrival, SLO_TTFT, remaining q, prefix) per LC request, already in
    the order of the LC policy (line 2).  lc_chunks = NextChunks(Q_LC) (line 12).
    Returns (admitted BE chunks, t_budget, estimate of the batch)."""
    p = 0.0
    s_min = math.inf                                                  # line 4
    for (t_arr, slo, q, prefix) in q_lc:                              # line 5
        p = p + est_batch_latency(model, [], [(q, prefix)])           # line 6
        s_j = (t_arr + slo) - t_now - p                               # line 7
        s_min = min(s_min, s_j)                                       # line 8
    t_budget = max(0.0, s_min)                                        # line 10
    B_lc = list(lc_chunks)                                            # line 12
    B_be: List[Chunk] = []                                            # line 13
    for c in q_be:                                                    # line 14
        if est_batch_latency(model, [], B_lc + B_be + [c]) > t_budget:   # line 15
            break                                                     # line 16 (reading R19)
        B_be.append(c)                                                # line 17
    return len(B_be), t_budget, est_batch_latency(model, [], B_lc + B_be)


def dynamic_chunk(model: dict, decode_L: Sequence[int], chunks: Sequence[Chunk], prefix: int, remaining: int,
                  max_chunk: int, granularity: int, budget: float) -> int:
    """The largest next chunk of a lookahead prefill (L59 "dynamic chunks", L359, L396) that keeps the batch
    within the budget: q = min(remaining, max_chunk) or a smaller multiple of `granularity`; 0 if none fits.
    Linear scan from the top."""
    top = min(remaining, max_chunk)
    cands = [top] + [q for q in range((top - 1) // granularity * granularity, 0, -granularity) if q < top]
    for q in cands:
        if q > 0 and est_batch_latency(model, decode_L, list(chunks) + [(q, prefix)]) <= budget:
            return q
    return 0


def fit(ms: Sequence[float], sums: Sequence[Tuple[int, int]], with_intercept: bool = True):
    """Least-squares fit of ms ~ c0 + alpha_d * sum_L + alpha_p * sum_A over profiled batches (L303, L309,
    L319 "profiled coefficient").  Returns (c0, alpha_d, alpha_p, max relative error over the points)."""
    y = np.asarray(ms, dtype=np.float64)
    S = np.asarray(sums, dtype=np.float64).reshape(-1, 2)
    cols = [S[:, 0], S[:, 1]]
    if with_intercept:
        cols = [np.ones_like(y)] + cols
    A = np.stack(cols, axis=1)
    use = [j for j in range(A.shape[1]) if np.any(A[:, j] != 0)]     # a column of zeros carries no information
    coef = np.zeros(A.shape[1])
    sol, *_ = np.linalg.lstsq(A[:, use] / np.abs(A[:, use]).max(axis=0), y, rcond=None)
    coef[use] = sol / np.abs(A[:, use]).max(axis=0)
    pred = A @ coef
    rel = np.abs(pred - y) / np.maximum(np.abs(y), 1e-300)
    if not with_intercept:
        coef = np.concatenate([[0.0], coef])
    return float(coef[0]), float(coef[1]), float(coef[2]), float(rel.max())
