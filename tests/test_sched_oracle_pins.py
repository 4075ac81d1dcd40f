"""Pins of the scheduler oracle (oracle/sched_oracle.py) against what PAPER.md section 4 and the
mathematics fix: hand-worked examples (tests/golden/sched_worked_example.txt), closed forms,
special cases and brute force.  CPU only."""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import sched_oracle as so

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sched_worked_example.txt")
MODEL = {"c0": 0.0, "alpha_d": 0.001, "alpha_p": 1e-6, "gemm": [(1, 1.0), (101, 2.0), (201, 4.0)]}


def _gold():
    out = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            out[k] = [float(x) for x in v]
    return out


def test_pair_count_closed_form():
    # L313: A_j = q*prefix + q(q+1)/2; the oracle sums the row lengths term by term
    for q, p in [(1, 0), (1, 20479), (7, 0), (128, 256), (2048, 24576), (256, 12345)]:
        assert so.pairs(q, p) == q * p + q * (q + 1) // 2
    gold_pairs = os.path.join(os.path.dirname(__file__), "golden", "pair_counts.txt")
    for line in open(gold_pairs):
        if line.strip() and not line.startswith("#"):
            q, p, a = (int(x) for x in line.split())
            assert so.pairs(q, p) == a


def test_worked_examples():
    g = _gold()
    assert so.est_batch_latency(MODEL, [1000, 3000], [(100, 500)]) == pytest.approx(g["e1_est"][0], abs=1e-9)
    nd, nl, nb, est = so.schedule_hybrid(MODEL, [1000, 3000, 8000], [(100, 500), (100, 600)], [(100, 1000), (100, 100)], 10.0)
    assert [nd, nl, nb] == [int(x) for x in g["e2_admitted"]] and est == pytest.approx(g["e2_est"][0], abs=1e-9)
    nb, budget, est = so.schedule_prefill_slack(MODEL, [(0.0, 100.0, 100, 500), (10.0, 50.0, 100, 600)], 20.0, [(100, 500)],
                                                [(500, 4000), (500, 6000), (500, 8000)])
    assert budget == pytest.approx(g["e3_budget"][0], abs=1e-9) and nb == int(g["e3_admitted"][0])
    assert est == pytest.approx(g["e3_est"][0], abs=1e-9)
    assert so.dynamic_chunk(MODEL, [1000, 3000], [], 500, 1000, 512, 64, 8.0) == int(g["e4_chunk"][0])


def test_t_gemm_shape():
    # near-constant for small M, exact at the table points, linear beyond (L301-303)
    assert so.t_gemm(MODEL, 0) == so.t_gemm(MODEL, 1) == 1.0
    assert so.t_gemm(MODEL, 101) == 2.0 and so.t_gemm(MODEL, 201) == 4.0
    assert so.t_gemm(MODEL, 51) == pytest.approx(1.5) and so.t_gemm(MODEL, 151) == pytest.approx(3.0)
    assert so.t_gemm(MODEL, 301) == pytest.approx(6.0)
    assert so.t_gemm({"gemm": []}, 1000) == 0.0 and so.t_gemm({"gemm": [(8, 0.5)]}, 1000) == 0.5


def test_eq1_is_additive_and_linear_in_its_sums():
    m = {"c0": 0.0, "alpha_d": 2e-4, "alpha_p": 3e-8, "gemm": []}
    # no GEMM table: decode part linear in sum L (L305-309), prefill part linear in sum A (L311-319)
    a = so.est_batch_latency(m, [100, 200], [])
    b = so.est_batch_latency(m, [], [(64, 1000)])
    assert so.est_batch_latency(m, [100, 200], [(64, 1000)]) == pytest.approx(a + b)
    assert a == pytest.approx(2e-4 * 300) and b == pytest.approx(3e-8 * (64 * 1000 + 64 * 65 // 2))
    assert so.est_batch_latency(m, [300], []) == pytest.approx(a)          # depends on the sum only
    assert so.est_batch_latency(m, [], []) == 0.0


def test_algorithm2_extremes_priorities_and_brute_force():
    rng = np.random.default_rng(0)
    for trial in range(40):
        dec = rng.integers(100, 30000, size=rng.integers(0, 6)).tolist()
        lc = [(int(q), int(p)) for q, p in zip(rng.integers(16, 512, size=rng.integers(0, 4)), rng.integers(0, 20000, size=4))]
        be = [(int(q), int(p)) for q, p in zip(rng.integers(16, 512, size=rng.integers(0, 5)), rng.integers(0, 20000, size=5))]
        full = so.est_batch_latency(MODEL, dec, lc + be)
        assert so.schedule_hybrid(MODEL, dec, lc, be, math.inf)[:3] == (len(dec), len(lc), len(be))
        assert so.schedule_hybrid(MODEL, dec, lc, be, full)[:3] == (len(dec), len(lc), len(be))
        assert so.schedule_hybrid(MODEL, dec, lc, be, 0.0)[:3] == (0, 0, 0) or not (dec or lc or be)
        delta = float(rng.uniform(0.5, 1.2 * full + 1.0))
        nd, nl, nb, est = so.schedule_hybrid(MODEL, dec, lc, be, delta)
        assert est <= delta or (nd, nl, nb) == (0, 0, 0)
        # brute force over prefixes: Eq. 1 is monotone in the batch, so each phase admits the longest prefix that fits
        bd = max(k for k in range(len(dec) + 1) if k == 0 or so.est_batch_latency(MODEL, dec[:k], []) <= delta)
        bl = max(k for k in range(len(lc) + 1) if k == 0 or so.est_batch_latency(MODEL, dec[:bd], lc[:k]) <= delta)
        bb = max(k for k in range(len(be) + 1) if k == 0 or so.est_batch_latency(MODEL, dec[:bd], lc[:bl] + be[:k]) <= delta)
        assert (nd, nl, nb) == (bd, bl, bb)
        # BE work never displaces LC work: removing the BE queue leaves the LC decisions unchanged
        assert so.schedule_hybrid(MODEL, dec, lc, [], delta)[:2] == (nd, nl)
        # a larger bound never admits less
        nd2, nl2, nb2, _ = so.schedule_hybrid(MODEL, dec, lc, be, delta * 1.5)
        assert (nd2, nl2, nb2) >= (nd, nl, nb) or nd2 > nd


def test_algorithm1_budget_and_admission():
    # no LC request waiting: unlimited slack; expired deadline: no budget, nothing admitted
    nb, budget, _ = so.schedule_prefill_slack(MODEL, [], 0.0, [], [(64, 100), (64, 200)])
    assert budget == math.inf and nb == 2
    nb, budget, _ = so.schedule_prefill_slack(MODEL, [(0.0, 10.0, 100, 500)], 50.0, [(100, 500)], [(64, 100)])
    assert budget == 0.0 and nb == 0
    # the binding request is the one with the least slack after the prefills queued before it (line 7)
    q = [(0.0, 1000.0, 200, 1000), (0.0, 30.0, 50, 100), (0.0, 500.0, 100, 100)]
    p1 = so.est_batch_latency(MODEL, [], [(200, 1000)])
    p2 = p1 + so.est_batch_latency(MODEL, [], [(50, 100)])
    _, budget, _ = so.schedule_prefill_slack(MODEL, q, 5.0, [], [])
    assert budget == pytest.approx(30.0 - 5.0 - p2)
    # in-order admission: a chunk that does not fit stops the scan even if a later, smaller one would fit (R19)
    be = [(64, 100), (4000, 30000), (16, 10)]
    nb, budget, est = so.schedule_prefill_slack(MODEL, [(0.0, 40.0, 64, 64)], 0.0, [(64, 64)], be)
    assert nb == 1 and est <= budget < so.est_batch_latency(MODEL, [], [(64, 64), (64, 100), (4000, 30000)])


def test_dynamic_chunk_is_the_largest_that_fits():
    m = {"c0": 0.01, "alpha_d": 1.5e-4, "alpha_p": 2.5e-8, "gemm": []}
    for prefix, remaining, budget in itertools.product([0, 5000, 30000], [100, 1000, 5000], [0.005, 0.05, 0.2, 1.0, 100.0]):
        q = so.dynamic_chunk(m, [8000] * 4, [], prefix, remaining, 2048, 128, budget)
        top = min(remaining, 2048)
        assert q == top or q % 128 == 0
        if q > 0:
            assert so.est_batch_latency(m, [8000] * 4, [(q, prefix)]) <= budget
        bigger = [x for x in [top] + list(range(128, top, 128)) if x > q]
        assert all(so.est_batch_latency(m, [8000] * 4, [(x, prefix)]) > budget for x in bigger)


def test_fit_recovers_exact_coefficients():
    rng = np.random.default_rng(1)
    sums = [(int(a), int(b)) for a, b in zip(rng.integers(0, 5_000_000, size=20), rng.integers(0, 400_000_000, size=20))]
    ms = [0.05 + 2e-7 * a + 3e-9 * b for a, b in sums]
    c0, ad, ap, err = so.fit(ms, sums, True)
    assert c0 == pytest.approx(0.05, rel=1e-8) and ad == pytest.approx(2e-7, rel=1e-8) and ap == pytest.approx(3e-9, rel=1e-8)
    assert err < 1e-9
    # Eq. 1 literally (no intercept): two points determine the two coefficients (Cramer's rule by hand)
    (l1, a1), (l2, a2) = (1000, 50_000), (4000, 10_000)
    y1, y2 = 2e-4 * l1 + 1e-6 * a1, 2e-4 * l2 + 1e-6 * a2
    c0, ad, ap, _ = so.fit([y1, y2], [(l1, a1), (l2, a2)], False)
    det = l1 * a2 - l2 * a1
    assert c0 == 0.0 and ad == pytest.approx((y1 * a2 - y2 * a1) / det) and ap == pytest.approx((l1 * y2 - l2 * y1) / det)
    # decode-only profile: alpha_p is not identifiable and stays 0
    c0, ad, ap, _ = so.fit([0.1 + 1e-6 * x for x in (10, 20, 30)], [(10, 0), (20, 0), (30, 0)], True)
    assert ap == 0.0 and ad == pytest.approx(1e-6) and c0 == pytest.approx(0.1)
