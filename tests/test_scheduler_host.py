"""The C++ scheduler core (sa_latency_fit, sa_est_batch_latency, sa_schedule_hybrid,
sa_schedule_prefill_slack, sa_dynamic_chunk) against the Python oracle written from PAPER.md
section 4: estimates equal to the last bit (both sides evaluate Eq. 1 in double in the order it is
written), integer decisions identical.  Host only, no GPU."""
import math

import numpy as np
import pytest

from oracle import sched_oracle as so
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.build import build


@pytest.fixture(scope="module", autouse=True)
def _built():
    build()


def _models():
    yield {"c0": 0.0, "alpha_d": 0.001, "alpha_p": 1e-6, "gemm": [(1, 1.0), (101, 2.0), (201, 4.0)]}
    yield {"c0": 0.012, "alpha_d": 1.79e-7, "alpha_p": 1.37e-8, "gemm": []}            # attention-only, like this build
    yield {"c0": 0.0, "alpha_d": 3.1e-7, "alpha_p": 2.2e-8, "gemm": [(16, 0.41)]}
    yield {"c0": 0.0, "alpha_d": 2.5e-7, "alpha_p": 1.9e-8,
           "gemm": [(1, 0.35), (64, 0.36), (256, 0.52), (1024, 1.61), (4096, 6.2), (8192, 12.3)]}


def _to(m):
    return sa.LatencyModel(m["c0"], m["alpha_d"], m["alpha_p"], m["gemm"])


def _rand_batch(rng):
    dec = rng.integers(1, 131072, size=rng.integers(0, 9)).tolist()
    lc = [(int(q), int(p)) for q, p in zip(rng.integers(1, 2049, size=rng.integers(0, 5)), rng.integers(0, 100000, size=5))]
    be = [(int(q), int(p)) for q, p in zip(rng.integers(1, 2049, size=rng.integers(0, 7)), rng.integers(0, 100000, size=7))]
    return dec, lc, be


def test_estimate_bit_equal_to_the_oracle():
    rng = np.random.default_rng(10)
    for m in _models():
        for _ in range(60):
            dec, lc, be = _rand_batch(rng)
            assert sa.sa_est_batch_latency(_to(m), dec, lc + be) == so.est_batch_latency(m, dec, lc + be)
        assert sa.sa_est_batch_latency(_to(m), [], []) == 0.0


def test_algorithm2_decisions_equal_the_oracle():
    rng = np.random.default_rng(11)
    for m in _models():
        for _ in range(80):
            dec, lc, be = _rand_batch(rng)
            full = so.est_batch_latency(m, dec, lc + be)
            for delta in (0.0, float(rng.uniform(0, full + 1e-3)), full, math.inf):
                got = sa.sa_schedule_hybrid(_to(m), dec, lc, be, delta)
                ref = so.schedule_hybrid(m, dec, lc, be, delta)
                assert got[:3] == ref[:3] and got[3] == ref[3], (m, dec, lc, be, delta)


def test_algorithm1_decisions_equal_the_oracle():
    rng = np.random.default_rng(12)
    for m in _models():
        for _ in range(80):
            _, lc, be = _rand_batch(rng)
            queue = [(float(rng.uniform(0, 50)), float(rng.uniform(5, 400)), int(rng.integers(1, 8192)), int(rng.integers(0, 60000)))
                     for _ in range(rng.integers(0, 5))]
            t_now = float(rng.uniform(0, 80))
            got = sa.sa_schedule_prefill_slack(_to(m), queue, t_now, lc[:1], be)
            ref = so.schedule_prefill_slack(m, queue, t_now, lc[:1], be)
            assert got == ref, (m, queue, t_now, lc[:1], be)


def test_dynamic_chunk_equals_the_oracle_scan():
    rng = np.random.default_rng(13)
    for m in _models():
        for _ in range(60):
            dec, lc, _ = _rand_batch(rng)
            prefix, remaining = int(rng.integers(0, 60000)), int(rng.integers(1, 9000))
            gran = int(rng.choice([16, 64, 128, 256]))
            top_est = so.est_batch_latency(m, dec, lc + [(min(remaining, 2048), prefix)])
            budget = float(rng.uniform(0, 1.3 * top_est))
            got = sa.sa_dynamic_chunk(_to(m), dec, lc, prefix, remaining, 2048, gran, budget)
            assert got == so.dynamic_chunk(m, dec, lc, prefix, remaining, 2048, gran, budget)


def test_dynamic_chunk_with_a_non_monotone_model_equals_the_oracle_scan():
    """A measured T_GEMM table (medians) or an unconstrained fit need not be monotone in q; "the largest chunk that fits"
    is then not found by bisection.  The C++ side must fall back to the definition (scan from the top), like the oracle."""
    rng = np.random.default_rng(15)
    models = [
        {"c0": 0.0, "alpha_d": 2.5e-7, "alpha_p": 1.9e-8,   # a dip at M = 256 (a faster kernel variant kicks in)
         "gemm": [(1, 0.35), (64, 0.50), (256, 0.30), (1024, 1.61), (2048, 1.2), (4096, 6.2)]},
        {"c0": 0.5, "alpha_d": 1e-7, "alpha_p": -2e-9, "gemm": [(1, 0.2), (2048, 3.0)]},   # a negative fitted coefficient
    ]
    differs_from_bisection = 0
    for m in models:
        for _ in range(150):
            dec, lc, _ = _rand_batch(rng)
            prefix, remaining = int(rng.integers(0, 60000)), int(rng.integers(1, 9000))
            gran = int(rng.choice([16, 64, 128]))
            top_est = so.est_batch_latency(m, dec, lc + [(min(remaining, 2048), prefix)])
            budget = float(rng.uniform(0.3, 1.1) * top_est)
            ref = so.dynamic_chunk(m, dec, lc, prefix, remaining, 2048, gran, budget)
            assert sa.sa_dynamic_chunk(_to(m), dec, lc, prefix, remaining, 2048, gran, budget) == ref
            # what a bisection that assumes monotonicity would have returned
            top = min(remaining, 2048)
            fits = lambda q: so.est_batch_latency(m, dec, lc + [(q, prefix)]) <= budget
            if not fits(top):
                lo, hi = 0, (top - 1) // gran
                while lo < hi:
                    mid = (lo + hi + 1) // 2
                    lo, hi = (mid, hi) if fits(mid * gran) else (lo, mid - 1)
                differs_from_bisection += int(lo * gran != ref)
    assert differs_from_bisection > 0   # the instances do exercise the difference
    with pytest.raises(sa.SAError):
        sa.sa_dynamic_chunk(_to(models[0]), [100, -1], [], 0, 100, 2048, 16, 1.0)


def test_fit_equals_numpy_least_squares():
    rng = np.random.default_rng(14)
    for with_c0 in (True, False):
        sums = np.stack([rng.integers(0, 21_000_000, size=20), rng.integers(0, 90_000_000, size=20)], axis=1)
        sums[::5, 1] = 0   # decode-only rows, like the p = 0 row of the latency table
        ms = (0.02 * with_c0 + 1.8e-7 * sums[:, 0] + 1.4e-8 * sums[:, 1]) * rng.uniform(0.97, 1.03, size=20)
        ms = ms.astype(np.float32)
        model, err = sa.sa_latency_fit(ms, sums, with_c0)
        c0, ad, ap, err_ref = so.fit(ms.astype(np.float64), sums, with_c0)
        assert model.c0_ms == pytest.approx(c0, rel=1e-7, abs=1e-12) and model.alpha_d_ms == pytest.approx(ad, rel=1e-7)
        assert model.alpha_p_ms == pytest.approx(ap, rel=1e-7) and err == pytest.approx(err_ref, rel=1e-6)
    # a profile with no prefill chunk leaves alpha_p at 0
    model, _ = sa.sa_latency_fit([0.1, 0.2, 0.3], [[10, 0], [20, 0], [30, 0]], True)
    assert model.alpha_p_ms == 0.0 and model.alpha_d_ms == pytest.approx(0.01)


def test_argument_checks():
    m = _to(next(_models()))
    with pytest.raises(sa.SAError):
        sa.sa_est_batch_latency(m, [-1], [])
    with pytest.raises(sa.SAError):
        sa.sa_dynamic_chunk(m, [], [], 0, 10, 0, 16, 1.0)
    bad = sa.LatencyModel(0, 1e-6, 1e-9, [(10, 1.0), (10, 2.0)])   # table not strictly increasing
    with pytest.raises(sa.SAError):
        sa.sa_est_batch_latency(bad, [5], [])
