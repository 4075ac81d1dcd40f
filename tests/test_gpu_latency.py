"""sa_latency_table: the measured attention terms of PAPER.md Eq. 1."""
import numpy as np
import pytest
import torch

from paper_2607_00151_b200 import binding as sa

pytestmark = pytest.mark.gpu


def _mix64(x):
    m = (1 << 64) - 1
    x = (x + 0x9E3779B97F4A7C15) & m
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & m
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & m
    return x ^ (x >> 31)


def test_latency_table_small_grid():
    cfg = sa.PoolConfig(32, 8, 128, 64, 4096, 64, 16384, 500000.0)
    pool = sa.sa_kv_pool_create(cfg)
    free0 = sa.sa_kv_pool_free_pages(pool)
    p_tok, d_bat = [0, 512, 2048, 3000], [0, 1, 16]
    prefix, lo, hi, seed = 4096, 2048, 8192, 9
    ms, sums = sa.sa_latency_table(pool, p_tok, d_bat, prefix, lo, hi, seed, warmup=2, iters=5)
    assert ms.shape == (4, 3) and sums.shape == (4, 3, 2)
    assert ms[0, 0] == 0.0 and (ms.reshape(-1)[1:] > 0).all()
    # scratch sessions are gone and every page is back
    assert sa.sa_kv_pool_free_pages(pool) == free0
    assert sa.sa_kv_session_open(pool) == 0
    # the sums Eq. 1 multiplies alpha_d and alpha_p with: decode contexts from the documented counter-based draw
    ctx = [lo + _mix64((seed * 0x100000001B3 + j) & ((1 << 64) - 1)) % (hi - lo + 1) for j in range(16)]
    for b, d in enumerate(d_bat):
        assert (sums[:, b, 0] == sum(ctx[:d])).all()
    A = lambda q: q * prefix + q * (q + 1) // 2
    assert (sums[:, :, 1] == np.array([0, A(512), A(2048), A(2048) + A(952)])[:, None]).all()
    # more work never measures (much) faster: allow 30 % noise on these microsecond-scale launches
    assert ms[2, 2] > ms[0, 1] and ms[3, 2] > 0.7 * ms[2, 2] and ms[0, 2] > 0.7 * ms[0, 1]
    print("latency table (ms):\n", ms)
    with pytest.raises(sa.SAError) as e:  # more decode contexts than the pool can hold
        sa.sa_latency_table(pool, [0], [4096], prefix, 8192, 8192)
    assert e.value.status in (sa.SA_ERR_OUT_OF_PAGES, sa.SA_ERR_OUT_OF_SESSIONS)
    assert sa.sa_kv_pool_free_pages(pool) == free0
