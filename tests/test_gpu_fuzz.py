"""Seeded boundary fuzz of the whole path (append + mixed attention) against the fp64 oracle: ragged batches whose
query lengths and prefixes sit on and around every boundary the kernels have -- the decode / prefill class switch
(q * G <= 16), the 128-row Q tile and 256-row item, the 128-key KV tile, the 1024-key decode split, page ends (16 /
64), empty prefixes and one-token sessions -- over every supported (head_dim, page, G) combination, with NaN in every
slot the sessions do not own.  Every output element is compared (the sizes are small enough for the full oracle)."""
import os

import numpy as np
import pytest
import torch

from paper_2607_00151_b200.workloads import Layer, SessionSpec, Workload

from gpu_util import check_derived, oracle_session, run_workload

pytestmark = pytest.mark.gpu

Q_EDGES = [1, 2, 3, 4, 5, 8, 9, 15, 16, 17, 31, 32, 33, 63, 64, 65, 127, 128, 129, 255, 256, 257, 300, 511, 513]
P_EDGES = [0, 1, 15, 16, 17, 63, 64, 65, 127, 128, 129, 255, 256, 1023, 1024, 1025, 2047, 2048, 2049, 3000]
BASE_SEED = int(os.environ.get("SA_FUZZ_SEED", "9000"))   # other seeds: SA_FUZZ_SEED=... pytest tests/test_gpu_fuzz.py -m gpu
SHAPES = [(128, 64, 4), (128, 64, 8), (128, 16, 1), (128, 16, 16), (64, 16, 4), (64, 64, 2), (64, 64, 8), (128, 64, 2)]


@pytest.mark.parametrize("case", range(40))
def test_boundary_fuzz_vs_oracle(case):
    rng = np.random.default_rng(BASE_SEED + case)
    D, B, G = SHAPES[case % len(SHAPES)]
    Hkv = int(rng.choice([1, 2, 4]))
    Hq = Hkv * G
    n = int(rng.integers(3, 8))
    sessions = []
    for _ in range(n):
        q = int(rng.choice(Q_EDGES))
        p = int(rng.choice(P_EDGES))
        sessions.append(SessionSpec(p, q))
    if case % 4 == 0:
        sessions.append(SessionSpec(0, 1))   # a one-token session: kv_len 1, the smallest legal request
    used = sum((s.total + B - 1) // B for s in sessions)
    w = Workload("fuzz%d" % case, Layer(Hq, Hkv, D, B, 10000.0 if case % 2 else 500000.0), sessions,
                 num_pages=used * 2 + 8, value_scale=D ** -0.25, seed=BASE_SEED + case)
    pool, r, data = run_workload(w, sentinel=0x7FC1)
    outs = r.outputs()
    for i, s in enumerate(sessions):
        ref = oracle_session(w, i, data)
        what = "fuzz %d (D %d B %d G %d Hkv %d) session %d (prefix %d, new %d)" % (case, D, B, G, Hkv, i, s.prefix, s.new)
        check_derived(outs[i][0], outs[i][1], ref, D ** -0.5, D ** -0.25, what)   # q, k, v ~ N(0, D^-1/2): scores of std D^-1/2
