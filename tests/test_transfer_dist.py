"""The N > 1 plumbing of the KV hand-over on CPU: world_size-3 gloo,
rank 0 plays the prefill instance and sends ranks 1 and 2 (two tensor-parallel decode ranks) their head
shards of a wire image; header, payload bits and head arithmetic are checked on the receivers against an
image they regenerate from the same seed.  (The gather / scatter kernels themselves are covered by
tests/test_gpu_transfer.py; this is the host protocol only.)"""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_2607_00151_b200 import transfer
dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
Hq, Hkv, D, n = 32, 8, 128, 77
g = torch.Generator(); g.manual_seed(123)
image = torch.randn((2, Hkv, n, D), generator=g).to(torch.bfloat16)   # every rank can rebuild the sender's image
out = {"rank": rank}
if rank == 0:
    sent = 0
    for i, dst in enumerate((1, 2)):
        _, _, hb, hc = transfer.head_shard(Hq, Hkv, i, 2)
        sent += transfer.send_image(image, dst, (hb, hc))
    sent += transfer.send_image(image[:, :, :0], 1)                    # an empty range is a header only
    out["sent"] = sent
else:
    part, hb = transfer.recv_image(0, torch.device("cpu"))
    qb, qh, kb, kh = transfer.head_shard(Hq, Hkv, rank - 1, 2)
    out.update(shape=list(part.shape), hb=hb, kb=kb, kh=kh, qb=qb, qh=qh,
               equal=bool(torch.equal(part.view(torch.int16), image[:, kb:kb + kh].contiguous().view(torch.int16))))
    if rank == 1:
        empty, hb0 = transfer.recv_image(0, torch.device("cpu"))
        out["empty"] = list(empty.shape)
print(json.dumps(out))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_gloo_world3_head_sharded_handover():
    port = _free_port()
    procs = []
    for rank in range(3):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="3", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    res = {r["rank"]: r for r in (json.loads(o.strip().splitlines()[-1]) for o, _ in outs)}
    assert res[0]["sent"] == 2 * 8 * 77 * 128 * 2          # both shards together are the whole image, once
    for r in (1, 2):
        assert res[r]["equal"] and res[r]["shape"] == [2, 4, 77, 128]
        assert (res[r]["hb"], res[r]["kb"], res[r]["kh"]) == (4 * (r - 1), 4 * (r - 1), 4)
        assert (res[r]["qb"], res[r]["qh"]) == (16 * (r - 1), 16)
    assert res[1]["empty"] == [2, 8, 0, 128]


def test_head_shard_arithmetic():
    from paper_2607_00151_b200 import transfer
    assert transfer.head_shard(64, 8, 3, 4) == (48, 16, 6, 2)
    assert transfer.head_shard(8, 2, 0, 1) == (0, 8, 0, 2)
    covered = []
    for r in range(8):
        qb, qh, kb, kh = transfer.head_shard(32, 8, r, 8)
        covered += list(range(qb, qb + qh))
        assert qh == 4 * kh and qb == 4 * kb          # whole GQA groups travel with their kv head
    assert covered == list(range(32))
    for bad in ((32, 8, 0, 3), (32, 8, 2, 2), (30, 8, 0, 2), (32, 8, -1, 2)):
        with pytest.raises(ValueError):
            transfer.head_shard(*bad)


GPU_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_2607_00151_b200 import binding as sa, transfer
from paper_2607_00151_b200.harness import gather_kv
dist.init_process_group(backend="gloo")      # host-staged transport: both ranks share the one GPU of the box
rank = dist.get_rank()
dev = torch.device("cuda:0")
Hq, Hkv, D, B, n = 32, 8, 128, 64, 300
def pool_of(hq, hkv, seed):
    cfg = sa.PoolConfig(hq, hkv, D, B, 12, 4, 1024, 500000.0, 0)
    st = torch.zeros(sa.sa_kv_pool_storage_bytes(cfg), dtype=torch.uint8, device=dev)
    return sa.sa_kv_pool_create(cfg, st, np.random.default_rng(seed).permutation(12).astype(np.int32))
g = torch.Generator(device=dev); g.manual_seed(9)
k = (torch.randn((n, Hkv, D), generator=g, device=dev) * 0.09).to(torch.bfloat16)
v = (torch.randn((n, Hkv, D), generator=g, device=dev) * 0.09).to(torch.bfloat16)
full = pool_of(Hq, Hkv, 1); s = sa.sa_kv_session_open(full)
sa.sa_rope_kv_append(full, [s], [0, n], k, v, None)      # every rank can rebuild the sender's session
out = {"rank": rank}
if rank == 0:
    out["sent"] = transfer.send_session(full, s, 0, 200, [1]) + transfer.send_session(full, s, 200, 100, [1])
else:
    mine = pool_of(Hq, Hkv, 2); s2 = sa.sa_kv_session_open(mine)
    got = transfer.recv_session(mine, s2, 0) + transfer.recv_session(mine, s2, 0)
    torch.cuda.synchronize()
    ln, pg = sa.sa_kv_session_query(mine, s2)
    k2, v2 = gather_kv(mine, pg, ln)
    k1, v1 = gather_kv(full, sa.sa_kv_session_query(full, s)[1], n)
    out.update(got=got, len=ln, equal=bool(torch.equal(k1.view(torch.int16), k2.view(torch.int16)) and
                                           torch.equal(v1.view(torch.int16), v2.view(torch.int16))))
print(json.dumps(out))
dist.destroy_process_group()
"""


@pytest.mark.gpu
def test_send_session_recv_session_two_processes_one_gpu():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", GPU_WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-3000:]
    res = {r["rank"]: r for r in (json.loads(o.strip().splitlines()[-1]) for o, _ in outs)}
    assert res[0]["sent"] == 2 * 8 * 300 * 128 * 2
    assert res[1]["got"] == 300 and res[1]["len"] == 300 and res[1]["equal"]
