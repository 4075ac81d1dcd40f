"""Helpers of the GPU parity tests: run a workload through the C-ABI (harness) and through the
fp64 oracle on the same bits, and compare with the gates of BASELINE.json / DESIGN.md."""
import numpy as np
import torch

from oracle import oracle as orc
from paper_2607_00151_b200 import binding as sa
from paper_2607_00151_b200.harness import Runner, make_pool
from paper_2607_00151_b200.workloads import gen_session

# BASELINE.json north_star gates + the binding relative gates of SURVEY 8(c) T-A
MAX_ABS, MEAN_ABS, REL_L2 = 2e-2, 2e-3, 1e-2


def oracle_session(w, i, data, rows=None, heads=None):
    """fp64 oracle of session i: re-prefill of its `new` tokens over its prefix."""
    s = w.sessions[i]
    k, v, q = (t.cpu() for t in data[i])
    P = s.prefix
    k_rot_prefix = orc.rope(k[:P], np.arange(P), w.layer.rope_base)
    return orc.oracle_cached(k_rot_prefix, orc.widen(v[:P]), q, k[P:], v[P:], P, w.layer.rope_base,
                             rows=rows, heads=heads)


def check_out(o_gpu, o_ref, what="", max_abs=MAX_ABS, mean_abs=MEAN_ABS, rel_l2=REL_L2):
    g = o_gpu.detach().double().cpu().numpy() if hasattr(o_gpu, "detach") else np.asarray(o_gpu, dtype=np.float64)
    assert np.isfinite(g).all(), "%s: non-finite output" % what
    err = np.abs(g - o_ref)
    rl2 = np.linalg.norm(g - o_ref) / max(np.linalg.norm(o_ref), 1e-300)
    assert err.max() <= max_abs, "%s: max-abs %.3e" % (what, err.max())
    assert err.mean() <= mean_abs, "%s: mean-abs %.3e" % (what, err.mean())
    assert rl2 <= rel_l2, "%s: normalised L2 error %.3e" % (what, rl2)
    return err.max(), err.mean(), rl2


def check_lse(l_gpu, l_ref, tol, what=""):
    g = l_gpu.detach().double().cpu().numpy() if hasattr(l_gpu, "detach") else np.asarray(l_gpu, dtype=np.float64)
    assert np.isfinite(g).all(), "%s: non-finite lse" % what
    e = np.abs(g - l_ref).max()
    assert e <= tol, "%s: lse error %.3e > %.1e" % (what, e, tol)
    return e


def bf16_rne(x64):
    """Round fp64 -> bf16 (nearest even), returned as float64."""
    return torch.from_numpy(np.asarray(x64, dtype=np.float64)).to(torch.bfloat16).double().numpy()


def check_rope_k(k_gpu, k_ref, what=""):
    """RoPE'd K gate with reading T-B: |err| <= 1e-2 wherever a perfectly rounded bf16 could meet
    it; within 1 bf16 ulp of RNE(k_ref) on the (counted) remainder."""
    g = k_gpu.detach().double().cpu().numpy()
    rne = bf16_rne(k_ref)
    attainable = np.abs(rne - k_ref) <= 1e-2
    err = np.abs(g - k_ref)
    assert err[attainable].max() <= 1e-2, "%s: K' error %.3e" % (what, err[attainable].max())
    rest = ~attainable
    if rest.any():
        ulp = 2.0 ** (np.floor(np.log2(np.abs(rne[rest]))) - 7)
        assert (np.abs(g[rest] - rne[rest]) <= ulp).all(), "%s: K' off by more than 1 ulp where 1e-2 is unattainable" % what
    return err.max(), int(rest.sum())


def run_workload(w, page_order="random", sentinel=None, scale=None, data=None, device=0, fill=True, num_pages=None):
    pool = make_pool(w, device, page_order, sentinel, num_pages=num_pages)
    if data is None:
        data = {i: gen_session(w, i, "cuda:%d" % device, scale) for i in range(len(w.sessions))}
    r = Runner(w, pool, data, device)
    if fill:
        r.fill_prefixes()
    r.step()
    torch.cuda.synchronize()
    return pool, r, data
