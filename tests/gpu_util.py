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
U_BF16 = 2.0 ** -9   # unit roundoff of bf16 (8 significand bits, round to nearest even)


def derived_gates(sigma_logit, o_absmax, v_rms, stored_rounded=False):
    """Gates for inputs that BASELINE.json's distributions do not cover (DESIGN.md section 3a derives every term).

    sigma_logit: standard deviation of the scaled scores the test's inputs produce (sm_scale * sigma_q * sigma_k *
    sqrt(D)); o_absmax: largest |o_ref|; v_rms: standard deviation of V.  Against the UNROUNDED fp64 oracle the
    path's own contract -- K' and Q' are STORED in bf16 -- perturbs every logit by
        sigma_delta = 1.5 * sqrt(2/3) * u * sigma_logit          (u = 2^-9; two operands, rel. error uniform in +-u each;
                                                                  the 1.5 covers keys whose |q.k| is above average)
    and a correct kernel then shows
        |d lse|      <= 4.5 sigma_delta                          (4.5 sigma: the largest of <= 1e5 rows)
        |d o| elem   <= half_ulp_bf16(|o|max) + 4.5 * sqrt(sigma_delta^2 + u^2/3) * v_rms   (output rounding + logit
                                                                  perturbation and bf16 P, with sum_j p_j^2 <= 1)
        mean |d o|   <= 0.8 * sqrt(sigma_delta^2 + 2 u^2/3) * v_rms
        rel-L2       <= 2.5 * sqrt(sigma_delta^2 + 2 u^2/3)
    stored_rounded=True: the reference is the oracle evaluated on q', k' rounded to bf16 (the diagnostic mode of SURVEY
    8(c)); what is left of sigma_delta is the <= 1 % of stored elements that sit one ulp from the correctly rounded
    value: a factor sqrt(0.01 * 4 / (1/3)) = 0.35.  No gate is ever tighter than BASELINE.json's 2e-2 / 2e-3 (and the
    1e-2 normalised / 1e-3 lse gates of reading T-A); on BASELINE.json's distributions (sigma_logit ~ 0.008) every
    derived term is far below them, so they apply unchanged.
    Returns (max_abs, mean_abs, rel_l2, lse_tol)."""
    sd = 1.5 * np.sqrt(2.0 / 3.0) * U_BF16 * sigma_logit * (0.35 if stored_rounded else 1.0)
    half_ulp = 2.0 ** (np.floor(np.log2(max(o_absmax, 1e-30))) - 8)
    max_abs = max(MAX_ABS, half_ulp + 4.5 * np.sqrt(sd ** 2 + U_BF16 ** 2 / 3) * v_rms)
    mean_abs = max(MEAN_ABS, 0.8 * np.sqrt(sd ** 2 + 2 * U_BF16 ** 2 / 3) * v_rms)
    rel_l2 = max(REL_L2, 2.5 * np.sqrt(sd ** 2 + 2 * U_BF16 ** 2 / 3))
    lse_tol = max(1e-3, 4.5 * sd)
    return float(max_abs), float(mean_abs), float(rel_l2), float(lse_tol)


def check_derived(o_gpu, l_gpu, ref, sigma_logit, v_rms, what="", stored_rounded=False):
    """check_out + check_lse with the gates derived_gates gives for these inputs."""
    mx, mn, rl, lt = derived_gates(sigma_logit, float(np.abs(ref["o"]).max()), v_rms, stored_rounded)
    e = check_out(o_gpu, ref["o"], what, max_abs=mx, mean_abs=mn, rel_l2=rl)
    le = check_lse(l_gpu, ref["lse"], lt, what) if l_gpu is not None else 0.0
    return e + (le,)


def oracle_session(w, i, data, rows=None, heads=None):
    """fp64 oracle of session i: re-prefill of its `new` tokens over its prefix."""
    s = w.sessions[i]
    k, v, q = (t.cpu() for t in data[i])
    P = s.prefix
    k_rot_prefix = orc.rope(k[:P], np.arange(P), w.layer.rope_base)
    return orc.oracle_cached(k_rot_prefix, orc.widen(v[:P]), q, k[P:], v[P:], P, w.layer.rope_base,
                             rows=rows, heads=heads)


def oracle_session_stored(w, i, data, rows=None, heads=None):
    """The diagnostic mode of SURVEY 8(c): the same oracle, but q' and k' are rounded to bf16 (nearest even, by torch on
    the CPU, from the ORACLE's own fp64 RoPE -- nothing comes from the CUDA path) before the scores, as the cache stores
    them.  Separates storage quantisation from kernel error."""
    s = w.sessions[i]
    k, v, q = (t.cpu() for t in data[i])
    P = s.prefix
    base = w.layer.rope_base
    k_rot = bf16_rne(orc.rope(k, np.arange(s.total), base))
    q_rot = bf16_rne(orc.rope(q, np.arange(P, s.total), base))
    return orc.attend(q_rot, k_rot, orc.widen(v), P, rows=rows, heads=heads)


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
