"""fp64 CPU oracle of the re-prefill hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin numpy/ctypes front of ``sa_oracle.c`` (same directory): the arithmetic is
in the C file, written straight from the definitions; this module only moves
arrays and concatenates prefix and segment the way the cache does.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this.  Nothing here imports, reads or
links anything of ``paper_2607_00151_b200``: the two sides share no code.

Entry points:

* ``rope(x, positions, base)``                       step 1
* ``attend(q_rot, k_rot, v, P, sm_scale, ...)``      steps 2-4
* ``oracle_full(q, k, v, base, sm_scale)``           one-shot prefill of a whole
  (transformed) context: every token is a query row
* ``oracle_cached(k_rot_prefix, v_prefix, q_seg, k_seg, v_seg, P, ...)``
  re-prefill of a segment over an already rotated, stored prefix
                                                     PAPER.md L311-313, L186-187
Decode row = ``oracle_cached`` with a one-token segment
* ``wire_image(k_rot, v, head_begin, head_count)``   the KV hand-over image (N4;
  PAPER.md L426 "KV transfer", L424 tensor parallelism): a pure re-indexing of
  the stored cache, image[c][h][t][d] = (K' if c == 0 else V)[t][head_begin+h][d]

Parity pins live in tests/test_oracle_pins.py.  Absolute output values are
otherwise unpinned (the paper prints no tensor).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sa_oracle.c")
_LIB = os.path.join(_HERE, "libsa_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile sa_oracle.c with gcc (-O2, OpenMP, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.sa_oracle_num_threads.restype = ctypes.c_int32
        lib.sa_oracle_rope.restype = None
        lib.sa_oracle_rope.argtypes = [dp, ctypes.POINTER(ctypes.c_int64), ctypes.c_int64,
                                       ctypes.c_int32, ctypes.c_int32, ctypes.c_double, dp]
        lib.sa_oracle_attend.restype = None
        lib.sa_oracle_attend.argtypes = [
            dp, dp, dp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32,
            ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_int64,
            ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int32), dp, dp, dp,
            ctypes.POINTER(ctypes.c_int64)]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().sa_oracle_num_threads())


def widen(x) -> np.ndarray:
    """Exact widening of the input bits (bf16/fp32 torch tensor or ndarray) to float64."""
    if hasattr(x, "detach"):  # torch tensor, without importing torch here
        x = x.detach().cpu().double().numpy()
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def rope(x, positions, base: float) -> np.ndarray:
    """x [n, H, D] -> rotated copy; positions [n] absolute positions (step 1)."""
    x = widen(x)
    n, H, D = x.shape
    assert D % 2 == 0
    pos = np.ascontiguousarray(np.asarray(positions, dtype=np.int64))
    assert pos.shape == (n,)
    out = np.empty_like(x)
    _load().sa_oracle_rope(_dptr(x), pos.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                           n, H, D, float(base), _dptr(out))
    return out


def attend(q_rot, k_rot, v, P: int, sm_scale: Optional[float] = None, rows=None, heads=None,
           return_probs: bool = False):
    """Steps 2-4.  q_rot [N,Hq,D] at positions P..P+N-1; k_rot, v [L,Hkv,D], L >= P+N.

    rows/heads None -> all (i, h): returns o [N,Hq,D], lse [N,Hq].
    else sampled pairs:            returns o [S,D],    lse [S].
    """
    q = widen(q_rot)
    k = widen(k_rot)
    vv = widen(v)
    N, Hq, D = q.shape
    L, Hkv, Dk = k.shape
    assert Dk == D and vv.shape == k.shape and Hq % Hkv == 0 and L >= P + N and P >= 0
    if sm_scale is None:
        sm_scale = 1.0 / np.sqrt(D)
    if rows is None:
        S = N * Hq
        rp = hp = None
    else:
        rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
        heads = np.ascontiguousarray(np.asarray(heads, dtype=np.int32))
        S = rows.shape[0]
        assert heads.shape == (S,)
        assert S == 0 or (rows.min() >= 0 and rows.max() < N and heads.min() >= 0 and heads.max() < Hq)
        rp = rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))
        hp = heads.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
    o = np.zeros((S, D), dtype=np.float64)
    lse = np.zeros((S,), dtype=np.float64)
    probs = np.zeros((S, L), dtype=np.float64) if return_probs else None
    pairs = ctypes.c_int64(0)
    _load().sa_oracle_attend(_dptr(q), _dptr(k), _dptr(vv), N, L, Hq, Hkv, D, int(P),
                             float(sm_scale), S, rp, hp, _dptr(o), _dptr(lse),
                             _dptr(probs) if return_probs else None, ctypes.byref(pairs))
    if rows is None:
        o = o.reshape(N, Hq, D)
        lse = lse.reshape(N, Hq)
        if return_probs:
            probs = probs.reshape(N, Hq, L)
    res = {"o": o, "lse": lse, "pairs": int(pairs.value)}
    if return_probs:
        res["probs"] = probs
    return res


def oracle_full(q, k, v, base: float, sm_scale: Optional[float] = None, use_rope: bool = True,
                return_probs: bool = False):
    """One-shot prefill of a whole context of L tokens: q [L,Hq,D], k,v [L,Hkv,D] (raw, pre-RoPE)."""
    q = widen(q)
    k = widen(k)
    L = k.shape[0]
    assert q.shape[0] == L
    pos = np.arange(L, dtype=np.int64)
    q_rot = rope(q, pos, base) if use_rope else q
    k_rot = rope(k, pos, base) if use_rope else k
    res = attend(q_rot, k_rot, v, 0, sm_scale, return_probs=return_probs)
    res["k_rot"] = k_rot
    res["q_rot"] = q_rot
    return res


def oracle_cached(k_rot_prefix, v_prefix, q_seg, k_seg, v_seg, P: int, base: float,
                  sm_scale: Optional[float] = None, rows=None, heads=None):
    """Re-prefill of a segment of N raw tokens at absolute positions P..P+N-1 over a stored
    prefix (k_rot_prefix [P,Hkv,D] already rotated, v_prefix [P,Hkv,D])."""
    kp = widen(k_rot_prefix)
    vp = widen(v_prefix)
    assert kp.shape[0] == P and vp.shape[0] == P
    q_seg = widen(q_seg)
    k_seg = widen(k_seg)
    v_seg = widen(v_seg)
    N = q_seg.shape[0]
    pos = np.arange(P, P + N, dtype=np.int64)
    q_rot = rope(q_seg, pos, base)
    k_rot_seg = rope(k_seg, pos, base)
    k_all = np.concatenate([kp, k_rot_seg], axis=0)
    v_all = np.concatenate([vp, v_seg], axis=0)
    res = attend(q_rot, k_all, v_all, P, sm_scale, rows=rows, heads=heads)
    res["k_rot_seg"] = k_rot_seg
    res["q_rot"] = q_rot
    return res


def wire_image(k_rot, v, head_begin: int = 0, head_count: Optional[int] = None) -> np.ndarray:
    """Hand-over image of a cached token range (N4; PAPER.md L426 / L424).

    k_rot, v: [n, Hkv, D], the rotated keys and the values as the cache stores them.  Returns
    image[2][head_count][n][D] with image[0][h][t][d] = k_rot[t][head_begin + h][d] and
    image[1][h][t][d] = v[t][head_begin + h][d]: no arithmetic, only the index order (written as
    explicit loops over c and h so that it can be checked against that sentence by eye)."""
    k_rot = np.asarray(k_rot)
    v = np.asarray(v)
    n, hkv, d = k_rot.shape
    if head_count is None:
        head_count = hkv - head_begin
    img = np.empty((2, head_count, n, d), dtype=k_rot.dtype)
    for h in range(head_count):
        for t in range(n):
            img[0, h, t, :] = k_rot[t, head_begin + h, :]
            img[1, h, t, :] = v[t, head_begin + h, :]
    return img
