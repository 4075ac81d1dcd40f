"""ctypes binding of libsmoothagent.so: the same names as include/smoothagent.h, argument
marshalling only.  Every step of the path runs in the library's CUDA kernels; torch is used for
device memory and streams.  There is no fallback: if the library is missing or a call fails, an
exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsmoothagent.so")

SA_OK = 0
SA_ERR_INVALID_ARG = -1
SA_ERR_OUT_OF_PAGES = -2
SA_ERR_UNSUPPORTED = -3
SA_ERR_CUDA = -4
SA_ERR_WORKSPACE_TOO_SMALL = -5
SA_ERR_OUT_OF_SESSIONS = -6


class SAError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s failed: %s (%d)" % (where, sa_status_string(status), status))


class sa_kv_pool_config(ctypes.Structure):
    _fields_ = [
        ("num_q_heads", ctypes.c_int32),
        ("num_kv_heads", ctypes.c_int32),
        ("head_dim", ctypes.c_int32),
        ("page_size", ctypes.c_int32),
        ("num_pages", ctypes.c_int64),
        ("max_sessions", ctypes.c_int32),
        ("device", ctypes.c_int32),
        ("max_session_tokens", ctypes.c_int64),
        ("rope_base", ctypes.c_double),
    ]


class sa_kv_layout(ctypes.Structure):
    _fields_ = [
        ("k_base", ctypes.c_void_p),
        ("v_base", ctypes.c_void_p),
        ("stride_page", ctypes.c_int64),
        ("stride_head", ctypes.c_int64),
        ("stride_slot", ctypes.c_int64),
    ]


SA_GEMM_TABLE_MAX = 64


class sa_latency_model(ctypes.Structure):
    _fields_ = [
        ("c0_ms", ctypes.c_double),
        ("alpha_d_ms", ctypes.c_double),
        ("alpha_p_ms", ctypes.c_double),
        ("n_gemm", ctypes.c_int32),
        ("reserved", ctypes.c_int32),
        ("gemm_m", ctypes.c_double * SA_GEMM_TABLE_MAX),
        ("gemm_ms", ctypes.c_double * SA_GEMM_TABLE_MAX),
    ]


class sa_chunk(ctypes.Structure):
    _fields_ = [("q", ctypes.c_int64), ("prefix", ctypes.c_int64)]


class sa_lc_request(ctypes.Structure):
    _fields_ = [("t_arrival_ms", ctypes.c_double), ("slo_ttft_ms", ctypes.c_double), ("q", ctypes.c_int64),
                ("prefix", ctypes.c_int64)]


class sa_layer_weights(ctypes.Structure):
    _fields_ = [("hidden", ctypes.c_int32), ("ffn", ctypes.c_int32), ("rms_eps", ctypes.c_float), ("reserved", ctypes.c_int32),
                ("norm1", ctypes.c_void_p), ("w_qkv", ctypes.c_void_p), ("w_o", ctypes.c_void_p), ("norm2", ctypes.c_void_p),
                ("w_gate", ctypes.c_void_p), ("w_up", ctypes.c_void_p), ("w_down", ctypes.c_void_p)]


_i32p = ctypes.POINTER(ctypes.c_int32)
_i64p = ctypes.POINTER(ctypes.c_int64)
_f32p = ctypes.POINTER(ctypes.c_float)
_f64p = ctypes.POINTER(ctypes.c_double)
_vp = ctypes.c_void_p
_modelp = ctypes.POINTER(sa_latency_model)
_chunkp = ctypes.POINTER(sa_chunk)

# name -> (restype, argtypes); also the list the symbol test checks against the header
PROTOTYPES = {
    "sa_status_string": (ctypes.c_char_p, [ctypes.c_int32]),
    "sa_kv_pool_storage_bytes": (ctypes.c_int32, [ctypes.POINTER(sa_kv_pool_config), ctypes.POINTER(ctypes.c_size_t)]),
    "sa_kv_pool_create": (ctypes.c_int32, [ctypes.POINTER(sa_kv_pool_config), _vp, ctypes.c_size_t, _i32p, ctypes.POINTER(_vp)]),
    "sa_kv_pool_destroy": (ctypes.c_int32, [_vp]),
    "sa_kv_pool_layout": (ctypes.c_int32, [_vp, ctypes.POINTER(sa_kv_layout)]),
    "sa_kv_pool_free_pages": (ctypes.c_int32, [_vp, _i64p]),
    "sa_kv_session_open": (ctypes.c_int32, [_vp, _i32p]),
    "sa_kv_session_close": (ctypes.c_int32, [_vp, ctypes.c_int32]),
    "sa_kv_session_truncate": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int64]),
    "sa_kv_session_query": (ctypes.c_int32, [_vp, ctypes.c_int32, _i64p, _i32p, _i32p]),
    "sa_kv_session_fork": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int64, _i32p, _vp]),
    "sa_kv_session_commit": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int32, _vp]),
    "sa_kv_page_refcount": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p]),
    "sa_rope_kv_append": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i32p, _vp, _vp, _vp, _vp]),
    "sa_mixed_attention_workspace_bytes": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i32p, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_mixed_attention": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i32p, _vp, _vp, _vp, ctypes.c_float, _vp, ctypes.c_size_t, _vp]),
    "sa_mixed_attention_plan": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i32p, _i64p]),
    "sa_mixed_attention_schedule": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i32p, _i32p, ctypes.c_int32, _i64p]),
    "sa_last_launch_count": (ctypes.c_int32, [_vp, _i32p]),
    "sa_latency_table_workspace_bytes": (ctypes.c_int32, [_vp, _i32p, ctypes.c_int32, _i32p, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64,
                                                          ctypes.c_int64, ctypes.c_uint64, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_latency_table": (ctypes.c_int32, [_vp, _i32p, ctypes.c_int32, _i32p, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64,
                                          ctypes.c_int64, ctypes.c_uint64, ctypes.c_int32, ctypes.c_int32, _f32p, _i64p, _vp,
                                          ctypes.c_size_t, _vp]),
    "sa_latency_fit": (ctypes.c_int32, [_f32p, _i64p, ctypes.c_int32, ctypes.c_int32, _modelp, _f64p]),
    "sa_est_batch_latency": (ctypes.c_int32, [_modelp, _i64p, ctypes.c_int32, _chunkp, ctypes.c_int32, _f64p]),
    "sa_schedule_hybrid": (ctypes.c_int32, [_modelp, _i64p, ctypes.c_int32, _chunkp, ctypes.c_int32, _chunkp, ctypes.c_int32,
                                            ctypes.c_double, _i32p, _f64p]),
    "sa_schedule_prefill_slack": (ctypes.c_int32, [_modelp, ctypes.POINTER(sa_lc_request), ctypes.c_int32, ctypes.c_double,
                                                   _chunkp, ctypes.c_int32, _chunkp, ctypes.c_int32, _i32p, _f64p, _f64p]),
    "sa_dynamic_chunk": (ctypes.c_int32, [_modelp, _i64p, ctypes.c_int32, _chunkp, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64,
                                          ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.POINTER(ctypes.c_int64)]),
    "sa_linear": (ctypes.c_int32, [_vp, _vp, _vp, _vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, _vp]),
    "sa_swiglu": (ctypes.c_int32, [_vp, _vp, _vp, _vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, _vp]),
    "sa_rmsnorm": (ctypes.c_int32, [_vp, _vp, ctypes.c_float, _vp, ctypes.c_int64, ctypes.c_int32, _vp]),
    "sa_qkv_rope_append_workspace_bytes": (ctypes.c_int32, [_vp, ctypes.c_int64, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_qkv_rope_append": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i32p, _vp, _vp, ctypes.c_int32, _vp, _vp,
                                            ctypes.c_size_t, _vp]),
    "sa_layer_workspace_bytes": (ctypes.c_int32, [_vp, ctypes.POINTER(sa_layer_weights), ctypes.c_int32, _i32p, _i32p,
                                                  ctypes.POINTER(ctypes.c_size_t)]),
    "sa_layer_forward": (ctypes.c_int32, [_vp, ctypes.POINTER(sa_layer_weights), ctypes.c_int32, _i32p, _i32p, _vp, _vp,
                                          ctypes.c_float, _vp, ctypes.c_size_t, _vp]),
    "sa_gemm_table_workspace_bytes": (ctypes.c_int32, [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _i32p,
                                                       ctypes.c_int32, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_gemm_table": (ctypes.c_int32, [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _i32p,
                                       ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _f32p, _vp, ctypes.c_size_t, _vp]),
    "sa_linear_workspace_bytes": (ctypes.c_int32, [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_linear_ws": (ctypes.c_int32, [_vp, _vp, _vp, _vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, _vp, ctypes.c_size_t, _vp]),
    "sa_linear_noalloc": (ctypes.c_int32, [_vp, _vp, _vp, _vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, _vp]),
    "sa_swiglu_workspace_bytes": (ctypes.c_int32, [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_swiglu_ws": (ctypes.c_int32, [_vp, _vp, _vp, _vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, _vp, ctypes.c_size_t, _vp]),
    "sa_kv_wire_bytes": (ctypes.c_int32, [_vp, ctypes.c_int64, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_kv_session_export": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64, _vp, ctypes.c_size_t, _vp]),
    "sa_kv_session_import": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int64, _vp, ctypes.c_int32, ctypes.c_int32, _vp]),
    "sa_kv_sessions_export": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i64p, _i64p, ctypes.POINTER(ctypes.c_void_p),
                                               ctypes.POINTER(ctypes.c_size_t), _vp]),
    "sa_kv_sessions_import": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p, _i64p, ctypes.POINTER(ctypes.c_void_p), ctypes.c_int32,
                                               ctypes.c_int32, _vp]),
    "sa_decode_step_device_bytes": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int64, ctypes.POINTER(ctypes.c_size_t)]),
    "sa_decode_step_create": (ctypes.c_int32, [_vp, ctypes.c_int32, ctypes.c_int64, _vp, ctypes.c_size_t, ctypes.POINTER(_vp)]),
    "sa_decode_step_destroy": (ctypes.c_int32, [_vp]),
    "sa_decode_step_prepare": (ctypes.c_int32, [_vp, ctypes.c_int32, _i32p]),
    "sa_decode_step_cancel": (ctypes.c_int32, [_vp]),
    "sa_decode_step_enqueue": (ctypes.c_int32, [_vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float, _vp]),
    "sa_decode_step_stats": (ctypes.c_int32, [_vp, _i64p]),
}

_lib = None


def load_library() -> ctypes.CDLL:
    """Load the in-tree library; fail loudly if it has not been built (no fallback path exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                "%s is missing: build it with `python -m paper_2607_00151_b200.build` "
                "(or __graft_entry__.build()); this package has no CPU or PyTorch fallback" % LIB_PATH)
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in PROTOTYPES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(status: int, where: str):
    if status != SA_OK:
        raise SAError(status, where)


def _i32(a: Sequence[int]):
    """-> (int32 array the caller keeps alive, something ctypes passes as const int32_t*).  On the per-call path:
    a ctypes array over the ndarray's buffer costs a third of ndarray.ctypes.data_as (which builds a helper object)."""
    if type(a) is np.ndarray and a.dtype == np.int32 and a.flags.c_contiguous:
        arr = a
    else:
        arr = np.ascontiguousarray(np.asarray(a, dtype=np.int32))
    if arr.size and arr.flags.writeable:
        return arr, (ctypes.c_int32 * arr.size).from_buffer(arr)
    return arr, arr.ctypes.data_as(_i32p)


def _ptr(t) -> Optional[int]:
    """Device (or host) pointer of a torch tensor / raw int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    assert t.is_contiguous()
    return t.data_ptr()


def _stream_ptr(stream, pool=None) -> Optional[int]:
    """None = torch's current stream ON THE POOL'S DEVICE (the library runs every call on that device, whatever device is
    current in the calling thread)."""
    if stream is None:
        import torch
        return torch.cuda.current_stream(pool.cfg.device if pool is not None else None).cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def sa_status_string(status: int) -> str:
    return load_library().sa_status_string(int(status)).decode()


@dataclass
class PoolConfig:
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    num_pages: int
    max_sessions: int
    max_session_tokens: int
    rope_base: float
    device: int = 0

    def to_c(self) -> sa_kv_pool_config:
        return sa_kv_pool_config(self.num_q_heads, self.num_kv_heads, self.head_dim, self.page_size, self.num_pages,
                                 self.max_sessions, self.device, self.max_session_tokens, self.rope_base)


def sa_kv_pool_storage_bytes(cfg: PoolConfig) -> int:
    out = ctypes.c_size_t(0)
    c = cfg.to_c()
    _check(load_library().sa_kv_pool_storage_bytes(ctypes.byref(c), ctypes.byref(out)), "sa_kv_pool_storage_bytes")
    return int(out.value)


class Pool:
    """Handle of an sa_kv_pool plus the torch tensor that owns its device storage."""

    def __init__(self, handle: int, cfg: PoolConfig, storage):
        self.handle = handle
        self.cfg = cfg
        self.storage = storage

    def __del__(self):
        try:
            if self.handle:
                sa_kv_pool_destroy(self)
        except Exception:
            pass


def sa_kv_pool_create(cfg: PoolConfig, storage=None, free_page_order=None, host_only: bool = False) -> Pool:
    """storage: a uint8 CUDA tensor of >= sa_kv_pool_storage_bytes(cfg) bytes (allocated here with
    torch.empty if None); host_only=True creates the metadata-only pool (no device needed)."""
    lib = load_library()
    c = cfg.to_c()
    nbytes = sa_kv_pool_storage_bytes(cfg)
    if host_only:
        storage, sptr = None, None
    else:
        import torch
        if storage is None:
            storage = torch.empty(nbytes, dtype=torch.uint8, device="cuda:%d" % cfg.device)
        assert storage.is_cuda and storage.numel() * storage.element_size() >= nbytes
        sptr = storage.data_ptr()
    order_keep, order_ptr = (None, None)
    if free_page_order is not None:
        order_keep, order_ptr = _i32(free_page_order)
        assert order_keep.shape == (cfg.num_pages,)
    out = _vp()
    _check(lib.sa_kv_pool_create(ctypes.byref(c), sptr, nbytes if not host_only else 0, order_ptr, ctypes.byref(out)),
           "sa_kv_pool_create")
    return Pool(out.value, cfg, storage)


def sa_kv_pool_destroy(pool: Pool) -> None:
    h, pool.handle = pool.handle, None
    if h:
        _check(load_library().sa_kv_pool_destroy(h), "sa_kv_pool_destroy")


def sa_kv_pool_layout(pool: Pool) -> sa_kv_layout:
    out = sa_kv_layout()
    _check(load_library().sa_kv_pool_layout(pool.handle, ctypes.byref(out)), "sa_kv_pool_layout")
    return out


def sa_kv_pool_free_pages(pool: Pool) -> int:
    out = ctypes.c_int64(0)
    _check(load_library().sa_kv_pool_free_pages(pool.handle, ctypes.byref(out)), "sa_kv_pool_free_pages")
    return int(out.value)


def sa_kv_session_open(pool: Pool) -> int:
    out = ctypes.c_int32(-1)
    _check(load_library().sa_kv_session_open(pool.handle, ctypes.byref(out)), "sa_kv_session_open")
    return int(out.value)


def sa_kv_session_close(pool: Pool, sid: int) -> None:
    _check(load_library().sa_kv_session_close(pool.handle, sid), "sa_kv_session_close")


def sa_kv_session_truncate(pool: Pool, sid: int, new_len: int) -> None:
    _check(load_library().sa_kv_session_truncate(pool.handle, sid, new_len), "sa_kv_session_truncate")


def sa_kv_session_fork(pool: Pool, src_sid: int, prefix_len: int, stream=None) -> int:
    out = ctypes.c_int32(-1)
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_kv_session_fork(pool.handle, src_sid, prefix_len, ctypes.byref(out), sp), "sa_kv_session_fork")
    return int(out.value)


def sa_kv_session_commit(pool: Pool, main_sid: int, lookahead_sid: int, stream=None) -> None:
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_kv_session_commit(pool.handle, main_sid, lookahead_sid, sp), "sa_kv_session_commit")


def sa_kv_page_refcount(pool: Pool, page: int) -> int:
    out = ctypes.c_int32(0)
    _check(load_library().sa_kv_page_refcount(pool.handle, page, ctypes.byref(out)), "sa_kv_page_refcount")
    return int(out.value)


def sa_kv_session_query(pool: Pool, sid: int):
    """-> (len, [page ids])"""
    lib = load_library()
    ln = ctypes.c_int64(0)
    n = ctypes.c_int32(0)
    _check(lib.sa_kv_session_query(pool.handle, sid, ctypes.byref(ln), None, ctypes.byref(n)), "sa_kv_session_query")
    pages = np.zeros(max(int(n.value), 1), dtype=np.int32)
    cap = ctypes.c_int32(int(n.value))
    _check(lib.sa_kv_session_query(pool.handle, sid, None, pages.ctypes.data_as(_i32p), ctypes.byref(cap)), "sa_kv_session_query")
    return int(ln.value), pages[: int(n.value)].tolist()


def sa_rope_kv_append(pool: Pool, sids, qo_indptr, k, v, q_inout=None, stream=None) -> None:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    assert i_keep.shape[0] == s_keep.shape[0] + 1
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_rope_kv_append(pool.handle, s_keep.shape[0], s_ptr, i_ptr, _ptr(k), _ptr(v), _ptr(q_inout), sp),
           "sa_rope_kv_append")


def sa_mixed_attention_workspace_bytes(pool: Pool, sids, qo_indptr) -> int:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    out = ctypes.c_size_t(0)
    _check(load_library().sa_mixed_attention_workspace_bytes(pool.handle, s_keep.shape[0], s_ptr, i_ptr, ctypes.byref(out)),
           "sa_mixed_attention_workspace_bytes")
    return int(out.value)


def sa_mixed_attention(pool: Pool, sids, qo_indptr, q, out, lse=None, sm_scale: float = 0.0, workspace=None, stream=None) -> None:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    assert i_keep.shape[0] == s_keep.shape[0] + 1
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_mixed_attention(pool.handle, s_keep.shape[0], s_ptr, i_ptr, _ptr(q), _ptr(out), _ptr(lse),
                                             float(sm_scale), _ptr(workspace), ws_bytes, sp), "sa_mixed_attention")


def sa_mixed_attention_plan(pool: Pool, sids, qo_indptr) -> dict:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    st = np.zeros(8, dtype=np.int64)
    _check(load_library().sa_mixed_attention_plan(pool.handle, s_keep.shape[0], s_ptr, i_ptr, st.ctypes.data_as(_i64p)),
           "sa_mixed_attention_plan")
    keys = ["decode_requests", "prefill_requests", "decode_ctas", "prefill_ctas", "partial_rows", "sum_decode_kv",
            "sum_prefill_A", "tcgen05"]
    return dict(zip(keys, (int(x) for x in st)))


def sa_mixed_attention_schedule(pool: Pool, sids, qo_indptr):
    """-> (parts int32 [n_parts, 8] = (cta, request, kv head, tile, u0, u1, n_kv, slot), summary dict)"""
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    lib = load_library()
    sm = np.zeros(6, dtype=np.int64)
    _check(lib.sa_mixed_attention_schedule(pool.handle, s_keep.shape[0], s_ptr, i_ptr, None, 0, sm.ctypes.data_as(_i64p)),
           "sa_mixed_attention_schedule")
    parts = np.zeros((int(sm[1]), 8), dtype=np.int32)
    _check(lib.sa_mixed_attention_schedule(pool.handle, s_keep.shape[0], s_ptr, i_ptr, parts.ctypes.data_as(_i32p),
                                           parts.shape[0], sm.ctypes.data_as(_i64p)), "sa_mixed_attention_schedule")
    keys = ["ctas", "parts", "split_items", "slots", "total_units", "makespan"]
    return parts, dict(zip(keys, (int(x) for x in sm)))


def sa_last_launch_count(pool: Pool) -> int:
    out = ctypes.c_int32(0)
    _check(load_library().sa_last_launch_count(pool.handle, ctypes.byref(out)), "sa_last_launch_count")
    return int(out.value)


def sa_latency_table_workspace_bytes(pool: Pool, prefill_tokens, decode_batch, prefill_prefix_len: int, decode_ctx_lo: int,
                                     decode_ctx_hi: int, seed: int = 0) -> int:
    p_keep, p_ptr = _i32(prefill_tokens)
    d_keep, d_ptr = _i32(decode_batch)
    out = ctypes.c_size_t(0)
    _check(load_library().sa_latency_table_workspace_bytes(pool.handle, p_ptr, p_keep.shape[0], d_ptr, d_keep.shape[0],
                                                           prefill_prefix_len, decode_ctx_lo, decode_ctx_hi, seed, ctypes.byref(out)),
           "sa_latency_table_workspace_bytes")
    return int(out.value)


def sa_latency_table(pool: Pool, prefill_tokens, decode_batch, prefill_prefix_len: int, decode_ctx_lo: int,
                     decode_ctx_hi: int, seed: int = 0, warmup: int = 3, iters: int = 10, stream=None, workspace=None):
    """-> (ms [n_p, n_d] float32, sums [n_p, n_d, 2] int64 = (sum L_j, sum A_j)).
    workspace: device uint8 tensor of >= sa_latency_table_workspace_bytes(...) bytes; None = one is taken from torch here."""
    p_keep, p_ptr = _i32(prefill_tokens)
    d_keep, d_ptr = _i32(decode_batch)
    ms = np.zeros((p_keep.shape[0], d_keep.shape[0]), dtype=np.float32)
    sums = np.zeros((p_keep.shape[0], d_keep.shape[0], 2), dtype=np.int64)
    if workspace is None and pool.storage is not None:
        import torch
        workspace = torch.empty(sa_latency_table_workspace_bytes(pool, prefill_tokens, decode_batch, prefill_prefix_len,
                                                                 decode_ctx_lo, decode_ctx_hi, seed), dtype=torch.uint8,
                                device=pool.storage.device)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(load_library().sa_latency_table(pool.handle, p_ptr, p_keep.shape[0], d_ptr, d_keep.shape[0], prefill_prefix_len,
                                           decode_ctx_lo, decode_ctx_hi, seed, warmup, iters, ms.ctypes.data_as(_f32p),
                                           sums.ctypes.data_as(_i64p), _ptr(workspace), ws_bytes,
                                           None if pool.storage is None else _stream_ptr(stream, pool)), "sa_latency_table")
    return ms, sums


# ---------------------------------------------------------------- scheduler core (host only)
@dataclass
class LatencyModel:
    """Eq. 1 of PAPER.md (L349-353): c0 + T_GEMM(M) + alpha_d * sum L_j + alpha_p * sum A_j, in ms."""
    c0_ms: float = 0.0
    alpha_d_ms: float = 0.0
    alpha_p_ms: float = 0.0
    gemm: Sequence = ()      # [(M, ms), ...] strictly increasing in M; empty: T_GEMM = 0

    def to_c(self) -> sa_latency_model:
        m = sa_latency_model()
        m.c0_ms, m.alpha_d_ms, m.alpha_p_ms = self.c0_ms, self.alpha_d_ms, self.alpha_p_ms
        assert len(self.gemm) <= SA_GEMM_TABLE_MAX
        m.n_gemm = len(self.gemm)
        for i, (x, y) in enumerate(self.gemm):
            m.gemm_m[i], m.gemm_ms[i] = float(x), float(y)
        return m


def _i64(a):
    arr = np.ascontiguousarray(np.asarray(a, dtype=np.int64).reshape(-1))
    return arr, arr.ctypes.data_as(_i64p)


def _chunks(cs):
    arr = (sa_chunk * max(len(cs), 1))()
    for i, (q, p) in enumerate(cs):
        arr[i].q, arr[i].prefix = int(q), int(p)
    return arr


def sa_latency_fit(ms, sum_kv, with_intercept: bool = True):
    """-> (LatencyModel, max relative error of the fit); ms and sum_kv as returned by sa_latency_table."""
    y = np.ascontiguousarray(np.asarray(ms, dtype=np.float32).reshape(-1))
    s_keep, s_ptr = _i64(sum_kv)
    assert s_keep.shape[0] == 2 * y.shape[0]
    m = sa_latency_model()
    err = ctypes.c_double(0.0)
    _check(load_library().sa_latency_fit(y.ctypes.data_as(_f32p), s_ptr, y.shape[0], int(with_intercept), ctypes.byref(m),
                                         ctypes.byref(err)), "sa_latency_fit")
    return LatencyModel(m.c0_ms, m.alpha_d_ms, m.alpha_p_ms, ()), float(err.value)


def sa_est_batch_latency(model: LatencyModel, decode_L, chunks) -> float:
    d_keep, d_ptr = _i64(decode_L)
    out = ctypes.c_double(0.0)
    cm = model.to_c()
    _check(load_library().sa_est_batch_latency(ctypes.byref(cm), d_ptr, d_keep.shape[0], _chunks(chunks), len(chunks),
                                               ctypes.byref(out)), "sa_est_batch_latency")
    return float(out.value)


def sa_schedule_hybrid(model: LatencyModel, decode_L, lc, be, delta_ms: float):
    """Algorithm 2 -> (admitted decode, LC chunks, BE chunks, estimate of the admitted batch in ms)"""
    d_keep, d_ptr = _i64(decode_L)
    adm = (ctypes.c_int32 * 3)()
    est = ctypes.c_double(0.0)
    cm = model.to_c()
    _check(load_library().sa_schedule_hybrid(ctypes.byref(cm), d_ptr, d_keep.shape[0], _chunks(lc), len(lc), _chunks(be), len(be),
                                             float(delta_ms), adm, ctypes.byref(est)), "sa_schedule_hybrid")
    return int(adm[0]), int(adm[1]), int(adm[2]), float(est.value)


def sa_schedule_prefill_slack(model: LatencyModel, lc_queue, t_now_ms: float, lc_chunks, be):
    """Algorithm 1; lc_queue: [(t_arrival_ms, slo_ttft_ms, q, prefix), ...] -> (admitted BE chunks, t_budget, estimate)"""
    qarr = (sa_lc_request * max(len(lc_queue), 1))()
    for i, (ta, slo, q, p) in enumerate(lc_queue):
        qarr[i].t_arrival_ms, qarr[i].slo_ttft_ms, qarr[i].q, qarr[i].prefix = float(ta), float(slo), int(q), int(p)
    n = ctypes.c_int32(0)
    budget, est = ctypes.c_double(0.0), ctypes.c_double(0.0)
    cm = model.to_c()
    _check(load_library().sa_schedule_prefill_slack(ctypes.byref(cm), qarr, len(lc_queue), float(t_now_ms), _chunks(lc_chunks),
                                                    len(lc_chunks), _chunks(be), len(be), ctypes.byref(n), ctypes.byref(budget),
                                                    ctypes.byref(est)), "sa_schedule_prefill_slack")
    return int(n.value), float(budget.value), float(est.value)


def sa_dynamic_chunk(model: LatencyModel, decode_L, chunks, prefix: int, remaining: int, max_chunk: int, granularity: int,
                     budget_ms: float) -> int:
    d_keep, d_ptr = _i64(decode_L)
    out = ctypes.c_int64(0)
    cm = model.to_c()
    _check(load_library().sa_dynamic_chunk(ctypes.byref(cm), d_ptr, d_keep.shape[0], _chunks(chunks), len(chunks), int(prefix),
                                           int(remaining), int(max_chunk), int(granularity), float(budget_ms), ctypes.byref(out)),
           "sa_dynamic_chunk")
    return int(out.value)


# ---------------------------------------------------------------- KV hand-over between pools (N4)
def sa_kv_wire_bytes(pool: Pool, n_tokens: int) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().sa_kv_wire_bytes(pool.handle, n_tokens, ctypes.byref(out)), "sa_kv_wire_bytes")
    return int(out.value)


def sa_kv_session_export(pool: Pool, sid: int, tok_begin: int, n_tokens: int, image, stream=None) -> None:
    """image: device bf16 tensor with >= 2*Hkv*n_tokens*D elements (local or peer-mapped)."""
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_kv_session_export(pool.handle, sid, tok_begin, n_tokens, _ptr(image), _nbytes(image), sp),
           "sa_kv_session_export")


def sa_kv_session_import(pool: Pool, sid: int, n_tokens: int, image, src_heads: int, head_begin: int = 0, stream=None) -> None:
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_kv_session_import(pool.handle, sid, n_tokens, _ptr(image), src_heads, head_begin, sp),
           "sa_kv_session_import")




def sa_kv_sessions_export(pool: Pool, sids, tok_begin, n_tokens, images, stream=None) -> None:
    """Many session ranges -> their wire images in one call (one kernel launch).  images: one device tensor per range."""
    s_keep, s_ptr = _i32(sids)
    b_keep, b_ptr = _i64(tok_begin)
    n_keep, n_ptr = _i64(n_tokens)
    n = s_keep.shape[0]
    assert b_keep.shape[0] == n and n_keep.shape[0] == n and len(images) == n
    ptrs = (ctypes.c_void_p * max(n, 1))(*[_ptr(im) for im in images])
    sizes = (ctypes.c_size_t * max(n, 1))(*[0 if im is None else im.numel() * im.element_size() for im in images])
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_kv_sessions_export(pool.handle, n, s_ptr, b_ptr, n_ptr, ptrs, sizes, sp), "sa_kv_sessions_export")


def sa_kv_sessions_import(pool: Pool, sids, n_tokens, images, src_heads: int, head_begin: int = 0, stream=None) -> None:
    """Many sessions grow from their wire images in one call (one kernel launch; page allocation all-or-nothing)."""
    s_keep, s_ptr = _i32(sids)
    n_keep, n_ptr = _i64(n_tokens)
    n = s_keep.shape[0]
    assert n_keep.shape[0] == n and len(images) == n
    ptrs = (ctypes.c_void_p * max(n, 1))(*[_ptr(im) for im in images])
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_kv_sessions_import(pool.handle, n, s_ptr, n_ptr, ptrs, src_heads, head_begin, sp), "sa_kv_sessions_import")

# ---------------------------------------------------------------- capturable decode step
class DecodeStep:
    """Handle of an sa_decode_step plus the torch tensor that owns its device memory."""

    def __init__(self, handle: int, pool: Pool, mem, max_requests: int, max_kv_tokens: int):
        self.handle = handle
        self.pool = pool
        self.mem = mem
        self.max_requests = max_requests
        self.max_kv_tokens = max_kv_tokens

    def __del__(self):
        try:
            if self.handle:
                sa_decode_step_destroy(self)
        except Exception:
            pass


def sa_decode_step_device_bytes(pool: Pool, max_requests: int, max_kv_tokens: int) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().sa_decode_step_device_bytes(pool.handle, max_requests, max_kv_tokens, ctypes.byref(out)),
           "sa_decode_step_device_bytes")
    return int(out.value)


def sa_decode_step_create(pool: Pool, max_requests: int, max_kv_tokens: int, mem=None) -> DecodeStep:
    """mem: a uint8 CUDA tensor of >= sa_decode_step_device_bytes(...) bytes (allocated here if None; None stays None
    for a host-only pool)."""
    nbytes = sa_decode_step_device_bytes(pool, max_requests, max_kv_tokens)
    if pool.storage is not None and mem is None:
        import torch
        mem = torch.empty(nbytes, dtype=torch.uint8, device="cuda:%d" % pool.cfg.device)
    out = _vp()
    _check(load_library().sa_decode_step_create(pool.handle, max_requests, max_kv_tokens, _ptr(mem), _nbytes(mem), ctypes.byref(out)),
           "sa_decode_step_create")
    return DecodeStep(out.value, pool, mem, max_requests, max_kv_tokens)


def sa_decode_step_destroy(step: DecodeStep) -> None:
    h, step.handle = step.handle, None
    if h:
        _check(load_library().sa_decode_step_destroy(h), "sa_decode_step_destroy")


def sa_decode_step_prepare(step: DecodeStep, sids) -> None:
    """Host half of one decode iteration: every session grows by one token, the step's metadata is rewritten."""
    keep, ptr = _i32(sids)
    _check(load_library().sa_decode_step_prepare(step.handle, keep.shape[0], ptr), "sa_decode_step_prepare")


def sa_decode_step_cancel(step: DecodeStep) -> None:
    """Undo the step's last prepare (one that will not be executed): lengths and pages as before it, the step empty."""
    _check(load_library().sa_decode_step_cancel(step.handle), "sa_decode_step_cancel")


def sa_decode_step_enqueue(step: DecodeStep, k, v, q_inout, out, lse=None, sm_scale: float = 0.0, stream=None) -> None:
    """Device half (two launches, capturable): RoPE + placement of the new tokens, split-KV attention of the rows."""
    _check(load_library().sa_decode_step_enqueue(step.handle, _ptr(k), _ptr(v), _ptr(q_inout), _ptr(out), _ptr(lse),
                                                 float(sm_scale), _stream_ptr(stream, step.pool)), "sa_decode_step_enqueue")


def sa_decode_step_stats(step: DecodeStep) -> dict:
    out = np.zeros(6, dtype=np.int64)
    _check(load_library().sa_decode_step_stats(step.handle, out.ctypes.data_as(_i64p)), "sa_decode_step_stats")
    return {"requests": int(out[0]), "items": int(out[1]), "grid_ctas": int(out[2]), "launches": int(out[3]),
            "max_part_rows": int(out[4]), "capacity": int(out[5])}


# ---------------------------------------------------------------- dense operators of the layer (N3)
def _nbytes(t) -> int:
    return 0 if t is None else t.numel() * t.element_size()


def sa_linear(x, w, y, residual=None, stream=None) -> None:
    """y[M, N] = x[M, K] w[N, K]^T (+ residual)."""
    M, K = x.shape
    N = w.shape[0]
    assert w.shape[1] == K and tuple(y.shape) == (M, N)
    _check(load_library().sa_linear(_ptr(x), _ptr(w), _ptr(residual), _ptr(y), M, N, K, _stream_ptr(stream)), "sa_linear")


def sa_swiglu(x, w_gate, w_up, act, stream=None) -> None:
    M, K = x.shape
    F = w_gate.shape[0]
    assert w_gate.shape == w_up.shape and w_gate.shape[1] == K and tuple(act.shape) == (M, F)
    _check(load_library().sa_swiglu(_ptr(x), _ptr(w_gate), _ptr(w_up), _ptr(act), M, F, K, _stream_ptr(stream)), "sa_swiglu")


def sa_linear_workspace_bytes(M: int, N: int, K: int) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().sa_linear_workspace_bytes(M, N, K, ctypes.byref(out)), "sa_linear_workspace_bytes")
    return int(out.value)


def sa_linear_ws(x, w, y, workspace, residual=None, stream=None) -> None:
    """sa_linear with a split-K scratch (small M)."""
    M, K = x.shape
    N = w.shape[0]
    assert w.shape[1] == K and tuple(y.shape) == (M, N)
    _check(load_library().sa_linear_ws(_ptr(x), _ptr(w), _ptr(residual), _ptr(y), M, N, K, _ptr(workspace), _nbytes(workspace),
                                       _stream_ptr(stream)), "sa_linear_ws")


SA_LINEAR_NOALLOC_SCRATCH_BYTES = 160 * 128 * 256 * 4 + 512


def sa_linear_noalloc(x, w, y, residual=None, stream=None) -> None:
    """sa_linear_ws without the workspace argument, for code that cannot get device memory of its own (it runs inside
    someone else's fixed memory plan, or next to a KV pool that has taken all of HBM, or must not stall the device with
    cudaMalloc / cudaFree).  The split-K partials go to a 20 MiB array built into the library; nothing is allocated.
    Decode-sized shapes only (those sa_linear_workspace_bytes gives a non-zero size for), otherwise SAError with
    SA_ERR_UNSUPPORTED.  Bit-equal to sa_linear_ws.  Calls share the array: keep them on one stream, and make the first
    call on a device before any stream capture."""
    M, K = x.shape
    N = w.shape[0]
    assert w.shape[1] == K and tuple(y.shape) == (M, N)
    _check(load_library().sa_linear_noalloc(_ptr(x), _ptr(w), _ptr(residual), _ptr(y), M, N, K, _stream_ptr(stream)),
           "sa_linear_noalloc")


def sa_swiglu_workspace_bytes(M: int, F: int, K: int) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().sa_swiglu_workspace_bytes(M, F, K, ctypes.byref(out)), "sa_swiglu_workspace_bytes")
    return int(out.value)


def sa_swiglu_ws(x, w_gate, w_up, act, workspace, stream=None) -> None:
    M, K = x.shape
    F = w_gate.shape[0]
    assert w_gate.shape == w_up.shape and w_gate.shape[1] == K and tuple(act.shape) == (M, F)
    _check(load_library().sa_swiglu_ws(_ptr(x), _ptr(w_gate), _ptr(w_up), _ptr(act), M, F, K, _ptr(workspace), _nbytes(workspace),
                                       _stream_ptr(stream)), "sa_swiglu_ws")


def sa_rmsnorm(x, w, eps: float, y, stream=None) -> None:
    M, H = x.shape
    assert w.shape[0] == H and y.shape == x.shape
    _check(load_library().sa_rmsnorm(_ptr(x), _ptr(w), float(eps), _ptr(y), M, H, _stream_ptr(stream)), "sa_rmsnorm")


def sa_qkv_rope_append_workspace_bytes(pool: Pool, total_tokens: int) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().sa_qkv_rope_append_workspace_bytes(pool.handle, total_tokens, ctypes.byref(out)),
           "sa_qkv_rope_append_workspace_bytes")
    return int(out.value)


def sa_qkv_rope_append(pool: Pool, sids, qo_indptr, h, w_qkv, q_out, workspace, stream=None) -> None:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    assert i_keep.shape[0] == s_keep.shape[0] + 1
    hidden = w_qkv.shape[1]
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_qkv_rope_append(pool.handle, s_keep.shape[0], s_ptr, i_ptr, _ptr(h), _ptr(w_qkv), hidden,
                                             _ptr(q_out), _ptr(workspace), _nbytes(workspace), sp), "sa_qkv_rope_append")


@dataclass
class LayerWeights:
    """Device bf16 tensors of one decoder layer, weights [out_features, in_features]."""
    norm1: object
    w_qkv: object
    w_o: object
    norm2: object
    w_gate: object
    w_up: object
    w_down: object
    rms_eps: float = 1e-5

    def to_c(self) -> sa_layer_weights:
        return sa_layer_weights(self.w_qkv.shape[1], self.w_gate.shape[0], self.rms_eps, 0, _ptr(self.norm1), _ptr(self.w_qkv),
                                _ptr(self.w_o), _ptr(self.norm2), _ptr(self.w_gate), _ptr(self.w_up), _ptr(self.w_down))


def sa_layer_workspace_bytes(pool: Pool, layer: LayerWeights, sids, qo_indptr) -> int:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    c = layer.to_c()
    out = ctypes.c_size_t(0)
    _check(load_library().sa_layer_workspace_bytes(pool.handle, ctypes.byref(c), s_keep.shape[0], s_ptr, i_ptr, ctypes.byref(out)),
           "sa_layer_workspace_bytes")
    return int(out.value)


def sa_layer_forward(pool: Pool, layer: LayerWeights, sids, qo_indptr, x, y, workspace, sm_scale: float = 0.0, stream=None) -> None:
    s_keep, s_ptr = _i32(sids)
    i_keep, i_ptr = _i32(qo_indptr)
    assert i_keep.shape[0] == s_keep.shape[0] + 1
    c = layer.to_c()
    sp = None if pool.storage is None else _stream_ptr(stream, pool)
    _check(load_library().sa_layer_forward(pool.handle, ctypes.byref(c), s_keep.shape[0], s_ptr, i_ptr, _ptr(x), _ptr(y),
                                           float(sm_scale), _ptr(workspace), _nbytes(workspace), sp), "sa_layer_forward")


def sa_gemm_table_workspace_bytes(hidden: int, ffn: int, num_q_heads: int, num_kv_heads: int, head_dim: int, m_list) -> int:
    m_keep, m_ptr = _i32(m_list)
    out = ctypes.c_size_t(0)
    _check(load_library().sa_gemm_table_workspace_bytes(hidden, ffn, num_q_heads, num_kv_heads, head_dim, m_ptr, m_keep.shape[0],
                                                        ctypes.byref(out)), "sa_gemm_table_workspace_bytes")
    return int(out.value)


def sa_gemm_table(hidden: int, ffn: int, num_q_heads: int, num_kv_heads: int, head_dim: int, m_list, warmup: int = 3,
                  iters: int = 10, stream=None, workspace=None):
    """-> ms float32 [len(m_list)]: T_GEMM(M) of PAPER.md L299-303 measured on this library's kernels.
    workspace: device uint8 tensor of >= sa_gemm_table_workspace_bytes(...) bytes; None = one is taken from torch here."""
    m_keep, m_ptr = _i32(m_list)
    ms = np.zeros(m_keep.shape[0], dtype=np.float32)
    if workspace is None:
        import torch
        workspace = torch.empty(sa_gemm_table_workspace_bytes(hidden, ffn, num_q_heads, num_kv_heads, head_dim, m_list),
                                dtype=torch.uint8, device="cuda")
    _check(load_library().sa_gemm_table(hidden, ffn, num_q_heads, num_kv_heads, head_dim, m_ptr, m_keep.shape[0], warmup, iters,
                                        ms.ctypes.data_as(_f32p), _ptr(workspace), workspace.numel() * workspace.element_size(),
                                        _stream_ptr(stream)), "sa_gemm_table")
    return ms
