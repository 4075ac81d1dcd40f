"""KV hand-over between processes: one process per GPU, `torch.distributed` for the
plumbing (NCCL over NVLink on GPUs, gloo on CPU in the tests).

PAPER.md L426: the prefill instance hands a request's KV to the decode instance ("KV transfer via
NIXL"); L424: under tensor parallelism every rank holds a slice of the kv heads.  The data path is the
library's: `sa_kv_session_export` gathers the session's pages into a wire image [2][Hkv][n][D] on the
sender, `sa_kv_session_import` scatters an image (or a head slice of it) into the receiver's pages.
This module only moves the image: a 4-int64 header (n_tokens, kv_heads in the message, head_dim,
first head), then the payload.  Because one kv head's part of the image is contiguous, a sender
serving tensor-parallel receivers sends each rank only its own heads (`send_image(..., heads=...)`).

Where sender and receiver sit in one process with peer access enabled (or share a buffer through CUDA
IPC), skip this module: pass the peer-mapped buffer as `image` to `sa_kv_session_export` and the copy
goes over NVLink inside the gather kernel itself.
"""
from __future__ import annotations

from typing import Optional, Tuple

import torch
import torch.distributed as dist


def head_shard(num_q_heads: int, num_kv_heads: int, rank: int, world: int) -> Tuple[int, int, int, int]:
    """-> (q_head_begin, q_heads, kv_head_begin, kv_heads) of `rank`: contiguous kv heads with their whole
    GQA groups, so attention needs no exchange (the all-reduce of L424 sits after the output projection)."""
    if world <= 0 or not (0 <= rank < world) or num_kv_heads % world or num_q_heads % num_kv_heads:
        raise ValueError("kv heads must divide evenly over the ranks")
    hk = num_kv_heads // world
    g = num_q_heads // num_kv_heads
    return rank * hk * g, hk * g, rank * hk, hk


def image_heads(image: torch.Tensor, head_begin: int, head_count: int) -> torch.Tensor:
    """The [2][head_count][n][D] part of an image that holds heads [head_begin, head_begin + head_count)."""
    if image.dim() != 4 or image.shape[0] != 2 or head_begin < 0 or head_begin + head_count > image.shape[1]:
        raise ValueError("head slice outside the image")
    return image[:, head_begin:head_begin + head_count]


def _wire_device(device, group=None):
    """NCCL moves device buffers over NVLink; gloo (the CPU tests, or a box without NCCL) stages through the host."""
    return torch.device("cpu") if dist.get_backend(group) == "gloo" else torch.device(device)


def send_image(image: torch.Tensor, dst: int, heads: Optional[Tuple[int, int]] = None, group=None) -> int:
    """Send `image` (or heads = (begin, count) of it) to rank `dst`; returns the payload bytes."""
    hb, hc = heads if heads is not None else (0, image.shape[1])
    wire = _wire_device(image.device, group)
    part = image_heads(image, hb, hc).contiguous().to(wire)
    header = torch.tensor([part.shape[2], hc, part.shape[3], hb], dtype=torch.int64, device=wire)
    dist.send(header, dst, group=group)
    if part.numel():
        dist.send(part.view(torch.int16), dst, group=group)  # bit pattern: every backend moves int16
    return part.numel() * part.element_size()


def recv_image(src: int, device, group=None) -> Tuple[torch.Tensor, int]:
    """-> (image [2][heads][n][D] bf16 on `device`, first head it holds)."""
    wire = _wire_device(device, group)
    header = torch.empty(4, dtype=torch.int64, device=wire)
    dist.recv(header, src, group=group)
    n, hc, d, hb = (int(x) for x in header.tolist())
    buf = torch.empty((2, hc, n, d), dtype=torch.int16, device=wire)
    if buf.numel():
        dist.recv(buf, src, group=group)
    return buf.to(device).view(torch.bfloat16), hb


def send_session(pool, sid: int, tok_begin: int, n_tokens: int, dst_ranks, group=None, stream=None) -> int:
    """Export tokens [tok_begin, tok_begin + n_tokens) of a session once and send every rank of `dst_ranks`
    its head shard (one rank: the whole image).  Returns the bytes sent."""
    from . import binding as sa
    cfg = pool.cfg
    image = torch.empty((2, cfg.num_kv_heads, n_tokens, cfg.head_dim), dtype=torch.bfloat16, device=pool.storage.device)
    sa.sa_kv_session_export(pool, sid, tok_begin, n_tokens, image, stream)
    if stream is not None:
        stream.synchronize()
    else:
        torch.cuda.current_stream(pool.storage.device).synchronize()
    sent = 0
    world = len(dst_ranks)
    for i, dst in enumerate(dst_ranks):
        _, _, hb, hc = head_shard(cfg.num_q_heads, cfg.num_kv_heads, i, world)
        sent += send_image(image, dst, (hb, hc), group)
    return sent


def recv_session(pool, sid: int, src: int, group=None, stream=None) -> int:
    """Receive an image whose head count equals this pool's and append it to session `sid`; returns n_tokens."""
    from . import binding as sa
    image, _ = recv_image(src, pool.storage.device, group)
    if image.shape[1] != pool.cfg.num_kv_heads or image.shape[3] != pool.cfg.head_dim:
        raise ValueError("image holds %d heads of dim %d, the pool %d of %d" % (image.shape[1], image.shape[3],
                                                                               pool.cfg.num_kv_heads, pool.cfg.head_dim))
    sa.sa_kv_session_import(pool, sid, image.shape[2], image, image.shape[1], 0, stream)
    if stream is not None:
        image.record_stream(stream)  # the scatter kernel reads it after this function returns
    return int(image.shape[2])
