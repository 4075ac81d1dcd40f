// sa_transfer.cu -- KV hand-over between pools ("KV transfer via NIXL"
// between prefill and decode instances, L456 PD-disaggregated serving, L424 tensor parallelism).
//
// A session's cached tokens leave a pool as a WIRE IMAGE, a dense bf16 array [2 (K', V)][Hkv][n][D]
// (K' is the rotated key exactly as stored: positions travel with the data, the receiver does not
// rotate again), and enter another pool from one.  Both directions are one HBM-bound gather /
// scatter kernel with 128-bit accesses; the far end of either may be a peer GPU's memory mapped
// into this process (NVLink P2P under unified addressing), so a prefill instance can write a
// lookahead session's rebuilt KV straight into the decode instance's staging buffer, or a decode
// instance can pull it, with no bounce through the host.  Per kv head the image is contiguous, so
// a head-sharded (tensor-parallel) receiver imports only its heads: `src_heads` / `head_begin`.
#include <cuda_bf16.h>

#include "sa_internal.h"

namespace sa {

namespace {

constexpr int kXferThreads = 256;
constexpr int kXferTok = 8;  // tokens per CTA

// EXPORT: pages -> image.  One thread per 16-byte chunk of one (token, K|V, head) row.
__global__ void __launch_bounds__(kXferThreads)
kv_export_kernel(const __nv_bfloat16 *__restrict__ k_base, const __nv_bfloat16 *__restrict__ v_base,
                 const int32_t *__restrict__ bt_row, int32_t log2_page, int64_t stride_page, int64_t stride_head,
                 int32_t Hkv, int32_t D, int32_t tok_begin, int32_t n_tok, __nv_bfloat16 *__restrict__ image) {
    __shared__ int64_t s_src[kXferTok];
    const int t0 = blockIdx.x * kXferTok;
    const int nt = min(kXferTok, n_tok - t0);
    if (threadIdx.x < nt) {
        const int pos = tok_begin + t0 + threadIdx.x;
        const int32_t page = bt_row[pos >> log2_page];
        s_src[threadIdx.x] = int64_t(page) * stride_page + int64_t(pos & ((1 << log2_page) - 1)) * D;
    }
    __syncthreads();
    // 16-byte chunks; D is 64 or 128, so chunk-in-row is a shift.  Four chunks in flight per thread: all loads, then
    // all stores (one dependent load -> store pair at a time left the kernel latency-bound at 80 % of the copy peak).
    const int lc = D == 128 ? 4 : 3;            // log2(chunks per row)
    const int rows = nt * 2 * Hkv;              // (token, K|V head) rows of this CTA
    const int total = rows << lc;
    constexpr int U = 4;
    for (int base = threadIdx.x; base < total; base += kXferThreads * U) {
        uint4 val[U];
        __nv_bfloat16 *dst[U];
#pragma unroll
        for (int i = 0; i < U; ++i) {
            const int e = base + i * kXferThreads;
            dst[i] = nullptr;
            if (e >= total) continue;
            const int row = e >> lc, c = e & ((1 << lc) - 1);
            const int tl = row / (2 * Hkv), hk = row % (2 * Hkv);   // hk in [0, 2 Hkv): K heads then V heads
            const bool is_v = hk >= Hkv;
            const int h = is_v ? hk - Hkv : hk;
            const __nv_bfloat16 *src = (is_v ? v_base : k_base) + s_src[tl] + int64_t(h) * stride_head + c * 8;
            dst[i] = image + ((int64_t(is_v) * Hkv + h) * n_tok + (t0 + tl)) * D + c * 8;
            val[i] = *reinterpret_cast<const uint4 *>(src);
        }
#pragma unroll
        for (int i = 0; i < U; ++i)
            if (dst[i]) *reinterpret_cast<uint4 *>(dst[i]) = val[i];
    }
}

// IMPORT: image -> pages of the tokens an append_prepare has just made room for.  INLINE: the request and its new page
// ids ride in the kernel parameters (no upload launch, no block-table launch; the placing thread writes the entry), as
// in rope_append_kernel.
template <bool INLINE>
__global__ void __launch_bounds__(kXferThreads)
kv_import_kernel(const __grid_constant__ InlineAppendMeta im, const ReqMeta *__restrict__ req, __nv_bfloat16 *__restrict__ k_base, __nv_bfloat16 *__restrict__ v_base,
                 int32_t *block_table, int64_t mpps, int32_t log2_page, int64_t stride_page,
                 int64_t stride_head, int32_t Hkv, int32_t D, int32_t src_heads, int32_t head_begin, int32_t n_tok,
                 const __nv_bfloat16 *__restrict__ image) {
    __shared__ int64_t s_dst[kXferTok];
    const ReqMeta r = INLINE ? im.reqs[0] : req[0];
    const int t0 = blockIdx.x * kXferTok;
    const int nt = min(kXferTok, n_tok - t0);
    if (threadIdx.x < nt) {
        const int pos = r.kv_len + t0 + threadIdx.x;
        const int32_t pi = pos >> log2_page;
        int32_t page;
        if (INLINE && pi >= r.part_begin && pi - r.part_begin < r.n_splits) {
            page = im.pages[r.item_begin + pi - r.part_begin];
            block_table[int64_t(r.sid) * mpps + pi] = page;
        } else {
            page = block_table[int64_t(r.sid) * mpps + pi];
        }
        s_dst[threadIdx.x] = int64_t(page) * stride_page + int64_t(pos & ((1 << log2_page) - 1)) * D;
    }
    __syncthreads();
    const int lc = D == 128 ? 4 : 3;
    const int rows = nt * 2 * Hkv;
    const int total = rows << lc;
    constexpr int U = 4;   // chunks in flight per thread, as in the export kernel
    for (int base = threadIdx.x; base < total; base += kXferThreads * U) {
        uint4 val[U];
        __nv_bfloat16 *dst[U];
#pragma unroll
        for (int i = 0; i < U; ++i) {
            const int e = base + i * kXferThreads;
            dst[i] = nullptr;
            if (e >= total) continue;
            const int row = e >> lc, c = e & ((1 << lc) - 1);
            const int tl = row / (2 * Hkv), hk = row % (2 * Hkv);
            const bool is_v = hk >= Hkv;
            const int h = is_v ? hk - Hkv : hk;
            const __nv_bfloat16 *src = image + ((int64_t(is_v) * src_heads + head_begin + h) * n_tok + (t0 + tl)) * D + c * 8;
            dst[i] = (is_v ? v_base : k_base) + s_dst[tl] + int64_t(h) * stride_head + c * 8;
            val[i] = *reinterpret_cast<const uint4 *>(src);
        }
#pragma unroll
        for (int i = 0; i < U; ++i)
            if (dst[i]) *reinterpret_cast<uint4 *>(dst[i]) = val[i];
    }
}

}  // namespace

}  // namespace sa

extern "C" int32_t sa_kv_wire_bytes(const sa_kv_pool *pool, int64_t n_tokens, size_t *out_bytes) {
    if (!pool || !out_bytes || n_tokens < 0) return SA_ERR_INVALID_ARG;
    *out_bytes = size_t(2) * size_t(pool->cfg.num_kv_heads) * size_t(n_tokens) * size_t(pool->cfg.head_dim) * 2;
    return SA_OK;
}

extern "C" int32_t sa_kv_session_export(sa_kv_pool *pool, int32_t sid, int64_t tok_begin, int64_t n_tokens, void *image,
                                        size_t image_bytes, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    if (!pool || sid < 0 || size_t(sid) >= pool->sessions.size() || !pool->sessions[size_t(sid)].open)
        return SA_ERR_INVALID_ARG;
    const sa::Session &s = pool->sessions[size_t(sid)];
    if (tok_begin < 0 || n_tokens < 0 || tok_begin + n_tokens > s.len) return SA_ERR_INVALID_ARG;
    size_t need = 0;
    sa_kv_wire_bytes(pool, n_tokens, &need);
    if (image_bytes < need) return SA_ERR_WORKSPACE_TOO_SMALL;
    pool->last_launches = 0;
    if (n_tokens == 0) return SA_OK;
    if (pool->host_only) return SA_ERR_CUDA;
    if (!image || (reinterpret_cast<uintptr_t>(image) & 15)) return SA_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const unsigned grid = unsigned((n_tokens + sa::kXferTok - 1) / sa::kXferTok);
    sa::kv_export_kernel<<<grid, sa::kXferThreads, 0, stream>>>(
        static_cast<const __nv_bfloat16 *>(pool->k_base), static_cast<const __nv_bfloat16 *>(pool->v_base),
        pool->block_table + int64_t(sid) * pool->max_pages_per_session, pool->log2_page, pool->stride_page,
        pool->stride_head, pool->cfg.num_kv_heads, pool->cfg.head_dim, int32_t(tok_begin), int32_t(n_tokens),
        static_cast<__nv_bfloat16 *>(image));
    ++pool->last_launches;
    return cudaGetLastError() == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}

extern "C" int32_t sa_kv_session_import(sa_kv_pool *pool, int32_t sid, int64_t n_tokens, const void *image,
                                        int32_t src_heads, int32_t head_begin, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    if (!pool || n_tokens < 0 || n_tokens > INT32_MAX) return SA_ERR_INVALID_ARG;
    if (src_heads <= 0 || head_begin < 0 || head_begin + pool->cfg.num_kv_heads > src_heads) return SA_ERR_INVALID_ARG;
    if (!pool->host_only && n_tokens > 0 && (!image || (reinterpret_cast<uintptr_t>(image) & 15))) return SA_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int32_t indptr[2] = {0, int32_t(n_tokens)};
    const sa::ReqMeta *req_dev = nullptr;
    int64_t total = 0;
    sa::InlineAppendMeta im;
    // page allocation, copy-on-write of a shared partial page, block-table update and failure behaviour are the append's
    const int32_t st = sa::append_prepare(pool, 1, &sid, indptr, image != nullptr, stream, &req_dev, &total, &im);
    if (st != SA_OK || (!req_dev && !im.used) || total == 0) return st;
    const unsigned grid = unsigned((n_tokens + sa::kXferTok - 1) / sa::kXferTok);
    if (im.used)
        sa::kv_import_kernel<true><<<grid, sa::kXferThreads, 0, stream>>>(
            im, nullptr, static_cast<__nv_bfloat16 *>(pool->k_base), static_cast<__nv_bfloat16 *>(pool->v_base), pool->block_table,
            pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head, pool->cfg.num_kv_heads,
            pool->cfg.head_dim, src_heads, head_begin, int32_t(n_tokens), static_cast<const __nv_bfloat16 *>(image));
    else
        sa::kv_import_kernel<false><<<grid, sa::kXferThreads, 0, stream>>>(
            im, req_dev, static_cast<__nv_bfloat16 *>(pool->k_base), static_cast<__nv_bfloat16 *>(pool->v_base), pool->block_table,
            pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head, pool->cfg.num_kv_heads,
            pool->cfg.head_dim, src_heads, head_begin, int32_t(n_tokens), static_cast<const __nv_bfloat16 *>(image));
    ++pool->last_launches;
    return cudaGetLastError() == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}
