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
#include <string.h>

#include <algorithm>
#include <vector>

#include "sa_internal.h"

namespace sa {

namespace {

constexpr int kXferThreads = 256;
constexpr int kXferTok = 8;  // tokens per CTA

// One session range of a hand-over call.  The tokens of all ranges of a call form one concatenated index space
// [0, total); t_start is where this range begins in it.
struct XferReq {
    int32_t sid, tok_begin, n_tok, t_start;
    uint64_t image;   // device address of this range's wire image
    uint64_t pad;
};
struct InlineXfer {
    XferReq reqs[kInlineReqs];
};
struct InlineImages {
    uint64_t image[kInlineReqs];
};

// last request whose first token index is <= t (empty requests share their start with the next one and never match last)
template <typename R, typename F>
__device__ __forceinline__ int find_by_start(const R *reqs, int n, int t, F start_of) {
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (start_of(reqs[mid]) <= t) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// The copy loop both directions share: CTA-local token tl has its page row at element offset s_page[tl] (head 0, K and V
// alike) and its image row for (K|V, head h) at s_img[tl] + ((is_v * img_heads + img_head0 + h) * s_ntok[tl]) * D.
// One thread per 16-byte chunk; D is 64 or 128, so chunk-in-row is a shift.  Four chunks in flight per thread: all loads,
// then all stores (one dependent load -> store pair at a time left the kernels latency-bound at 80 % of the copy peak).
template <bool TO_IMAGE>
__device__ __forceinline__ void copy_rows(__nv_bfloat16 *k_base, __nv_bfloat16 *v_base, const int64_t *s_page,
                                          __nv_bfloat16 *const *s_img, const int *s_ntok, int nt, int64_t stride_head,
                                          int Hkv, int D, int img_heads, int img_head0) {
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
            __nv_bfloat16 *pg = (is_v ? v_base : k_base) + s_page[tl] + int64_t(h) * stride_head + c * 8;
            __nv_bfloat16 *im = s_img[tl] + (int64_t(is_v) * img_heads + img_head0 + h) * s_ntok[tl] * D + c * 8;
            dst[i] = TO_IMAGE ? im : pg;
            val[i] = *reinterpret_cast<const uint4 *>(TO_IMAGE ? pg : im);
        }
#pragma unroll
        for (int i = 0; i < U; ++i)
            if (dst[i]) *reinterpret_cast<uint4 *>(dst[i]) = val[i];
    }
}

// EXPORT: pages -> images, any number of session ranges in one launch.  INLINE: the ranges ride in the kernel parameters.
template <bool INLINE>
__global__ void __launch_bounds__(kXferThreads)
kv_export_kernel(const __grid_constant__ InlineXfer ix, const XferReq *__restrict__ reqs_slab, int32_t n_req, int32_t total_tok,
                 __nv_bfloat16 *k_base, __nv_bfloat16 *v_base, const int32_t *__restrict__ block_table, int64_t mpps,
                 int32_t log2_page, int64_t stride_page, int64_t stride_head, int32_t Hkv, int32_t D) {
    __shared__ int64_t s_page[kXferTok];
    __shared__ __nv_bfloat16 *s_img[kXferTok];
    __shared__ int s_ntok[kXferTok];
    const XferReq *reqs = INLINE ? ix.reqs : reqs_slab;
    const int t0 = blockIdx.x * kXferTok;
    const int nt = min(kXferTok, total_tok - t0);
    if (threadIdx.x < nt) {
        const int t = t0 + threadIdx.x;
        const XferReq r = reqs[find_by_start(reqs, n_req, t, [](const XferReq &x) { return x.t_start; })];
        const int tl = t - r.t_start;
        const int pos = r.tok_begin + tl;
        const int32_t page = block_table[int64_t(r.sid) * mpps + (pos >> log2_page)];
        s_page[threadIdx.x] = int64_t(page) * stride_page + int64_t(pos & ((1 << log2_page) - 1)) * D;
        s_img[threadIdx.x] = reinterpret_cast<__nv_bfloat16 *>(r.image) + int64_t(tl) * D;
        s_ntok[threadIdx.x] = r.n_tok;
    }
    __syncthreads();
    copy_rows<true>(k_base, v_base, s_page, s_img, s_ntok, nt, stride_head, Hkv, D, Hkv, 0);
}

// IMPORT: images -> pages of the tokens an append_prepare has just made room for (requests as the append's: kv_len = the
// position of the request's first new token, q_start = its first token in the call's concatenated index space).  INLINE:
// the requests, their new page ids and the image addresses ride in the kernel parameters (no upload launch, no block-table
// launch; the placing thread writes the entry), as in rope_append_kernel.
template <bool INLINE>
__global__ void __launch_bounds__(kXferThreads)
kv_import_kernel(const __grid_constant__ InlineAppendMeta im, const __grid_constant__ InlineImages ii, const ReqMeta *__restrict__ reqs_slab,
                 const uint64_t *__restrict__ images_slab, int32_t n_req_slab, int32_t total_tok, __nv_bfloat16 *k_base,
                 __nv_bfloat16 *v_base, int32_t *block_table, int64_t mpps, int32_t log2_page, int64_t stride_page,
                 int64_t stride_head, int32_t Hkv, int32_t D, int32_t src_heads, int32_t head_begin) {
    __shared__ int64_t s_page[kXferTok];
    __shared__ __nv_bfloat16 *s_img[kXferTok];
    __shared__ int s_ntok[kXferTok];
    const ReqMeta *reqs = INLINE ? im.reqs : reqs_slab;
    const int n_req = INLINE ? im.n_req : n_req_slab;
    const int t0 = blockIdx.x * kXferTok;
    const int nt = min(kXferTok, total_tok - t0);
    if (threadIdx.x < nt) {
        const int t = t0 + threadIdx.x;
        const int ri = find_by_start(reqs, n_req, t, [](const ReqMeta &x) { return x.q_start; });
        const ReqMeta r = reqs[ri];
        const int tl = t - r.q_start;
        const int pos = r.kv_len + tl;
        const int32_t pi = pos >> log2_page;
        int32_t page;
        if (INLINE && pi >= r.part_begin && pi - r.part_begin < r.n_splits) {
            page = im.pages[r.item_begin + pi - r.part_begin];
            block_table[int64_t(r.sid) * mpps + pi] = page;
        } else {
            page = block_table[int64_t(r.sid) * mpps + pi];
        }
        s_page[threadIdx.x] = int64_t(page) * stride_page + int64_t(pos & ((1 << log2_page) - 1)) * D;
        s_img[threadIdx.x] = reinterpret_cast<__nv_bfloat16 *>(INLINE ? ii.image[ri] : images_slab[ri]) + int64_t(tl) * D;
        s_ntok[threadIdx.x] = r.q_len;
    }
    __syncthreads();
    copy_rows<false>(k_base, v_base, s_page, s_img, s_ntok, nt, stride_head, Hkv, D, src_heads, head_begin);
}

}  // namespace

}  // namespace sa

extern "C" int32_t sa_kv_wire_bytes(const sa_kv_pool *pool, int64_t n_tokens, size_t *out_bytes) {
    if (!pool || !out_bytes || n_tokens < 0) return SA_ERR_INVALID_ARG;
    *out_bytes = size_t(2) * size_t(pool->cfg.num_kv_heads) * size_t(n_tokens) * size_t(pool->cfg.head_dim) * 2;
    return SA_OK;
}

extern "C" int32_t sa_kv_sessions_export(sa_kv_pool *pool, int32_t n_ranges, const int32_t *sids, const int64_t *tok_begin,
                                         const int64_t *n_tokens, void *const *images, const size_t *image_bytes,
                                         void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    if (!pool || n_ranges < 0) return SA_ERR_INVALID_ARG;
    if (n_ranges > 0 && (!sids || !tok_begin || !n_tokens || !images || !image_bytes)) return SA_ERR_INVALID_ARG;
    if (n_ranges > int64_t(pool->cfg.max_sessions) * 4) return SA_ERR_INVALID_ARG;   // the documented limit of a call
    std::vector<sa::XferReq> reqs(static_cast<size_t>(n_ranges));
    int64_t total = 0;
    for (int i = 0; i < n_ranges; ++i) {
        const int32_t sid = sids[i];
        if (sid < 0 || size_t(sid) >= pool->sessions.size() || !pool->sessions[size_t(sid)].open) return SA_ERR_INVALID_ARG;
        const sa::Session &s = pool->sessions[size_t(sid)];
        if (tok_begin[i] < 0 || n_tokens[i] < 0 || tok_begin[i] + n_tokens[i] > s.len) return SA_ERR_INVALID_ARG;
        size_t need = 0;
        sa_kv_wire_bytes(pool, n_tokens[i], &need);
        if (image_bytes[i] < need) return SA_ERR_WORKSPACE_TOO_SMALL;
        if (n_tokens[i] > 0 && !pool->host_only && (!images[i] || (reinterpret_cast<uintptr_t>(images[i]) & 15))) return SA_ERR_INVALID_ARG;
        sa::XferReq &r = reqs[size_t(i)];
        r.sid = sid;
        r.tok_begin = int32_t(tok_begin[i]);
        r.n_tok = int32_t(n_tokens[i]);
        r.t_start = int32_t(total);
        r.image = reinterpret_cast<uint64_t>(images[i]);
        r.pad = 0;
        total += n_tokens[i];
    }
    if (total > INT32_MAX) return SA_ERR_UNSUPPORTED;
    pool->last_launches = 0;
    if (total == 0) return SA_OK;
    if (pool->host_only) return SA_ERR_CUDA;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const unsigned grid = unsigned((total + sa::kXferTok - 1) / sa::kXferTok);
    auto kb = static_cast<__nv_bfloat16 *>(pool->k_base);
    auto vb = static_cast<__nv_bfloat16 *>(pool->v_base);
    if (n_ranges <= sa::kInlineReqs) {
        sa::InlineXfer ix;
        memcpy(ix.reqs, reqs.data(), sizeof(sa::XferReq) * size_t(n_ranges));
        sa::kv_export_kernel<true><<<grid, sa::kXferThreads, 0, stream>>>(
            ix, nullptr, n_ranges, int32_t(total), kb, vb, pool->block_table, pool->max_pages_per_session, pool->log2_page,
            pool->stride_page, pool->stride_head, pool->cfg.num_kv_heads, pool->cfg.head_dim);
    } else {
        // The ranges go through the pinned metadata slab, as many per launch as one slab holds (a slab is sized for a
        // call's requests and page ids, not for 4 x max_sessions ranges: a pool with many sessions and few pages has
        // slabs smaller than that).  Ranges are independent, so a longer list is cut into several launches, each over
        // its own slab of the ring with its token offsets rebased; the result does not depend on where the cuts fall.
        static const sa::InlineXfer none{};
        const size_t per_slab = pool->meta_slab_bytes / sizeof(sa::XferReq);
        if (per_slab == 0) return SA_ERR_UNSUPPORTED;
        for (size_t i0 = 0; i0 < size_t(n_ranges); i0 += per_slab) {
            const size_t n = std::min(per_slab, size_t(n_ranges) - i0);
            const int32_t t_base = reqs[i0].t_start;
            const int64_t t_end = i0 + n < size_t(n_ranges) ? int64_t(reqs[i0 + n].t_start) : total;
            if (t_end == t_base) continue;  // nothing but empty ranges
            char *mh = nullptr, *md = nullptr;
            const int32_t st = sa::acquire_meta(pool, sizeof(sa::XferReq) * n, &mh, &md);
            if (st != SA_OK) return st;
            sa::XferReq *dst = reinterpret_cast<sa::XferReq *>(mh);
            for (size_t i = 0; i < n; ++i) {
                dst[i] = reqs[i0 + i];
                dst[i].t_start -= t_base;
            }
            if (sa::commit_meta(pool, sizeof(sa::XferReq) * n, stream) != SA_OK) return SA_ERR_CUDA;  // counts its launch
            const int32_t sub_total = int32_t(t_end - t_base);
            sa::kv_export_kernel<false><<<unsigned((sub_total + sa::kXferTok - 1) / sa::kXferTok), sa::kXferThreads, 0, stream>>>(
                none, reinterpret_cast<const sa::XferReq *>(md), int32_t(n), sub_total, kb, vb, pool->block_table,
                pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head, pool->cfg.num_kv_heads,
                pool->cfg.head_dim);
            ++pool->last_launches;
            if (cudaGetLastError() != cudaSuccess) return SA_ERR_CUDA;
        }
        return SA_OK;
    }
    ++pool->last_launches;
    return cudaGetLastError() == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}

extern "C" int32_t sa_kv_session_export(sa_kv_pool *pool, int32_t sid, int64_t tok_begin, int64_t n_tokens, void *image,
                                        size_t image_bytes, void *stream_) {
    return sa_kv_sessions_export(pool, 1, &sid, &tok_begin, &n_tokens, &image, &image_bytes, stream_);
}

extern "C" int32_t sa_kv_sessions_import(sa_kv_pool *pool, int32_t n_sessions, const int32_t *sids, const int64_t *n_tokens,
                                         const void *const *images, int32_t src_heads, int32_t head_begin, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    if (!pool || n_sessions < 0) return SA_ERR_INVALID_ARG;
    if (n_sessions > 0 && (!sids || !n_tokens || (!images && !pool->host_only))) return SA_ERR_INVALID_ARG;
    if (src_heads <= 0 || head_begin < 0 || head_begin + pool->cfg.num_kv_heads > src_heads) return SA_ERR_INVALID_ARG;
    std::vector<int32_t> indptr(size_t(n_sessions) + 1, 0);
    bool have_data = true;
    for (int i = 0; i < n_sessions; ++i) {
        if (n_tokens[i] < 0 || int64_t(indptr[size_t(i)]) + n_tokens[i] > INT32_MAX) return SA_ERR_INVALID_ARG;
        indptr[size_t(i) + 1] = indptr[size_t(i)] + int32_t(n_tokens[i]);
        if (!pool->host_only && n_tokens[i] > 0) {
            if (!images[i] || (reinterpret_cast<uintptr_t>(images[i]) & 15)) return SA_ERR_INVALID_ARG;
        }
        if (n_tokens[i] > 0 && (!images || !images[i])) have_data = false;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const sa::ReqMeta *req_dev = nullptr;
    int64_t total = 0;
    sa::InlineAppendMeta im;
    // page allocation, copy-on-write of a shared partial page, block-table update and failure behaviour are the append's
    const int32_t st = sa::append_prepare(pool, n_sessions, sids, indptr.data(), have_data, stream, &req_dev, &total, &im);
    if (st != SA_OK || (!req_dev && !im.used) || total == 0) return st;
    const unsigned grid = unsigned((total + sa::kXferTok - 1) / sa::kXferTok);
    auto kb = static_cast<__nv_bfloat16 *>(pool->k_base);
    auto vb = static_cast<__nv_bfloat16 *>(pool->v_base);
    if (im.used) {
        sa::InlineImages ii;
        for (int i = 0; i < n_sessions; ++i) ii.image[i] = reinterpret_cast<uint64_t>(images[i]);
        sa::kv_import_kernel<true><<<grid, sa::kXferThreads, 0, stream>>>(
            im, ii, nullptr, nullptr, 0, int32_t(total), kb, vb, pool->block_table, pool->max_pages_per_session, pool->log2_page,
            pool->stride_page, pool->stride_head, pool->cfg.num_kv_heads, pool->cfg.head_dim, src_heads, head_begin);
    } else {
        // the image addresses follow the requests through a slab of their own
        char *mh = nullptr, *md = nullptr;
        const int32_t s2 = sa::acquire_meta(pool, sizeof(uint64_t) * size_t(n_sessions), &mh, &md);
        if (s2 != SA_OK) return s2;
        memcpy(mh, images, sizeof(uint64_t) * size_t(n_sessions));
        if (sa::commit_meta(pool, sizeof(uint64_t) * size_t(n_sessions), stream) != SA_OK) return SA_ERR_CUDA;  // counts its launch
        static const sa::InlineImages none{};
        sa::kv_import_kernel<false><<<grid, sa::kXferThreads, 0, stream>>>(
            im, none, req_dev, reinterpret_cast<const uint64_t *>(md), n_sessions, int32_t(total), kb, vb, pool->block_table,
            pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head, pool->cfg.num_kv_heads,
            pool->cfg.head_dim, src_heads, head_begin);
    }
    ++pool->last_launches;
    return cudaGetLastError() == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}

extern "C" int32_t sa_kv_session_import(sa_kv_pool *pool, int32_t sid, int64_t n_tokens, const void *image,
                                        int32_t src_heads, int32_t head_begin, void *stream_) {
    if (n_tokens < 0 || n_tokens > INT32_MAX) return SA_ERR_INVALID_ARG;
    return sa_kv_sessions_import(pool, 1, &sid, &n_tokens, &image, src_heads, head_begin, stream_);
}
