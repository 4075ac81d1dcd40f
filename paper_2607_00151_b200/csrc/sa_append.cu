// sa_append.cu -- sa_rope_kv_append: fused RoPE + scatter of new K/V into pool pages
// ("KV cache construction that depends on the previously
// transformed prefix").  HBM-bound: every byte is read once and written once, 128-bit accesses.
#include <cuda_bf16.h>

#include <algorithm>
#include <utility>
#include <vector>

#include "sa_internal.h"

namespace sa {

constexpr int kAppendTok = 8;       // tokens per CTA (4: 84 %, 8: 89 %, 16: 89 % of the HBM copy peak on config 4's fill)
constexpr int kAppendThreads = 256;

__device__ __forceinline__ void unpack8(const uint4 &u, float (&f)[8]) {
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        f[2 * i] = __uint_as_float(w[i] << 16);
        f[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
}

__device__ __forceinline__ uint4 pack8(const float (&f)[8]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        __nv_bfloat162 p = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);  // round-to-nearest-even
        w[i] = *reinterpret_cast<uint32_t *>(&p);
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}

// New page ids of this call -> device block table.  One CTA per request that gained pages.
__global__ void block_table_update_kernel(const ReqMeta *__restrict__ reqs, const int32_t *__restrict__ new_pages,
                                          int32_t *__restrict__ block_table, int64_t mpps) {
    const ReqMeta r = reqs[blockIdx.x];
    int32_t *row = block_table + int64_t(r.sid) * mpps + r.part_begin;
    for (int i = threadIdx.x; i < r.n_splits; i += blockDim.x) row[i] = new_pages[r.item_begin + i];
}

// RoPE tables of the CTA's tokens, then the copy itself.  s_pos / s_dst: position and destination (element offset of
// the token's slot inside a (page, head 0) block) of each of the CTA's n_tok tokens, filled by the caller.
template <int D>
__device__ __forceinline__ void append_rows(int64_t t0, int n_tok, const int32_t *s_pos, const int64_t *s_dst,
                                            float2 (*s_cs)[D / 2], const __nv_bfloat16 *__restrict__ k,
                                            const __nv_bfloat16 *__restrict__ v, __nv_bfloat16 *__restrict__ q,
                                            __nv_bfloat16 *__restrict__ k_base, __nv_bfloat16 *__restrict__ v_base,
                                            int64_t stride_head, const float2 *__restrict__ rope_tab, int32_t Hq,
                                            int32_t Hkv, int tid) {
    constexpr int HALF = D / 2;
    constexpr int UPH = D / 16;  // units per head
    for (int e = tid; e < n_tok * HALF; e += kAppendThreads) {
        const int tl = e / HALF, m = e % HALF;
        s_cs[tl][m] = rope_cos_sin(s_pos[tl], rope_tab[m]);
    }
    __syncthreads();

    const int heads = 2 * Hkv + (q ? Hq : 0);
    const int units_per_tok = heads * UPH;
    const int total_units = n_tok * units_per_tok;
    constexpr int U = 2;  // units in flight per thread
    for (int base = tid; base < total_units; base += kAppendThreads * U) {
        uint4 a[U], b[U];
        __nv_bfloat16 *dst[U];
        int tl_[U], j_[U];
        bool rot[U], live[U];
#pragma unroll
        for (int i = 0; i < U; ++i) {
            const int e = base + i * kAppendThreads;
            live[i] = e < total_units;
            if (!live[i]) continue;
            const int tl = e / units_per_tok, u = e % units_per_tok;
            const int hu = u / UPH, j = u % UPH;
            const int64_t row = t0 + tl;
            const __nv_bfloat16 *src;
            if (hu < Hkv) {
                src = k + (row * Hkv + hu) * D;
                dst[i] = k_base + s_dst[tl] + int64_t(hu) * stride_head;
                rot[i] = true;
            } else if (hu < 2 * Hkv) {
                src = v + (row * Hkv + (hu - Hkv)) * D;
                dst[i] = v_base + s_dst[tl] + int64_t(hu - Hkv) * stride_head;
                rot[i] = false;
            } else {
                __nv_bfloat16 *qp = q + (row * Hq + (hu - 2 * Hkv)) * D;
                src = qp;
                dst[i] = qp;
                rot[i] = true;
            }
            tl_[i] = tl;
            j_[i] = j;
            a[i] = *reinterpret_cast<const uint4 *>(src + 8 * j);
            b[i] = *reinterpret_cast<const uint4 *>(src + HALF + 8 * j);
        }
#pragma unroll
        for (int i = 0; i < U; ++i) {
            if (!live[i]) continue;
            if (rot[i]) {
                float x0[8], x1[8], y0[8], y1[8];
                unpack8(a[i], x0);
                unpack8(b[i], x1);
#pragma unroll
                for (int d = 0; d < 8; ++d) {
                    const float2 c = s_cs[tl_[i]][8 * j_[i] + d];
                    y0[d] = fmaf(x0[d], c.x, -(x1[d] * c.y));
                    y1[d] = fmaf(x1[d], c.x, x0[d] * c.y);
                }
                a[i] = pack8(y0);
                b[i] = pack8(y1);
            }
            *reinterpret_cast<uint4 *>(dst[i] + 8 * j_[i]) = a[i];
            *reinterpret_cast<uint4 *>(dst[i] + HALF + 8 * j_[i]) = b[i];
        }
    }
}

// Per token: (2*Hkv + Hq) heads, each D/16 "units" of two 16-byte vectors (dims [8j, 8j+8) and
// [D/2+8j, D/2+8j+8)): K and Q units are rotated, V units are copied bit for bit.
// INLINE: the call's metadata (requests, new page ids) rides in the kernel parameters instead of the slab: no upload
// launch, no block-table launch -- the thread that places a token in a page this call allocated also writes that
// page's block-table entry (every new page receives at least one new token; equal values from several threads).
template <int D, bool INLINE>
__global__ void __launch_bounds__(kAppendThreads)
rope_append_kernel(const __grid_constant__ InlineAppendMeta im, const ReqMeta *__restrict__ reqs_slab, int32_t n_req_slab, int64_t total_rows,
                   const __nv_bfloat16 *__restrict__ k, const __nv_bfloat16 *__restrict__ v,
                   __nv_bfloat16 *__restrict__ q, __nv_bfloat16 *__restrict__ k_base,
                   __nv_bfloat16 *__restrict__ v_base, int32_t *block_table, int64_t mpps,
                   int32_t log2_page, int64_t stride_page, int64_t stride_head,
                   const float2 *__restrict__ rope_tab, int32_t Hq, int32_t Hkv) {
    // staged behind the kernel before it in the stream, and the next one behind it (programmatic dependent launch);
    // everything it reads and writes is ordered by the stream, so it waits first
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const ReqMeta *reqs = INLINE ? im.reqs : reqs_slab;
    const int32_t n_req = INLINE ? im.n_req : n_req_slab;
    constexpr int HALF = D / 2;
    constexpr int UPH = D / 16;  // units per head
    __shared__ int64_t s_dst[kAppendTok];
    __shared__ float2 s_cs[kAppendTok][HALF];
    __shared__ int32_t s_pos[kAppendTok];

    const int64_t t0 = int64_t(blockIdx.x) * kAppendTok;
    const int n_tok = int(min(int64_t(kAppendTok), total_rows - t0));
    const int tid = threadIdx.x;

    if (tid < n_tok) {
        const int64_t t = t0 + tid;
        int lo = 0, hi = n_req - 1;  // last request with q_start <= t (empty requests never match last)
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (reqs[mid].q_start <= t) lo = mid; else hi = mid - 1;
        }
        const ReqMeta r = reqs[lo];
        const int32_t pos = r.kv_len + int32_t(t - r.q_start);
        const int32_t pi = pos >> log2_page;
        int32_t page;
        if (INLINE && pi >= r.part_begin && pi - r.part_begin < r.n_splits) {
            page = im.pages[r.item_begin + pi - r.part_begin];       // allocated (or copied on write) by this call
            block_table[int64_t(r.sid) * mpps + pi] = page;
        } else {
            page = block_table[int64_t(r.sid) * mpps + pi];
        }
        const int32_t slot = pos & ((1 << log2_page) - 1);
        s_pos[tid] = pos;
        s_dst[tid] = int64_t(page) * stride_page + int64_t(slot) * D;
    }
    __syncthreads();
    append_rows<D>(t0, n_tok, s_pos, s_dst, s_cs, k, v, q, k_base, v_base, stride_head, rope_tab, Hq, Hkv, tid);
}

// The new token of every request of a captured decode step (sa_decode_step_enqueue).  The step's metadata sits in a
// pinned host slab that sa_decode_step_prepare rewrites between replays: this kernel copies it to its device twin
// (the attention kernels behind it read that) and places the tokens from the host copy directly -- position and page
// of every token are decided on the host, so the block table is only written here, never read.  Same arithmetic as
// rope_append_kernel (append_rows), so the stored bits are those of sa_rope_kv_append.
template <int D>
__global__ void __launch_bounds__(kAppendThreads)
step_append_kernel(const uint32_t *__restrict__ slab_host, uint32_t *__restrict__ slab_dev, int32_t words, int32_t cap,
                   const __nv_bfloat16 *__restrict__ k, const __nv_bfloat16 *__restrict__ v, __nv_bfloat16 *__restrict__ q,
                   __nv_bfloat16 *__restrict__ k_base, __nv_bfloat16 *__restrict__ v_base, int32_t *block_table,
                   int64_t mpps, int32_t log2_page, int64_t stride_page, int64_t stride_head,
                   const float2 *__restrict__ rope_tab, int32_t Hq, int32_t Hkv) {
    __shared__ int64_t s_dst[kAppendTok];
    __shared__ float2 s_cs[kAppendTok][D / 2];
    __shared__ int32_t s_pos[kAppendTok];
    const int tid = threadIdx.x;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the attention grid may be staged behind this one
    // the CTA's own records and the request count come straight from the pinned slab, all reads issued together (one
    // PCIe round trip); the copy to the device twin rides along
    const StepHeader *hd = reinterpret_cast<const StepHeader *>(slab_host);
    const StepAppend *ap = reinterpret_cast<const StepAppend *>(reinterpret_cast<const char *>(slab_host) + step_append_offset(cap));
    const int64_t t0 = int64_t(blockIdx.x) * kAppendTok;
    StepAppend x = {0, 0, 0, 0};
    if (tid < kAppendTok && t0 + tid < cap) x = ap[t0 + tid];
    {   // while the slab crosses PCIe: pull the rows this CTA may place (and the RoPE table) into L2
        const int64_t n_max = min(int64_t(kAppendTok), int64_t(cap) - t0);
        const char *kp = reinterpret_cast<const char *>(k + t0 * Hkv * D), *vp = reinterpret_cast<const char *>(v + t0 * Hkv * D);
        const char *qp = reinterpret_cast<const char *>(q + t0 * Hq * D);
        const int64_t kv_bytes = n_max * Hkv * D * 2, q_bytes = n_max * Hq * D * 2;
        for (int64_t o = int64_t(tid) * 128; o < kv_bytes; o += int64_t(kAppendThreads) * 128) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(kp + o));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(vp + o));
        }
        for (int64_t o = int64_t(tid) * 128; o < q_bytes; o += int64_t(kAppendThreads) * 128)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(qp + o));
        if (tid * 128 < int(D / 2 * sizeof(float2)))
            asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(rope_tab) + tid * 128));
    }
    const int n_req = hd->n_req;
    for (int i = blockIdx.x * kAppendThreads + tid; i < words; i += gridDim.x * kAppendThreads) slab_dev[i] = slab_host[i];
    const int n_tok = int(max(int64_t(0), min(int64_t(kAppendTok), int64_t(n_req) - t0)));
    if (tid < n_tok) {
        block_table[int64_t(x.sid) * mpps + (x.pos >> log2_page)] = x.page;
        s_pos[tid] = x.pos;
        s_dst[tid] = int64_t(x.page) * stride_page + int64_t(x.pos & ((1 << log2_page) - 1)) * D;
    }
    __syncthreads();
    if (n_tok > 0) append_rows<D>(t0, n_tok, s_pos, s_dst, s_cs, k, v, q, k_base, v_base, stride_head, rope_tab, Hq, Hkv, tid);
}

template <bool INLINE>
static cudaError_t launch_rope_append_t(const sa_kv_pool *pool, const InlineAppendMeta &im, const ReqMeta *reqs_dev,
                                        int32_t n_req, int64_t total_rows, const void *k, const void *v, void *q,
                                        cudaStream_t stream, int32_t *launches) {
    if (total_rows == 0) return cudaSuccess;
    const unsigned grid = unsigned((total_rows + kAppendTok - 1) / kAppendTok);
    auto kb = static_cast<__nv_bfloat16 *>(pool->k_base);
    auto vb = static_cast<__nv_bfloat16 *>(pool->v_base);
    cudaError_t e;
    if (pool->cfg.head_dim == 128)
        e = launch_pdl(rope_append_kernel<128, INLINE>, dim3(grid), dim3(kAppendThreads), 0, stream, im, reqs_dev, n_req, total_rows,
                       static_cast<const __nv_bfloat16 *>(k), static_cast<const __nv_bfloat16 *>(v), static_cast<__nv_bfloat16 *>(q), kb,
                       vb, pool->block_table, pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head,
                       static_cast<const float2 *>(pool->rope_tab), pool->cfg.num_q_heads, pool->cfg.num_kv_heads);
    else
        e = launch_pdl(rope_append_kernel<64, INLINE>, dim3(grid), dim3(kAppendThreads), 0, stream, im, reqs_dev, n_req, total_rows,
                       static_cast<const __nv_bfloat16 *>(k), static_cast<const __nv_bfloat16 *>(v), static_cast<__nv_bfloat16 *>(q), kb,
                       vb, pool->block_table, pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head,
                       static_cast<const float2 *>(pool->rope_tab), pool->cfg.num_q_heads, pool->cfg.num_kv_heads);
    ++*launches;
    return e;
}

cudaError_t launch_step_append(const sa_kv_pool *pool, const void *slab_host, void *slab_dev, int32_t cap, const void *k,
                               const void *v, void *q, cudaStream_t stream, int32_t *launches) {
    const unsigned grid = unsigned((cap + kAppendTok - 1) / kAppendTok);
    const int32_t words = int32_t(step_slab_bytes(cap) / 4);
    auto kb = static_cast<__nv_bfloat16 *>(pool->k_base);
    auto vb = static_cast<__nv_bfloat16 *>(pool->v_base);
    if (pool->cfg.head_dim == 128)
        step_append_kernel<128><<<grid, kAppendThreads, 0, stream>>>(
            static_cast<const uint32_t *>(slab_host), static_cast<uint32_t *>(slab_dev), words, cap,
            static_cast<const __nv_bfloat16 *>(k), static_cast<const __nv_bfloat16 *>(v), static_cast<__nv_bfloat16 *>(q), kb, vb,
            pool->block_table, pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head,
            pool->rope_tab, pool->cfg.num_q_heads, pool->cfg.num_kv_heads);
    else
        step_append_kernel<64><<<grid, kAppendThreads, 0, stream>>>(
            static_cast<const uint32_t *>(slab_host), static_cast<uint32_t *>(slab_dev), words, cap,
            static_cast<const __nv_bfloat16 *>(k), static_cast<const __nv_bfloat16 *>(v), static_cast<__nv_bfloat16 *>(q), kb, vb,
            pool->block_table, pool->max_pages_per_session, pool->log2_page, pool->stride_page, pool->stride_head,
            pool->rope_tab, pool->cfg.num_q_heads, pool->cfg.num_kv_heads);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_rope_append(const sa_kv_pool *pool, const ReqMeta *reqs_dev, int32_t n_req,
                               int64_t total_rows, const void *k, const void *v, void *q,
                               cudaStream_t stream, int32_t *launches) {
    static const InlineAppendMeta none{};  // the slab variant never reads it
    return launch_rope_append_t<false>(pool, none, reqs_dev, n_req, total_rows, k, v, q, stream, launches);
}

}  // namespace sa

namespace sa {

// Host half of an append (step a1): validates the batch, allocates pages (copy-on-write of a shared
// partial page included), grows the sessions, sends the per-request metadata and the new page ids to
// the device and enqueues the block-table update.  *reqs_dev: the ReqMeta array of the call on the
// device (kv_len = position of the request's first new token).  Nothing is changed on failure.
int32_t append_prepare(sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr,
                       bool have_data, cudaStream_t stream, const ReqMeta **reqs_dev_out, int64_t *total_out,
                       InlineAppendMeta *im) {
    *reqs_dev_out = nullptr;
    *total_out = 0;
    if (im) im->used = 0;
    if (!pool || n_req < 0) return SA_ERR_INVALID_ARG;
    if (n_req == 0) {
        pool->last_launches = 0;
        return SA_OK;
    }
    if (!sids || !qo_indptr || qo_indptr[0] != 0 || n_req > pool->cfg.max_sessions) return SA_ERR_INVALID_ARG;
    const int B = pool->cfg.page_size;
    // ---- validate everything and size the page demand before touching any state
    std::vector<char> seen(pool->sessions.size(), 0);
    std::vector<std::pair<int32_t, int32_t>> shared_tail;  // (shared partial last page, appenders of it in this call)
    int64_t need_pages = 0;
    for (int r = 0; r < n_req; ++r) {
        const int32_t sid = sids[r];
        if (sid < 0 || size_t(sid) >= pool->sessions.size() || !pool->sessions[size_t(sid)].open || seen[size_t(sid)])
            return SA_ERR_INVALID_ARG;
        seen[size_t(sid)] = 1;
        const int64_t n = int64_t(qo_indptr[r + 1]) - qo_indptr[r];
        if (n < 0) return SA_ERR_INVALID_ARG;
        const Session &s = pool->sessions[size_t(sid)];
        if (s.len + n > pool->cfg.max_session_tokens) return SA_ERR_INVALID_ARG;
        need_pages += (s.len + n + B - 1) / B - int64_t(s.pages.size());
        // copy-on-write: appending into a partly filled last page that another session also holds
        if (n > 0 && s.len % B != 0 && pool->page_ref[size_t(s.pages.back())] > 1) {
            bool found = false;
            for (auto &sp : shared_tail)
                if (sp.first == s.pages.back()) {
                    ++sp.second;
                    found = true;
                }
            if (!found) shared_tail.push_back(std::make_pair(s.pages.back(), 1));
        }
    }
    // a page held by c sessions of which k append into it in this call is copied min(k, c - 1) times: every copy drops a
    // holder, and the last holder keeps the page itself
    for (const auto &sp : shared_tail) need_pages += std::min<int64_t>(sp.second, pool->page_ref[size_t(sp.first)] - 1);
    const int64_t total = qo_indptr[n_req];
    if (need_pages > int64_t(pool->free_pages.size())) return SA_ERR_OUT_OF_PAGES;
    if (!pool->host_only && total > 0 && !have_data) return SA_ERR_INVALID_ARG;

    // small calls carry their metadata in the kernel parameters (sa_rope_kv_append only: im != nullptr)
    const bool inline_meta = im && !pool->host_only && n_req <= kInlineReqs && need_pages <= kInlinePages;
    char *mh = nullptr, *md = nullptr;
    if (!pool->host_only && !inline_meta) {
        // upper bound of the slab layout written below: [ReqMeta x n_req][new page ids][ReqMeta x (gained <= n_req)]
        int32_t st = acquire_meta(pool, 2 * sizeof(ReqMeta) * size_t(n_req) + sizeof(int32_t) * size_t(need_pages + 1) + 16, &mh, &md);
        if (st != SA_OK) return st;
    }
    std::vector<ReqMeta> host_meta;  // host-only pools keep the same bookkeeping path
    ReqMeta *meta = nullptr;
    int32_t *page_list = nullptr;
    std::vector<int32_t> host_pages;
    if (pool->host_only) {
        host_meta.resize(size_t(n_req));
        host_pages.resize(size_t(need_pages) + 1);
        meta = host_meta.data();
        page_list = host_pages.data();
    } else if (inline_meta) {
        meta = im->reqs;
        page_list = im->pages;
    } else {
        meta = reinterpret_cast<ReqMeta *>(mh);
        page_list = reinterpret_cast<int32_t *>(mh + sizeof(ReqMeta) * size_t(n_req));
    }
    // ---- allocate pages (cannot fail any more) and build the metadata
    int32_t n_list = 0, n_gain = 0;
    std::vector<std::pair<int32_t, int32_t>> cow;  // (private copy, shared page) of this call
    std::vector<ReqMeta> gain;  // requests that gained pages, for the block-table update
    for (int r = 0; r < n_req; ++r) {
        Session &s = pool->sessions[size_t(sids[r])];
        const int64_t n = int64_t(qo_indptr[r + 1]) - qo_indptr[r];
        const int64_t want = (s.len + n + B - 1) / B;
        ReqMeta m{};
        m.sid = sids[r];
        m.q_start = qo_indptr[r];
        m.q_len = int32_t(n);
        m.kv_len = int32_t(s.len);  // position of the request's first new token
        m.item_begin = n_list;
        m.part_begin = int32_t(s.pages.size());
        if (n > 0 && s.len % B != 0 && pool->page_ref[size_t(s.pages.back())] > 1) {
            // the shared page keeps its bits for its other holders; this session continues in a private copy
            const int32_t shared = s.pages.back();
            const int32_t p = take_page(pool);
            if (!pool->host_only) cow.push_back(std::make_pair(p, shared));
            release_page(pool, shared);
            s.pages.back() = p;
            m.part_begin = int32_t(s.pages.size()) - 1;  // the block-table update rewrites this entry too
            page_list[n_list++] = p;
        }
        while (int64_t(s.pages.size()) < want) {
            const int32_t p = take_page(pool);
            s.pages.push_back(p);
            page_list[n_list++] = p;
        }
        m.n_splits = n_list - m.item_begin;
        meta[r] = m;
        if (m.n_splits > 0) {
            gain.push_back(m);
            ++n_gain;
        }
        s.len += n;
    }
    pool->last_launches = 0;
    if (pool->host_only) return SA_OK;

    for (const auto &c : cow)
        if (copy_page_async(pool, c.first, c.second, stream) != cudaSuccess) return SA_ERR_CUDA;
    if (inline_meta) {
        im->n_req = n_req;
        im->n_list = n_list;
        im->used = 1;
        *total_out = total;
        return SA_OK;
    }
    // slab layout: [ReqMeta x n_req][new page ids x n_list][ReqMeta x n_gain]
    size_t off_gain = sizeof(ReqMeta) * size_t(n_req) + sizeof(int32_t) * size_t(n_list);
    off_gain = (off_gain + 15) / 16 * 16;
    // (the slab is sized for 2 x max_sessions entries + num_pages ids, so this always fits)
    if (n_gain > 0) memcpy(mh + off_gain, gain.data(), sizeof(ReqMeta) * size_t(n_gain));
    const size_t bytes = n_gain > 0 ? off_gain + sizeof(ReqMeta) * size_t(n_gain) : off_gain;
    if (commit_meta(pool, bytes, stream) != SA_OK) return SA_ERR_CUDA;
    const ReqMeta *reqs_dev = reinterpret_cast<const ReqMeta *>(md);
    const int32_t *pages_dev = reinterpret_cast<const int32_t *>(md + sizeof(ReqMeta) * size_t(n_req));
    if (n_gain > 0) {
        block_table_update_kernel<<<unsigned(n_gain), 128, 0, stream>>>(
            reinterpret_cast<const ReqMeta *>(md + off_gain), pages_dev, pool->block_table, pool->max_pages_per_session);
        ++pool->last_launches;
    }
    if (cudaGetLastError() != cudaSuccess) return SA_ERR_CUDA;
    *reqs_dev_out = reqs_dev;
    *total_out = total;
    return SA_OK;
}

}  // namespace sa

extern "C" int32_t sa_rope_kv_append(sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                     const int32_t *qo_indptr, const void *k, const void *v, void *q_inout,
                                     void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    using namespace sa;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const ReqMeta *reqs_dev = nullptr;
    int64_t total = 0;
    InlineAppendMeta im;
    const int32_t st = append_prepare(pool, n_req, sids, qo_indptr, k && v, stream, &reqs_dev, &total, &im);
    if (st != SA_OK) return st;
    if (im.used) {
        if (launch_rope_append_t<true>(pool, im, nullptr, 0, total, k, v, q_inout, stream, &pool->last_launches) != cudaSuccess)
            return SA_ERR_CUDA;
        return SA_OK;
    }
    if (!reqs_dev) return st;
    if (launch_rope_append(pool, reqs_dev, n_req, total, k, v, q_inout, stream, &pool->last_launches) != cudaSuccess)
        return SA_ERR_CUDA;
    return SA_OK;
}
