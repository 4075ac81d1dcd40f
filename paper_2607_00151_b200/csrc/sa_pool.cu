// sa_pool.cu -- page pool, block tables and sessions (PAPER.md L490 paged
// KV cache, L37 "invalidates the existing KV cache", L494 prefix kept alive across turns).
// Host bookkeeping only; the device side is a mirror of the block tables that the kernels read.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "sa_internal.h"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Carve {
    size_t k_off, v_off, bt_off, rope_off, ticket_off, meta_off, total, kv_bytes, slab;
    int64_t mpps;
};

int32_t check_cfg(const sa_kv_pool_config *c) {
    if (!c) return SA_ERR_INVALID_ARG;
    if (c->num_q_heads <= 0 || c->num_kv_heads <= 0 || c->num_pages <= 0 || c->max_sessions <= 0 ||
        c->max_session_tokens <= 0 || !(c->rope_base > 1.0))
        return SA_ERR_INVALID_ARG;
    if (c->head_dim != 64 && c->head_dim != 128) return SA_ERR_UNSUPPORTED;
    if (c->page_size != 16 && c->page_size != 64) return SA_ERR_UNSUPPORTED;
    if (c->num_q_heads % c->num_kv_heads != 0) return SA_ERR_UNSUPPORTED;
    int g = c->num_q_heads / c->num_kv_heads;
    if (g != 1 && g != 2 && g != 4 && g != 8 && g != 16) return SA_ERR_UNSUPPORTED;
    // positions are carried as exact fp32 integers in the RoPE kernel and int32 in metadata
    if (c->max_session_tokens > (int64_t(1) << 24)) return SA_ERR_UNSUPPORTED;
    if (c->num_pages > (int64_t(1) << 30)) return SA_ERR_UNSUPPORTED;
    return SA_OK;
}

Carve carve(const sa_kv_pool_config *c) {
    Carve r;
    r.mpps = (c->max_session_tokens + c->page_size - 1) / c->page_size;
    r.kv_bytes = size_t(c->num_pages) * c->num_kv_heads * c->page_size * c->head_dim * 2;
    // room for the requests of a call, the new page ids of an append, and a tcgen05 schedule of ~2000 parts
    r.slab = align_up(2 * sizeof(sa::ReqMeta) * (size_t(c->max_sessions) + 8) + 4 * size_t(c->num_pages) + 64 + (64 << 10), 256);
    size_t off = 0;
    r.k_off = off;
    off = align_up(off + r.kv_bytes, 1024);
    r.v_off = off;
    off = align_up(off + r.kv_bytes, 1024);
    r.bt_off = off;
    off = align_up(off + size_t(c->max_sessions) * r.mpps * 4, 256);
    r.rope_off = off;
    off = align_up(off + size_t(c->head_dim / 2) * sizeof(float2), 256);
    r.ticket_off = off;  // one arrival counter per (request of a call, kv head): the last split to finish merges
    off = align_up(off + size_t(c->max_sessions) * c->num_kv_heads * 4, 256);
    r.meta_off = off;
    off += r.slab * sa::kMetaRing;
    r.total = off;
    return r;
}

}  // namespace

extern "C" const char *sa_status_string(int32_t s) {
    switch (s) {
        case SA_OK: return "SA_OK";
        case SA_ERR_INVALID_ARG: return "SA_ERR_INVALID_ARG";
        case SA_ERR_OUT_OF_PAGES: return "SA_ERR_OUT_OF_PAGES";
        case SA_ERR_UNSUPPORTED: return "SA_ERR_UNSUPPORTED";
        case SA_ERR_CUDA: return "SA_ERR_CUDA";
        case SA_ERR_WORKSPACE_TOO_SMALL: return "SA_ERR_WORKSPACE_TOO_SMALL";
        case SA_ERR_OUT_OF_SESSIONS: return "SA_ERR_OUT_OF_SESSIONS";
        default: return "SA_ERR_UNKNOWN";
    }
}

extern "C" int32_t sa_kv_pool_storage_bytes(const sa_kv_pool_config *cfg, size_t *out_bytes) {
    int32_t st = check_cfg(cfg);
    if (st != SA_OK) return st;
    if (!out_bytes) return SA_ERR_INVALID_ARG;
    *out_bytes = carve(cfg).total;
    return SA_OK;
}

extern "C" int32_t sa_kv_pool_create(const sa_kv_pool_config *cfg, void *dev_storage, size_t bytes,
                                     const int32_t *free_page_order, sa_kv_pool **out_pool) {
    int32_t st = check_cfg(cfg);
    if (st != SA_OK) return st;
    if (!out_pool) return SA_ERR_INVALID_ARG;
    Carve cv = carve(cfg);
    if (dev_storage && (bytes < cv.total || (reinterpret_cast<uintptr_t>(dev_storage) & 255)))
        return SA_ERR_INVALID_ARG;
    if (free_page_order) {  // must be a permutation of [0, num_pages)
        std::vector<char> seen(size_t(cfg->num_pages), 0);
        for (int64_t i = 0; i < cfg->num_pages; ++i) {
            int32_t p = free_page_order[i];
            if (p < 0 || p >= cfg->num_pages || seen[p]) return SA_ERR_INVALID_ARG;
            seen[p] = 1;
        }
    }
    sa_kv_pool *pool = new (std::nothrow) sa_kv_pool();
    if (!pool) return SA_ERR_INVALID_ARG;
    pool->cfg = *cfg;
    pool->plan_cache = sa::plan_cache_new();
    if (!pool->plan_cache) {
        delete pool;
        return SA_ERR_INVALID_ARG;
    }
    pool->G = cfg->num_q_heads / cfg->num_kv_heads;
    pool->log2_page = cfg->page_size == 16 ? 4 : 6;
    pool->max_pages_per_session = cv.mpps;
    pool->stride_slot = cfg->head_dim;
    pool->stride_head = int64_t(cfg->page_size) * cfg->head_dim;
    pool->stride_page = int64_t(cfg->num_kv_heads) * pool->stride_head;
    pool->meta_slab_bytes = cv.slab;
    pool->sessions.resize(size_t(cfg->max_sessions));
    pool->free_pages.resize(size_t(cfg->num_pages));
    pool->page_ref.assign(size_t(cfg->num_pages), 0);
    for (int64_t i = 0; i < cfg->num_pages; ++i)  // stack: first of the order is popped first
        pool->free_pages[size_t(cfg->num_pages - 1 - i)] = free_page_order ? free_page_order[i] : int32_t(i);
    pool->host_only = (dev_storage == nullptr);
    if (!pool->host_only) {
        char *base = static_cast<char *>(dev_storage);
        pool->storage = base;
        pool->storage_bytes = bytes;
        pool->k_base = base + cv.k_off;
        pool->v_base = base + cv.v_off;
        pool->block_table = reinterpret_cast<int32_t *>(base + cv.bt_off);
        pool->rope_tab = reinterpret_cast<float2 *>(base + cv.rope_off);
        pool->tickets = reinterpret_cast<int32_t *>(base + cv.ticket_off);
        pool->meta_dev = base + cv.meta_off;
        sa::DeviceGuard device_guard(cfg->device);  // the caller's current device is restored on return
        bool ok = device_guard.ok;
        ok = ok && cudaMallocHost(reinterpret_cast<void **>(&pool->meta_host), cv.slab * sa::kMetaRing) == cudaSuccess;
        for (int i = 0; ok && i < sa::kMetaRing; ++i)
            ok = cudaEventCreateWithFlags(&pool->meta_event[i], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&pool->big_event, cudaEventDisableTiming) == cudaSuccess;
        int sms = 0;
        ok = ok && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cfg->device) == cudaSuccess;
        if (ok) {
            pool->num_sms = sms;
            // RoPE frequencies as turns per position, split hi/lo so that pos * u keeps ~48 bits
            // (reading R9): u_m = rope_base^(-2m/D) / (2 pi).
            const int half = cfg->head_dim / 2;
            std::vector<float2> tab(static_cast<size_t>(half));
            for (int m = 0; m < half; ++m) {
                double u = pow(cfg->rope_base, -2.0 * double(m) / double(cfg->head_dim)) / (2.0 * M_PI);
                float hi = static_cast<float>(u);
                float lo = static_cast<float>(u - double(hi));
                tab[size_t(m)] = make_float2(hi, lo);
            }
            ok = cudaMemcpy(pool->rope_tab, tab.data(), sizeof(float2) * size_t(half), cudaMemcpyHostToDevice) == cudaSuccess;
            // the counters start at zero and every kernel that uses them leaves them at zero
            ok = ok && cudaMemset(pool->tickets, 0, size_t(cfg->max_sessions) * cfg->num_kv_heads * 4) == cudaSuccess;
        }
        if (ok) ok = sa::tc5_init(pool) == SA_OK;
        if (!ok) {
            (void)cudaGetLastError();
            sa_kv_pool_destroy(pool);
            return SA_ERR_CUDA;
        }
    }
    *out_pool = pool;
    return SA_OK;
}

extern "C" int32_t sa_kv_pool_destroy(sa_kv_pool *pool) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    if (!pool) return SA_ERR_INVALID_ARG;
    if (!pool->host_only) {
        for (int i = 0; i < sa::kMetaRing; ++i) {
            if (pool->meta_event[i]) {
                if (pool->meta_event_used[i]) cudaEventSynchronize(pool->meta_event[i]);
                cudaEventDestroy(pool->meta_event[i]);
            }
        }
        if (pool->meta_host) cudaFreeHost(pool->meta_host);
        if (pool->big_event) {
            if (pool->big_event_used) cudaEventSynchronize(pool->big_event);
            cudaEventDestroy(pool->big_event);
        }
        if (pool->big_host) cudaFreeHost(pool->big_host);
    }
    sa::plan_cache_delete(pool->plan_cache);
    delete pool;
    return SA_OK;
}

extern "C" int32_t sa_kv_pool_layout(const sa_kv_pool *pool, sa_kv_layout *out) {
    if (!pool || !out) return SA_ERR_INVALID_ARG;
    out->k_base = pool->k_base;
    out->v_base = pool->v_base;
    out->stride_page = pool->stride_page;
    out->stride_head = pool->stride_head;
    out->stride_slot = pool->stride_slot;
    return SA_OK;
}

extern "C" int32_t sa_kv_pool_free_pages(const sa_kv_pool *pool, int64_t *out_free_pages) {
    if (!pool || !out_free_pages) return SA_ERR_INVALID_ARG;
    *out_free_pages = int64_t(pool->free_pages.size());
    return SA_OK;
}

extern "C" int32_t sa_kv_session_open(sa_kv_pool *pool, int32_t *out_sid) {
    if (!pool || !out_sid) return SA_ERR_INVALID_ARG;
    for (size_t i = 0; i < pool->sessions.size(); ++i) {
        if (!pool->sessions[i].open) {
            pool->sessions[i].open = true;
            pool->sessions[i].len = 0;
            pool->sessions[i].pages.clear();
            *out_sid = int32_t(i);
            return SA_OK;
        }
    }
    return SA_ERR_OUT_OF_SESSIONS;
}

static sa::Session *get_session(sa_kv_pool *pool, int32_t sid) {
    if (!pool || sid < 0 || size_t(sid) >= pool->sessions.size() || !pool->sessions[size_t(sid)].open) return nullptr;
    return &pool->sessions[size_t(sid)];
}

extern "C" int32_t sa_kv_session_truncate(sa_kv_pool *pool, int32_t sid, int64_t new_len) {
    sa::Session *s = get_session(pool, sid);
    if (!s || new_len < 0 || new_len > s->len) return SA_ERR_INVALID_ARG;
    size_t keep = size_t((new_len + pool->cfg.page_size - 1) / pool->cfg.page_size);
    while (s->pages.size() > keep) {
        sa::release_page(pool, s->pages.back());
        s->pages.pop_back();
    }
    s->len = new_len;
    return SA_OK;
}

// ---- session operations of the commit splice ----
// Upload the session's page list into its row of the device block table.
static int32_t upload_row(sa_kv_pool *pool, int32_t sid, cudaStream_t stream) {
    const sa::Session &s = pool->sessions[size_t(sid)];
    if (pool->host_only || s.pages.empty()) return SA_OK;
    char *mh = nullptr, *md = nullptr;
    const size_t bytes = s.pages.size() * sizeof(int32_t);  // the slab holds 4 bytes per pool page: always fits
    int32_t st = sa::acquire_meta(pool, bytes, &mh, &md);
    if (st != SA_OK) return st;
    memcpy(mh, s.pages.data(), bytes);
    return sa::commit_meta_to(pool, pool->block_table + int64_t(sid) * pool->max_pages_per_session, bytes, stream);
}

extern "C" int32_t sa_kv_session_fork(sa_kv_pool *pool, int32_t src_sid, int64_t prefix_len, int32_t *out_sid, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    sa::Session *src = get_session(pool, src_sid);
    if (!src || !out_sid || prefix_len < 0 || prefix_len > src->len) return SA_ERR_INVALID_ARG;
    const int B = pool->cfg.page_size;
    const size_t full = size_t(prefix_len / B);
    const bool partial = prefix_len % B != 0;
    if (partial && pool->free_pages.empty()) return SA_ERR_OUT_OF_PAGES;
    int32_t sid = -1;
    int32_t st = sa_kv_session_open(pool, &sid);
    if (st != SA_OK) return st;
    src = get_session(pool, src_sid);
    sa::Session &dst = pool->sessions[size_t(sid)];
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    for (size_t i = 0; i < full; ++i) {  // whole pages of the retained prefix are shared, never written again
        dst.pages.push_back(src->pages[i]);
        ++pool->page_ref[size_t(src->pages[i])];
    }
    if (partial) {  // the page the prefix ends in will be appended to by the fork: it gets its own copy now
        const int32_t p = sa::take_page(pool);
        dst.pages.push_back(p);
        if (!pool->host_only && sa::copy_page_async(pool, p, src->pages[full], stream) != cudaSuccess) {
            sa_kv_session_close(pool, sid);
            return SA_ERR_CUDA;
        }
    }
    dst.len = prefix_len;
    st = upload_row(pool, sid, stream);
    if (st != SA_OK) {
        sa_kv_session_close(pool, sid);
        return st;
    }
    *out_sid = sid;
    return SA_OK;
}

extern "C" int32_t sa_kv_session_commit(sa_kv_pool *pool, int32_t main_sid, int32_t lookahead_sid, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    sa::Session *m = get_session(pool, main_sid);
    sa::Session *la = get_session(pool, lookahead_sid);
    if (!m || !la || main_sid == lookahead_sid) return SA_ERR_INVALID_ARG;
    // the main session takes over the lookahead's block table; the superseded pages lose a holder
    std::vector<int32_t> old;
    old.swap(m->pages);
    m->pages.swap(la->pages);
    m->len = la->len;
    la->len = 0;
    la->open = false;
    for (int32_t p : old) sa::release_page(pool, p);
    return upload_row(pool, main_sid, static_cast<cudaStream_t>(stream_));
}

extern "C" int32_t sa_kv_page_refcount(const sa_kv_pool *pool, int32_t page, int32_t *out_refs) {
    if (!pool || !out_refs || page < 0 || page >= pool->cfg.num_pages) return SA_ERR_INVALID_ARG;
    *out_refs = pool->page_ref[size_t(page)];
    return SA_OK;
}

extern "C" int32_t sa_kv_session_close(sa_kv_pool *pool, int32_t sid) {
    sa::Session *s = get_session(pool, sid);
    if (!s) return SA_ERR_INVALID_ARG;
    sa_kv_session_truncate(pool, sid, 0);
    s->open = false;
    return SA_OK;
}

extern "C" int32_t sa_kv_session_query(const sa_kv_pool *pool, int32_t sid, int64_t *len, int32_t *pages,
                                       int32_t *n_pages) {
    const sa::Session *s = get_session(const_cast<sa_kv_pool *>(pool), sid);
    if (!s) return SA_ERR_INVALID_ARG;
    if (len) *len = s->len;
    if (n_pages) {
        if (pages) {
            int32_t n = std::min<int32_t>(*n_pages, int32_t(s->pages.size()));
            if (n > 0) memcpy(pages, s->pages.data(), sizeof(int32_t) * size_t(n));
        }
        *n_pages = int32_t(s->pages.size());
    }
    return SA_OK;
}

extern "C" int32_t sa_last_launch_count(const sa_kv_pool *pool, int32_t *out_launches) {
    if (!pool || !out_launches) return SA_ERR_INVALID_ARG;
    *out_launches = pool->last_launches;
    return SA_OK;
}

namespace sa {

int32_t acquire_meta(sa_kv_pool *pool, size_t bytes, char **host, char **dev) {
    if (bytes > pool->meta_slab_bytes) return SA_ERR_UNSUPPORTED;
    int i = pool->meta_next;
    if (pool->meta_event_used[i]) {
        if (cudaEventSynchronize(pool->meta_event[i]) != cudaSuccess) return SA_ERR_CUDA;
        pool->meta_event_used[i] = false;
    }
    *host = pool->meta_host + size_t(i) * pool->meta_slab_bytes;
    *dev = pool->meta_dev + size_t(i) * pool->meta_slab_bytes;
    return SA_OK;
}

int32_t take_page(sa_kv_pool *pool) {
    const int32_t p = pool->free_pages.back();
    pool->free_pages.pop_back();
    pool->page_ref[size_t(p)] = 1;
    return p;
}

void release_page(sa_kv_pool *pool, int32_t page) {
    if (--pool->page_ref[size_t(page)] == 0) pool->free_pages.push_back(page);
}

cudaError_t copy_page_async(const sa_kv_pool *pool, int32_t dst_page, int32_t src_page, cudaStream_t stream) {
    const size_t bytes = size_t(pool->stride_page) * 2;
    const char *kb = static_cast<const char *>(pool->k_base), *vb = static_cast<const char *>(pool->v_base);
    cudaError_t e = cudaMemcpyAsync(const_cast<char *>(kb) + size_t(dst_page) * bytes, kb + size_t(src_page) * bytes, bytes,
                                    cudaMemcpyDeviceToDevice, stream);
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(const_cast<char *>(vb) + size_t(dst_page) * bytes, vb + size_t(src_page) * bytes, bytes,
                           cudaMemcpyDeviceToDevice, stream);
}

int32_t commit_meta(sa_kv_pool *pool, size_t bytes, cudaStream_t stream) {
    int i = pool->meta_next;
    char *dev = pool->meta_dev + size_t(i) * pool->meta_slab_bytes;
    return commit_meta_to(pool, dev, bytes, stream);
}

// Per-call metadata goes from the pinned slab to the device through the SMs, not the copy engine: a
// cudaMemcpyAsync would queue behind whatever bulk host-to-device upload the caller has in flight on
// another stream (there is one H2D engine), and the attention kernel behind it -- measured: +0.5 ms per
// 25 MB upload running beside the call.  Pinned memory is device-addressable under unified addressing.
__global__ void __launch_bounds__(256) meta_upload_kernel(uint32_t *__restrict__ dst, const uint32_t *__restrict__ src, size_t words) {
    // staged behind the kernel before it and in front of the one after it (programmatic dependent launch); it waits
    // before it writes: the slab's device twin may still be read by the kernels of an earlier call
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < words; i += size_t(gridDim.x) * blockDim.x) dst[i] = src[i];
}

static cudaError_t meta_upload(sa_kv_pool *pool, void *dev, const void *host, size_t bytes, cudaStream_t stream) {
    const size_t words = (bytes + 3) / 4;  // every metadata record is a whole number of 32-bit words
    if (words == 0) return cudaSuccess;
    const unsigned blocks = unsigned(std::min<size_t>((words + 255) / 256, 128));
    const cudaError_t e = sa::launch_pdl(meta_upload_kernel, dim3(blocks), dim3(256), 0, stream, static_cast<uint32_t *>(dev),
                                         static_cast<const uint32_t *>(host), words);
    ++pool->last_launches;
    return e;
}

int32_t commit_meta_to(sa_kv_pool *pool, void *dev, size_t bytes, cudaStream_t stream) {
    int slot = 0;
    const int32_t st = commit_meta_deferred(pool, dev, bytes, stream, &slot);
    return st == SA_OK ? meta_mark(pool, slot, stream) : st;
}

// The same without the event that frees the pinned slab for reuse: the caller records it (meta_mark) after the kernels
// that follow the upload -- an event record between two kernels would keep the second from being staged behind the first.
int32_t commit_meta_deferred(sa_kv_pool *pool, void *dev, size_t bytes, cudaStream_t stream, int *slot) {
    const int i = pool->meta_next;
    char *host = pool->meta_host + size_t(i) * pool->meta_slab_bytes;
    if (!dev) dev = pool->meta_dev + size_t(i) * pool->meta_slab_bytes;
    if (meta_upload(pool, dev, host, bytes, stream) != cudaSuccess) return SA_ERR_CUDA;
    pool->meta_next = (i + 1) % kMetaRing;
    *slot = i;
    return SA_OK;
}

int32_t meta_mark(sa_kv_pool *pool, int slot, cudaStream_t stream) {
    if (cudaEventRecord(pool->meta_event[slot], stream) != cudaSuccess) return SA_ERR_CUDA;
    pool->meta_event_used[slot] = true;
    return SA_OK;
}

int32_t acquire_big_meta(sa_kv_pool *pool, size_t bytes, char **host) {
    if (pool->big_event_used) {
        if (cudaEventSynchronize(pool->big_event) != cudaSuccess) return SA_ERR_CUDA;
        pool->big_event_used = false;
    }
    if (bytes > pool->big_cap) {
        if (pool->big_host) cudaFreeHost(pool->big_host);
        pool->big_host = nullptr;
        pool->big_cap = 0;
        const size_t cap = std::max(bytes * 2, size_t(1) << 20);
        if (cudaMallocHost(reinterpret_cast<void **>(&pool->big_host), cap) != cudaSuccess) {
            (void)cudaGetLastError();
            return SA_ERR_CUDA;
        }
        pool->big_cap = cap;
    }
    *host = pool->big_host;
    return SA_OK;
}

int32_t commit_big_meta(sa_kv_pool *pool, void *dev_dst, size_t bytes, cudaStream_t stream) {
    if (meta_upload(pool, dev_dst, pool->big_host, bytes, stream) != cudaSuccess) return SA_ERR_CUDA;
    if (cudaEventRecord(pool->big_event, stream) != cudaSuccess) return SA_ERR_CUDA;
    pool->big_event_used = true;
    return SA_OK;
}

}  // namespace sa
