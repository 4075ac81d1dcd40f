// sa_decode_step.cu -- one decode iteration of the latency-critical class as a CUDA-graph-capturable pair of calls
// ("a single query token that attends to its full KV cache of length L_j", the step whose time is
// the TBT the scheduler protects, L392-398).
//
// sa_rope_kv_append + sa_mixed_attention plan on the host and carry their metadata in kernel parameters or through
// a ring of pinned slabs guarded by events: neither can be recorded once and replayed on the next token.  Here the
// two halves are separated for good:
//   sa_decode_step_prepare  host only.  The host half of the append of ONE token per session (page allocation,
//                           session growth) and of the attention plan (splits per request); everything the kernels
//                           need goes into the step's pinned slab.
//   sa_decode_step_enqueue  device only.  Two launches with fixed grids and fixed pointers: slab -> device twin +
//                           RoPE/placement of the new tokens, split-KV decode attention (CTAs stride over the items,
//                           counts read on the device; the last split of a row merges).  Legal under stream capture; a captured
//                           graph is replayed after every prepare.
// The arithmetic is sa_rope_kv_append's and sa_mixed_attention's own (same device functions), so the stored K'/V and
// the output rows are bit-equal to the eager calls.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "sa_internal.h"

struct sa_decode_step {
    sa_kv_pool *pool = nullptr;
    bool host_only = false;      // copies of the pool's, so that destroying the step never reads the pool
    int device = 0;
    int32_t cap = 0;             // most requests a step can carry
    int64_t max_kv = 0;          // longest cache (own token included) a request of a step can have
    int64_t max_part_rows = 0;   // partial rows the workspace holds
    char *slab_host = nullptr;   // pinned (plain memory for a host-only pool)
    char *slab_dev = nullptr;    // inside the caller's device memory
    float *part_o = nullptr, *part_lse = nullptr;
    int32_t grid_ctas = 0;
    int32_t last_launches = 0;
    bool prepared = false;
    // what the last successful prepare did, for sa_decode_step_cancel: (session, length before it, page it took or -1)
    struct Undo {
        int32_t sid;
        int64_t len_before;
        int32_t page_taken;
    };
    std::vector<Undo> undo;
    bool can_cancel = false;
};

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct StepLayout {
    size_t off_part_o, off_part_lse, total;
    int64_t max_part_rows;
};

StepLayout step_layout(const sa_kv_pool *pool, int32_t cap, int64_t max_kv) {
    StepLayout l;
    const int64_t splits = (max_kv + sa::kDecodeSplitKeys - 1) / sa::kDecodeSplitKeys;
    l.max_part_rows = int64_t(cap) * pool->cfg.num_q_heads * splits;
    l.off_part_o = align_up(sa::step_slab_bytes(cap), 256);
    l.off_part_lse = l.off_part_o + align_up(size_t(l.max_part_rows) * size_t(pool->cfg.head_dim) * 4, 256);
    l.total = l.off_part_lse + align_up(size_t(l.max_part_rows) * 4, 256);
    return l;
}

bool args_ok(const sa_kv_pool *pool, int32_t cap, int64_t max_kv) {
    return pool && cap >= 1 && cap <= pool->cfg.max_sessions && max_kv >= 1 && max_kv <= pool->cfg.max_session_tokens;
}

}  // namespace

extern "C" int32_t sa_decode_step_device_bytes(const sa_kv_pool *pool, int32_t max_requests, int64_t max_kv_tokens,
                                               size_t *out_bytes) {
    if (!out_bytes || !args_ok(pool, max_requests, max_kv_tokens)) return SA_ERR_INVALID_ARG;
    *out_bytes = step_layout(pool, max_requests, max_kv_tokens).total;
    return SA_OK;
}

extern "C" int32_t sa_decode_step_create(sa_kv_pool *pool, int32_t max_requests, int64_t max_kv_tokens, void *dev_mem,
                                         size_t dev_bytes, sa_decode_step **out_step) {
    if (!out_step || !args_ok(pool, max_requests, max_kv_tokens)) return SA_ERR_INVALID_ARG;
    const StepLayout l = step_layout(pool, max_requests, max_kv_tokens);
    if (!pool->host_only && (!dev_mem || dev_bytes < l.total || (reinterpret_cast<uintptr_t>(dev_mem) & 255))) return SA_ERR_INVALID_ARG;
    sa_decode_step *st = new (std::nothrow) sa_decode_step();
    if (!st) return SA_ERR_INVALID_ARG;
    st->pool = pool;
    st->host_only = pool->host_only;
    st->device = pool->cfg.device;
    st->cap = max_requests;
    st->max_kv = max_kv_tokens;
    st->max_part_rows = l.max_part_rows;
    const size_t slab = sa::step_slab_bytes(max_requests);
    if (pool->host_only) {
        st->slab_host = static_cast<char *>(calloc(1, slab));
        if (!st->slab_host) {
            delete st;
            return SA_ERR_INVALID_ARG;
        }
    } else {
        sa::DeviceGuard device_guard(pool);
        bool ok = device_guard.ok;
        ok = ok && cudaMallocHost(reinterpret_cast<void **>(&st->slab_host), slab) == cudaSuccess;
        ok = ok && sa::flash_loop_prepare(pool) == cudaSuccess;
        if (!ok) {
            (void)cudaGetLastError();
            if (st->slab_host) cudaFreeHost(st->slab_host);
            delete st;
            return SA_ERR_CUDA;
        }
        memset(st->slab_host, 0, slab);
        char *base = static_cast<char *>(dev_mem);
        st->slab_dev = base;
        st->part_o = reinterpret_cast<float *>(base + l.off_part_o);
        st->part_lse = reinterpret_cast<float *>(base + l.off_part_lse);
        // Two 100 KiB CTAs fit an SM.  The fixed grid holds eight times that many CTAs, each striding over the step's
        // items: the block scheduler hands a freed slot to the next CTA, so uneven items (the ragged last split of a
        // row) balance as they do in the one-CTA-per-item launch; CTAs beyond the step's item count leave at once.
        const int64_t cap_items = int64_t(max_requests) * pool->cfg.num_kv_heads *
                                  ((max_kv_tokens + sa::kDecodeSplitKeys - 1) / sa::kDecodeSplitKeys);
        st->grid_ctas = int32_t(std::min<int64_t>(cap_items, int64_t(16) * pool->num_sms));
    }
    *out_step = st;
    return SA_OK;
}

extern "C" int32_t sa_decode_step_destroy(sa_decode_step *step) {
    if (!step) return SA_ERR_INVALID_ARG;
    if (step->slab_host) {  // the pool may be gone already: nothing of it is read here
        if (step->host_only) {
            free(step->slab_host);
        } else {
            sa::DeviceGuard device_guard(step->device);
            cudaFreeHost(step->slab_host);
        }
    }
    delete step;
    return SA_OK;
}

extern "C" int32_t sa_decode_step_prepare(sa_decode_step *step, int32_t n_req, const int32_t *sids) {
    using namespace sa;
    if (!step || n_req < 0 || n_req > step->cap || (n_req > 0 && !sids)) return SA_ERR_INVALID_ARG;
    sa_kv_pool *pool = step->pool;
    const int B = pool->cfg.page_size;
    // ---- validate and size the page demand before touching any state
    std::vector<char> seen(pool->sessions.size(), 0);
    int64_t need_pages = 0;
    for (int r = 0; r < n_req; ++r) {
        const int32_t sid = sids[r];
        if (sid < 0 || size_t(sid) >= pool->sessions.size() || !pool->sessions[size_t(sid)].open || seen[size_t(sid)])
            return SA_ERR_INVALID_ARG;
        seen[size_t(sid)] = 1;
        const Session &s = pool->sessions[size_t(sid)];
        if (s.len + 1 > step->max_kv) return SA_ERR_INVALID_ARG;
        if (s.len % B == 0) {
            ++need_pages;
        } else if (pool->page_ref[size_t(s.pages.back())] > 1) {
            // a shared partial last page must be copied before it is written (copy-on-write): that is a device copy
            // ordered before the placement, which a prepared, replayable step cannot hold.  sa_rope_kv_append does it.
            return SA_ERR_UNSUPPORTED;
        }
    }
    if (need_pages > int64_t(pool->free_pages.size())) return SA_ERR_OUT_OF_PAGES;
    // ---- cannot fail any more: grow the sessions and write the step's metadata
    StepHeader *hd = reinterpret_cast<StepHeader *>(step->slab_host);
    ReqMeta *meta = reinterpret_cast<ReqMeta *>(step->slab_host + sizeof(StepHeader));
    StepAppend *app = reinterpret_cast<StepAppend *>(step->slab_host + step_append_offset(step->cap));
    const int Hkv = pool->cfg.num_kv_heads, Hq = pool->cfg.num_q_heads;
    int64_t items = 0, parts = 0;
    step->undo.clear();
    for (int r = 0; r < n_req; ++r) {
        Session &s = pool->sessions[size_t(sids[r])];
        sa_decode_step::Undo u{sids[r], s.len, -1};
        if (s.len % B == 0) {
            s.pages.push_back(take_page(pool));
            u.page_taken = s.pages.back();
        }
        step->undo.push_back(u);
        StepAppend a{};
        a.sid = sids[r];
        a.pos = int32_t(s.len);
        a.page = s.pages.back();
        app[r] = a;
        s.len += 1;
        ReqMeta m{};
        m.sid = sids[r];
        m.q_start = r;
        m.q_len = 1;
        m.kv_len = int32_t(s.len);
        m.n_splits = int32_t((s.len + kDecodeSplitKeys - 1) / kDecodeSplitKeys);
        m.item_begin = int32_t(items);
        m.part_begin = int32_t(parts);
        meta[r] = m;
        items += int64_t(Hkv) * m.n_splits;
        parts += int64_t(m.n_splits) * Hq;
    }
    hd->n_req = n_req;
    hd->n_items = int32_t(items);
    step->prepared = true;
    step->can_cancel = true;
    return SA_OK;
}

extern "C" int32_t sa_decode_step_cancel(sa_decode_step *step) {
    using namespace sa;
    if (!step || !step->can_cancel) return SA_ERR_INVALID_ARG;
    sa_kv_pool *pool = step->pool;
    // every session must still be as the prepare left it, or nothing is undone
    for (const sa_decode_step::Undo &u : step->undo) {
        if (u.sid < 0 || size_t(u.sid) >= pool->sessions.size()) return SA_ERR_INVALID_ARG;
        const Session &s = pool->sessions[size_t(u.sid)];
        if (!s.open || s.len != u.len_before + 1 || s.pages.empty()) return SA_ERR_INVALID_ARG;
        if (u.page_taken >= 0 && (s.pages.back() != u.page_taken || pool->page_ref[size_t(u.page_taken)] != 1)) return SA_ERR_INVALID_ARG;
    }
    // in reverse, so that the free list hands the same pages out in the same order again
    for (size_t i = step->undo.size(); i-- > 0;) {
        const sa_decode_step::Undo &u = step->undo[i];
        Session &s = pool->sessions[size_t(u.sid)];
        if (u.page_taken >= 0) {
            release_page(pool, s.pages.back());
            s.pages.pop_back();
        }
        s.len = u.len_before;
    }
    step->undo.clear();
    step->can_cancel = false;
    step->prepared = false;  // the slab describes a batch that no longer exists: enqueue is refused until the next prepare
    StepHeader *hd = reinterpret_cast<StepHeader *>(step->slab_host);
    hd->n_req = 0;
    hd->n_items = 0;
    return SA_OK;
}

extern "C" int32_t sa_decode_step_enqueue(sa_decode_step *step, const void *k, const void *v, void *q_inout, void *out,
                                          float *lse, float sm_scale, void *stream_) {
    using namespace sa;
    if (!step || !k || !v || !q_inout || !out) return SA_ERR_INVALID_ARG;
    sa_kv_pool *pool = step->pool;
    if (pool->host_only) return SA_ERR_CUDA;
    if (!step->prepared) return SA_ERR_INVALID_ARG;
    DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    if (!(sm_scale > 0.f)) sm_scale = 1.0f / sqrtf(float(pool->cfg.head_dim));
    step->last_launches = 0;
    if (launch_step_append(pool, step->slab_host, step->slab_dev, step->cap, k, v, q_inout, stream, &step->last_launches) != cudaSuccess)
        return SA_ERR_CUDA;
    AttnPlan plan;
    plan.n_dec = step->cap;  // length of the step's request array; the count of this step is read on the device
    const ReqMeta *reqs_dev = reinterpret_cast<const ReqMeta *>(step->slab_dev + sizeof(StepHeader));
    const int32_t *dyn = reinterpret_cast<const int32_t *>(step->slab_dev);
    if (launch_flash_decode(pool, reqs_dev, nullptr, plan, q_inout, out, lse, sm_scale, step->part_o, step->part_lse, stream,
                            &step->last_launches, step->grid_ctas, dyn) != cudaSuccess)
        return SA_ERR_CUDA;
    return SA_OK;
}

extern "C" int32_t sa_decode_step_stats(const sa_decode_step *step, int64_t *out_stats) {
    if (!step || !out_stats) return SA_ERR_INVALID_ARG;
    const sa::StepHeader *hd = reinterpret_cast<const sa::StepHeader *>(step->slab_host);
    out_stats[0] = hd->n_req;
    out_stats[1] = hd->n_items;
    out_stats[2] = step->grid_ctas;
    out_stats[3] = step->last_launches;
    out_stats[4] = step->max_part_rows;
    out_stats[5] = step->cap;
    return SA_OK;
}
