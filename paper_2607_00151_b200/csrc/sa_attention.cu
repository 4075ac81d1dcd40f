// sa_attention.cu -- sa_mixed_attention: host-side batch planning and the
// dispatch of a ragged batch of prefill chunks and decode rows to the kernels (steps a4-a6).
// lookahead (BE) prefill chunks are co-batched with LC decode rows; L311-313
// and L305 define what each row attends to.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "sa_internal.h"

namespace sa {

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct HostPlan {
    AttnPlan plan;
    std::vector<ReqMeta> dec, pre;
    int64_t total_q = 0;
    int64_t sum_decode_kv = 0;   // sum_j L_j over decode-like requests   (Eq. 1, alpha_d term)
    int64_t sum_prefill_A = 0;   // sum_j A_j over prefill requests       (Eq. 1, alpha_p term)
    bool use_tc5 = false;
    Tc5Schedule sched;            // tcgen05 path: parts per persistent CTA, merges of split items
    std::vector<int32_t> pre_orig;  // prefill request -> index in the caller's request list
};

// The split of a request depends only on that request (never on its batch), so co-batching
// cannot change the bits of a row.
int32_t build_plan_uncached(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr,
                   HostPlan *hp, bool before_append = false) {
    if (!pool || n_req < 0) return SA_ERR_INVALID_ARG;
    if (n_req == 0) return SA_OK;
    if (!sids || !qo_indptr || qo_indptr[0] != 0 || n_req > pool->cfg.max_sessions) return SA_ERR_INVALID_ARG;
    const int G = pool->G, Hq = pool->cfg.num_q_heads, Hkv = pool->cfg.num_kv_heads;
    hp->use_tc5 = tc5_supported(pool);  // every supported shape (head_dim 64 / 128, page 16 / 64) has a tcgen05 instantiation
    if (!hp->use_tc5) return SA_ERR_UNSUPPORTED;
    const int tile_m = kTc5TileM;
    std::vector<std::pair<ReqMeta, int32_t>> pre;
    for (int r = 0; r < n_req; ++r) {
        const int32_t sid = sids[r];
        if (sid < 0 || size_t(sid) >= pool->sessions.size() || !pool->sessions[size_t(sid)].open) return SA_ERR_INVALID_ARG;
        const int64_t n = int64_t(qo_indptr[r + 1]) - qo_indptr[r];
        if (n < 0) return SA_ERR_INVALID_ARG;
        const int64_t kv = pool->sessions[size_t(sid)].len + (before_append ? n : 0);
        if (n > kv) return SA_ERR_INVALID_ARG;  // the request's own tokens must already be appended
        if (n == 0) continue;
        ReqMeta m{};
        m.sid = sid;
        m.q_start = qo_indptr[r];
        m.q_len = int32_t(n);
        m.kv_len = int32_t(kv);
        if (n * G <= 16) {
            m.n_splits = int32_t((kv + kDecodeSplitKeys - 1) / kDecodeSplitKeys);
            hp->dec.push_back(m);
            hp->sum_decode_kv += kv * n;
        } else {
            m.n_tiles = int32_t((n * G + tile_m - 1) / tile_m);
            pre.push_back(std::make_pair(m, int32_t(r)));
            hp->sum_prefill_A += n * (kv - n) + n * (n + 1) / 2;
        }
    }
    hp->total_q = qo_indptr[n_req];
    // prefill: longest context first (its tiles carry the most work)
    std::stable_sort(pre.begin(), pre.end(), [](const std::pair<ReqMeta, int32_t> &a, const std::pair<ReqMeta, int32_t> &b) {
        return a.first.kv_len > b.first.kv_len;
    });
    for (const auto &pr : pre) {
        hp->pre.push_back(pr.first);
        hp->pre_orig.push_back(pr.second);
    }
    int64_t items = 0, parts = 0, rows = 0;
    for (ReqMeta &m : hp->dec) {
        m.item_begin = int32_t(items);
        m.part_begin = int32_t(parts);
        items += int64_t(Hkv) * m.n_splits;
        parts += int64_t(m.n_splits) * m.q_len * Hq;
        rows += int64_t(m.q_len) * Hq;
    }
    if (items > INT32_MAX || parts > INT32_MAX) return SA_ERR_UNSUPPORTED;
    hp->plan.n_dec = int32_t(hp->dec.size());
    hp->plan.dec_items = int32_t(items);
    hp->plan.part_rows = parts;
    hp->plan.dec_rows = rows;
    items = 0;
    for (ReqMeta &m : hp->pre) {
        m.item_begin = int32_t(items);
        items += int64_t(Hkv) * m.n_tiles;
    }
    if (items > INT32_MAX) return SA_ERR_UNSUPPORTED;
    hp->plan.n_pre = int32_t(hp->pre.size());
    hp->plan.pre_items = int32_t(items);
    if (!hp->pre.empty()) {
        tc5_schedule(hp->pre, G, Hkv, pool->num_sms, &hp->sched);
        hp->plan.pre_items = int32_t(hp->sched.parts.size());
    }
    return SA_OK;
}

}  // namespace

// The plan of the last batch planned on this pool.  sa_mixed_attention_workspace_bytes and the sa_mixed_attention call
// that follows it name the same batch on unchanged sessions: the second of them takes the plan (classes, splits,
// the stream-K schedule: 10-80 us of host time for a chunked batch) from here instead of building it again.
struct PlanCache {
    bool valid = false;
    bool before_append = false;
    std::vector<int32_t> sids, indptr;
    std::vector<int64_t> lens;  // session lengths the plan was built on
    HostPlan hp;
};

namespace {

int32_t build_plan(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr, const HostPlan **out,
                   bool before_append = false) {
    static const HostPlan empty;
    *out = &empty;
    if (!pool || n_req < 0) return SA_ERR_INVALID_ARG;
    if (n_req == 0) return SA_OK;
    if (!sids || !qo_indptr || n_req > pool->cfg.max_sessions) return SA_ERR_INVALID_ARG;
    PlanCache &pc = *pool->plan_cache;
    bool hit = pc.valid && pc.before_append == before_append && pc.sids.size() == size_t(n_req);
    for (int r = 0; hit && r < n_req; ++r) {
        const int32_t sid = sids[r];
        hit = sid == pc.sids[size_t(r)] && qo_indptr[r + 1] == pc.indptr[size_t(r) + 1] && sid >= 0 &&
              size_t(sid) < pool->sessions.size() && pool->sessions[size_t(sid)].open &&
              pool->sessions[size_t(sid)].len == pc.lens[size_t(r)];
    }
    if (hit && qo_indptr[0] == 0) {
        *out = &pc.hp;
        return SA_OK;
    }
    pc.valid = false;
    pc.hp = HostPlan();
    const int32_t st = build_plan_uncached(pool, n_req, sids, qo_indptr, &pc.hp, before_append);
    if (st != SA_OK) return st;
    pc.before_append = before_append;
    pc.sids.assign(sids, sids + n_req);
    pc.indptr.assign(qo_indptr, qo_indptr + n_req + 1);
    pc.lens.resize(size_t(n_req));
    for (int r = 0; r < n_req; ++r) pc.lens[size_t(r)] = pool->sessions[size_t(sids[r])].len;
    pc.valid = true;
    *out = &pc.hp;
    return SA_OK;
}

// workspace: [decode partial O f32][decode partial lse f32][tcgen05 partial slots][tcgen05 schedule payload]
struct WsLayout {
    size_t off_part_lse, off_slots, off_sched, total;
};
WsLayout workspace_layout(const sa_kv_pool *pool, const HostPlan &hp) {
    const size_t D = size_t(pool->cfg.head_dim);
    WsLayout w;
    w.off_part_lse = align_up(size_t(hp.plan.part_rows) * D * 4, 256);
    w.off_slots = w.off_part_lse + align_up(size_t(hp.plan.part_rows) * 4, 256);
    w.off_sched = w.off_slots + align_up(size_t(hp.sched.n_slots) * kTc5SlotBytes, 256);
    w.total = w.off_sched + align_up(hp.sched.parts.empty() ? 0 : hp.sched.payload_bytes(), 256) + 256;
    return w;
}
size_t workspace_need(const sa_kv_pool *pool, const HostPlan &hp) { return workspace_layout(pool, hp).total; }

void write_sched_payload(const Tc5Schedule &sc, char *dst) {
    const size_t off_parts = (sc.cta_begin.size() * 4 + 31) / 32 * 32;
    memset(dst, 0, off_parts);
    memcpy(dst, sc.cta_begin.data(), sc.cta_begin.size() * 4);
    if (!sc.parts.empty()) memcpy(dst + off_parts, sc.parts.data(), sc.parts.size() * sizeof(Tc5Part));
    if (!sc.merges.empty())
        memcpy(dst + off_parts + sc.parts.size() * sizeof(Tc5Part), sc.merges.data(), sc.merges.size() * sizeof(Tc5Merge));
}

}  // namespace

PlanCache *plan_cache_new() { return new (std::nothrow) PlanCache(); }
void plan_cache_delete(PlanCache *pc) { delete pc; }

int32_t attention_workspace_after_append(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                         const int32_t *qo_indptr, size_t *out_bytes) {
    const HostPlan *hpp = nullptr;
    const int32_t st = build_plan(pool, n_req, sids, qo_indptr, &hpp, true);
    if (st != SA_OK) return st;
    *out_bytes = workspace_need(pool, *hpp);
    return SA_OK;
}

}  // namespace sa

extern "C" int32_t sa_mixed_attention_workspace_bytes(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                                      const int32_t *qo_indptr, size_t *out_bytes) {
    if (!out_bytes) return SA_ERR_INVALID_ARG;
    const sa::HostPlan *hpp = nullptr;
    int32_t st = sa::build_plan(pool, n_req, sids, qo_indptr, &hpp);
    if (st != SA_OK) return st;
    *out_bytes = sa::workspace_need(pool, *hpp);
    return SA_OK;
}

extern "C" int32_t sa_mixed_attention_plan(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                           const int32_t *qo_indptr, int64_t *out_stats) {
    if (!out_stats) return SA_ERR_INVALID_ARG;
    const sa::HostPlan *hpp = nullptr;
    int32_t st = sa::build_plan(pool, n_req, sids, qo_indptr, &hpp);
    if (st != SA_OK) return st;
    const sa::HostPlan &hp = *hpp;
    out_stats[0] = hp.plan.n_dec;
    out_stats[1] = hp.plan.n_pre;
    out_stats[2] = hp.plan.dec_items;
    out_stats[3] = hp.plan.pre_items;
    out_stats[4] = hp.plan.part_rows;
    out_stats[5] = hp.sum_decode_kv;
    out_stats[6] = hp.sum_prefill_A;
    out_stats[7] = hp.use_tc5 ? 1 : 0;
    return SA_OK;
}

extern "C" int32_t sa_mixed_attention_schedule(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                               const int32_t *qo_indptr, int32_t *out_parts, int32_t cap,
                                               int64_t *out_summary) {
    if (!out_summary || cap < 0) return SA_ERR_INVALID_ARG;
    const sa::HostPlan *hpp = nullptr;
    int32_t st = sa::build_plan(pool, n_req, sids, qo_indptr, &hpp);
    if (st != SA_OK) return st;
    const sa::HostPlan &hp = *hpp;
    if (!sa::tc5_supported(pool)) return SA_ERR_UNSUPPORTED;
    const sa::Tc5Schedule &sc = hp.sched;
    out_summary[0] = pool->num_sms;
    out_summary[1] = int64_t(sc.parts.size());
    out_summary[2] = int64_t(sc.merges.size());
    out_summary[3] = sc.n_slots;
    out_summary[4] = sc.total_units;
    out_summary[5] = sc.makespan;
    if (out_parts) {
        const size_t n = std::min(size_t(cap), sc.parts.size());
        for (size_t i = 0; i < n; ++i) {
            const sa::Tc5Part &p = sc.parts[i];
            int32_t *o = out_parts + 8 * i;
            o[0] = p.cta;
            o[1] = hp.pre_orig[size_t(p.req)];
            o[2] = p.g;
            o[3] = p.tile;
            o[4] = p.u0;
            o[5] = p.u1;
            o[6] = p.n_kv;
            o[7] = p.slot;
        }
    }
    return SA_OK;
}

extern "C" int32_t sa_mixed_attention(sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr,
                                      const void *q, void *out, float *lse, float sm_scale, void *workspace,
                                      size_t workspace_bytes, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    using namespace sa;
    const HostPlan *hpp = nullptr;
    int32_t st = build_plan(pool, n_req, sids, qo_indptr, &hpp);
    if (st != SA_OK) return st;
    const HostPlan &hp = *hpp;
    if (pool->host_only) return SA_ERR_CUDA;
    pool->last_launches = 0;
    if (hp.plan.n_dec + hp.plan.n_pre == 0) return SA_OK;
    if (!q || !out) return SA_ERR_INVALID_ARG;
    const WsLayout wl = workspace_layout(pool, hp);
    const bool needs_ws = hp.plan.part_rows > 0 || !hp.sched.parts.empty();
    if (needs_ws && (!workspace || workspace_bytes < wl.total)) return SA_ERR_WORKSPACE_TOO_SMALL;
    if (!(sm_scale > 0.f)) sm_scale = 1.0f / sqrtf(float(pool->cfg.head_dim));
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    uintptr_t w = (reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255);

    float *part_o = reinterpret_cast<float *>(w);
    float *part_lse = reinterpret_cast<float *>(w + wl.off_part_lse);
    // a small decode-only call (the latency-critical one) carries its requests in the kernel parameters: no upload launch
    if (hp.pre.empty() && hp.dec.size() <= size_t(kInlineReqs)) {
        const cudaError_t e0 = launch_flash_decode(pool, nullptr, hp.dec.data(), hp.plan, q, out, lse, sm_scale, part_o, part_lse,
                                                   stream, &pool->last_launches);
        return e0 == cudaSuccess ? SA_OK : SA_ERR_CUDA;
    }
    // otherwise the per-call metadata [decode ReqMeta][prefill ReqMeta][tcgen05 schedule] goes through the pinned slab
    // ring; a schedule too long for the slab goes through the pool's growable pinned buffer into the workspace
    char *mh = nullptr, *md = nullptr;
    const size_t dec_bytes = sizeof(ReqMeta) * hp.dec.size(), pre_bytes = sizeof(ReqMeta) * hp.pre.size();
    st = acquire_meta(pool, dec_bytes + pre_bytes, &mh, &md);
    if (st != SA_OK) return st;
    const size_t sched_bytes = hp.sched.parts.empty() ? 0 : hp.sched.payload_bytes();
    const size_t off_sched = align_up(dec_bytes + pre_bytes, 32);
    if (dec_bytes) memcpy(mh, hp.dec.data(), dec_bytes);
    if (pre_bytes) memcpy(mh + dec_bytes, hp.pre.data(), pre_bytes);
    const char *sched_dev = nullptr;
    size_t slab_used = dec_bytes + pre_bytes;
    if (sched_bytes > 0) {
        if (off_sched + sched_bytes <= pool->meta_slab_bytes) {
            write_sched_payload(hp.sched, mh + off_sched);
            sched_dev = md + off_sched;
            slab_used = off_sched + sched_bytes;
        } else {
            char *big = nullptr;
            st = acquire_big_meta(pool, sched_bytes, &big);
            if (st != SA_OK) return st;
            write_sched_payload(hp.sched, big);
            char *dst = reinterpret_cast<char *>(w + wl.off_sched);
            if (commit_big_meta(pool, dst, sched_bytes, stream) != SA_OK) return SA_ERR_CUDA;
            sched_dev = dst;
        }
    }
    int meta_slot = 0;
    if (commit_meta_deferred(pool, nullptr, slab_used, stream, &meta_slot) != SA_OK) return SA_ERR_CUDA;
    const ReqMeta *dec_dev = reinterpret_cast<const ReqMeta *>(md);
    const ReqMeta *pre_dev = reinterpret_cast<const ReqMeta *>(md + dec_bytes);

    char *tc5_partials = reinterpret_cast<char *>(w + wl.off_slots);

    // Latency-critical rows first (Alg. 2 lines 3-6: decode requests are admitted before any prefill
    // chunk because they are the latency-critical class): the decode rows' outputs are complete after the HBM-bound
    // decode kernel (whose last splits merge), before the best-effort lookahead chunks' tensor-bound kernel has started.  The two
    // classes write disjoint rows and disjoint workspace regions, so the order does not change any bit.
    cudaError_t e;
    e = launch_flash_decode(pool, dec_dev, nullptr, hp.plan, q, out, lse, sm_scale, part_o, part_lse, stream, &pool->last_launches);
    if (e != cudaSuccess) return SA_ERR_CUDA;
    e = launch_prefill_tc5(pool, pre_dev, hp.plan, hp.sched, sched_dev, tc5_partials, hp.total_q, q, out, lse, sm_scale,
                           stream, &pool->last_launches);
    if (e != cudaSuccess) return SA_ERR_CUDA;
    return meta_mark(pool, meta_slot, stream);  // the pinned slab is free again when everything above has run
}
