// sa_latency.cu -- sa_latency_table: measured attention time vs prefill-chunk tokens and decode
// batch size.  PAPER.md Eq. 1 (L349-353) models a mixed batch as
// T_GEMM(M) + alpha_d * sum L_j + alpha_p * sum A_j with "profiled" coefficients (L309, L319) and
// an "offline-profiled" table (L303); Fig. 15 (L476) checks such a model.  This call is the
// profiling run on this library's kernels.  Not a hot call: it allocates and synchronises.
#include <cuda_bf16.h>

#include <algorithm>
#include <vector>

#include "sa_internal.h"

namespace {

// counter-based generator: splitmix64 of (seed, index)
inline uint64_t mix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

// uniform bf16 in [-0.15, 0.15): about the spread of N(0,1)/sqrt(128), the bench distribution
__global__ void fill_uniform_kernel(__nv_bfloat16 *p, size_t n, uint32_t salt) {
    for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < n; i += size_t(gridDim.x) * blockDim.x) {
        uint32_t x = uint32_t(i) * 2654435761u + salt;
        x ^= x >> 15;
        x *= 2246822519u;
        x ^= x >> 13;
        p[i] = __float2bfloat16((float(x >> 8) * (1.0f / 16777216.0f) - 0.5f) * 0.3f);
    }
}

// Scratch sessions of the run (closed on every exit path) and a bump allocator over the CALLER's workspace: this call
// allocates no device memory of its own.
struct Scratch {
    std::vector<int32_t> sids;
    sa_kv_pool *pool = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    char *base = nullptr;
    size_t cap = 0, used = 0;
    ~Scratch() {
        for (int32_t s : sids) sa_kv_session_close(pool, s);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    }
    void *alloc(size_t bytes) {
        const size_t b = (std::max<size_t>(bytes, 256) + 255) / 256 * 256;
        if (used + b > cap) return nullptr;
        void *p = base + used;
        used += b;
        return p;
    }
};
inline size_t up256(size_t b) { return (std::max<size_t>(b, 256) + 255) / 256 * 256; }
constexpr size_t kFlushBytes = size_t(256) << 20;  // larger than the 126 MB L2

constexpr int kFillTok = 4096;

// Bring session `sid` to `len` tokens by appending pieces of the shared source buffer.
int32_t fill_session(sa_kv_pool *pool, int32_t sid, int64_t len, const void *k, const void *v, cudaStream_t st) {
    int64_t cur = 0;
    int32_t rc = sa_kv_session_query(pool, sid, &cur, nullptr, nullptr);
    while (rc == SA_OK && cur < len) {
        const int32_t n = int32_t(std::min<int64_t>(kFillTok, len - cur));
        const int32_t indptr[2] = {0, n};
        rc = sa_rope_kv_append(pool, 1, &sid, indptr, k, v, nullptr, st);
        cur += n;
    }
    return rc;
}

}  // namespace

namespace {

struct TableGeom {
    int32_t d_max = 0, p_max = 0, c_max = 0;
    std::vector<int64_t> ctx;   // contexts of the decode rows
    int64_t need_pages = 0;
};

// argument checks and the geometry of the run, shared by the sizing call and the run itself
int32_t table_geom(const sa_kv_pool *pool, const int32_t *prefill_tokens, int32_t n_p, const int32_t *decode_batch, int32_t n_d,
                   int64_t prefill_prefix_len, int64_t decode_ctx_lo, int64_t decode_ctx_hi, uint64_t seed, TableGeom *g) {
    if (!pool || !prefill_tokens || !decode_batch || n_p <= 0 || n_d <= 0 || prefill_prefix_len < 0 || decode_ctx_lo < 1 ||
        decode_ctx_hi < decode_ctx_lo)
        return SA_ERR_INVALID_ARG;
    const sa_kv_pool_config &c = pool->cfg;
    for (int i = 0; i < n_d; ++i) {
        if (decode_batch[i] < 0) return SA_ERR_INVALID_ARG;
        g->d_max = std::max(g->d_max, decode_batch[i]);
    }
    for (int i = 0; i < n_p; ++i) {
        if (prefill_tokens[i] < 0) return SA_ERR_INVALID_ARG;
        g->p_max = std::max(g->p_max, prefill_tokens[i]);
    }
    g->c_max = (g->p_max + sa::kMaxChunkLatency - 1) / sa::kMaxChunkLatency;
    if (decode_ctx_hi > c.max_session_tokens || prefill_prefix_len + sa::kMaxChunkLatency > c.max_session_tokens)
        return SA_ERR_INVALID_ARG;
    if (g->d_max + g->c_max > c.max_sessions) return SA_ERR_OUT_OF_SESSIONS;
    g->ctx.assign(size_t(g->d_max), 0);
    const int B = c.page_size;
    for (int j = 0; j < g->d_max; ++j) {
        g->ctx[size_t(j)] = decode_ctx_lo + int64_t(mix64(seed * 0x100000001B3ull + uint64_t(j)) % uint64_t(decode_ctx_hi - decode_ctx_lo + 1));
        g->need_pages += (g->ctx[size_t(j)] + B - 1) / B;
    }
    g->need_pages += int64_t(g->c_max) * ((prefill_prefix_len + sa::kMaxChunkLatency + B - 1) / B);
    return SA_OK;
}

// the requests of grid point (p prefill tokens, d decode rows) over the run's scratch sessions
void point_requests(int32_t p, int32_t d, const std::vector<int32_t> &pre_sids, const std::vector<int32_t> &dec_sids,
                    std::vector<int32_t> *sids, std::vector<int32_t> *indptr) {
    sids->clear();
    indptr->assign(1, 0);
    const int32_t n_chunks = (p + sa::kMaxChunkLatency - 1) / sa::kMaxChunkLatency;
    for (int j = 0; j < n_chunks; ++j) {
        sids->push_back(pre_sids[size_t(j)]);
        indptr->push_back(indptr->back() + std::min<int32_t>(sa::kMaxChunkLatency, p - j * sa::kMaxChunkLatency));
    }
    for (int j = 0; j < d; ++j) {
        sids->push_back(dec_sids[size_t(j)]);
        indptr->push_back(indptr->back() + 1);
    }
}

size_t fixed_buffers_bytes(const sa_kv_pool_config &c, const TableGeom &g) {
    const size_t kv_elems = size_t(kFillTok) * c.num_kv_heads * c.head_dim;
    const size_t q_elems = size_t(std::max<int64_t>(int64_t(g.p_max) + g.d_max, 1)) * c.num_q_heads * c.head_dim;
    return 2 * up256(kv_elems * 2) + 2 * up256(q_elems * 2) + up256(kFlushBytes);
}

}  // namespace

// The sessions the run will open are replayed on a host-only twin of the pool (same shape, same planner, no device), so
// the attention workspace of every grid point is the planner's own figure, not an estimate.
extern "C" int32_t sa_latency_table_workspace_bytes(const sa_kv_pool *pool, const int32_t *prefill_tokens, int32_t n_p,
                                                    const int32_t *decode_batch, int32_t n_d, int64_t prefill_prefix_len,
                                                    int64_t decode_ctx_lo, int64_t decode_ctx_hi, uint64_t seed,
                                                    size_t *out_bytes) {
    if (!out_bytes) return SA_ERR_INVALID_ARG;
    TableGeom g;
    int32_t rc = table_geom(pool, prefill_tokens, n_p, decode_batch, n_d, prefill_prefix_len, decode_ctx_lo, decode_ctx_hi, seed, &g);
    if (rc != SA_OK) return rc;
    sa_kv_pool_config c = pool->cfg;
    c.num_pages = std::max<int64_t>(g.need_pages, 1);
    c.max_sessions = std::max(g.d_max + g.c_max, 1);
    sa_kv_pool *twin = nullptr;
    rc = sa_kv_pool_create(&c, nullptr, 0, nullptr, &twin);
    if (rc != SA_OK) return rc;
    twin->num_sms = pool->num_sms;  // the tcgen05 schedule (and with it the partial slots) depends on the SM count
    std::vector<int32_t> dec_sids, pre_sids, sids, indptr;
    auto grow = [&](int32_t sid, int64_t len) {
        int64_t cur = 0;
        int32_t r = sa_kv_session_query(twin, sid, &cur, nullptr, nullptr);
        const int32_t ip[2] = {0, int32_t(len - cur)};
        return r == SA_OK && len > cur ? sa_rope_kv_append(twin, 1, &sid, ip, nullptr, nullptr, nullptr, nullptr) : r;
    };
    for (int j = 0; rc == SA_OK && j < g.d_max + g.c_max; ++j) {
        int32_t sid = -1;
        rc = sa_kv_session_open(twin, &sid);
        (j < g.d_max ? dec_sids : pre_sids).push_back(sid);
        if (rc == SA_OK && j < g.d_max) rc = grow(sid, g.ctx[size_t(j)]);
    }
    size_t ws_max = 0;
    for (int a = 0; rc == SA_OK && a < n_p; ++a) {
        const int32_t p = prefill_tokens[a];
        const int32_t n_chunks = (p + sa::kMaxChunkLatency - 1) / sa::kMaxChunkLatency;
        for (int j = 0; rc == SA_OK && j < n_chunks; ++j) {
            rc = sa_kv_session_truncate(twin, pre_sids[size_t(j)], 0);
            if (rc == SA_OK) rc = grow(pre_sids[size_t(j)], prefill_prefix_len + std::min<int32_t>(sa::kMaxChunkLatency, p - j * sa::kMaxChunkLatency));
        }
        for (int b = 0; rc == SA_OK && b < n_d; ++b) {
            point_requests(p, decode_batch[b], pre_sids, dec_sids, &sids, &indptr);
            size_t ws = 0;
            if (!sids.empty()) rc = sa_mixed_attention_workspace_bytes(twin, int32_t(sids.size()), sids.data(), indptr.data(), &ws);
            ws_max = std::max(ws_max, ws);
        }
    }
    sa_kv_pool_destroy(twin);
    if (rc != SA_OK) return rc;
    *out_bytes = fixed_buffers_bytes(pool->cfg, g) + up256(ws_max) + 256;
    return SA_OK;
}

extern "C" int32_t sa_latency_table(sa_kv_pool *pool, const int32_t *prefill_tokens, int32_t n_p,
                                    const int32_t *decode_batch, int32_t n_d, int64_t prefill_prefix_len,
                                    int64_t decode_ctx_lo, int64_t decode_ctx_hi, uint64_t seed, int32_t warmup,
                                    int32_t iters, float *out_ms, int64_t *out_sum_kv, void *workspace,
                                    size_t workspace_bytes, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    if (!out_ms || iters <= 0 || warmup < 0) return SA_ERR_INVALID_ARG;
    TableGeom g;
    {
        const int32_t rc = table_geom(pool, prefill_tokens, n_p, decode_batch, n_d, prefill_prefix_len, decode_ctx_lo, decode_ctx_hi, seed, &g);
        if (rc != SA_OK) return rc;
    }
    if (pool->host_only) return SA_ERR_CUDA;
    const sa_kv_pool_config &c = pool->cfg;
    const int32_t d_max = g.d_max, p_max = g.p_max, c_max = g.c_max;
    const std::vector<int64_t> &ctx = g.ctx;
    int64_t free_pages = 0;
    sa_kv_pool_free_pages(pool, &free_pages);
    if (g.need_pages > free_pages) return SA_ERR_OUT_OF_PAGES;
    if (!workspace || workspace_bytes < fixed_buffers_bytes(c, g) + 512) return SA_ERR_WORKSPACE_TOO_SMALL;

    cudaStream_t st = static_cast<cudaStream_t>(stream_);
    Scratch sc;
    sc.pool = pool;
    sc.base = reinterpret_cast<char *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
    sc.cap = workspace_bytes - size_t(sc.base - static_cast<char *>(workspace));
    if (cudaEventCreate(&sc.e0) != cudaSuccess || cudaEventCreate(&sc.e1) != cudaSuccess) return SA_ERR_CUDA;
    const size_t kv_elems = size_t(kFillTok) * c.num_kv_heads * c.head_dim;
    const int64_t t_max = int64_t(p_max) + d_max;
    const size_t q_elems = size_t(std::max<int64_t>(t_max, 1)) * c.num_q_heads * c.head_dim;
    auto *src_k = static_cast<__nv_bfloat16 *>(sc.alloc(kv_elems * 2));
    auto *src_v = static_cast<__nv_bfloat16 *>(sc.alloc(kv_elems * 2));
    auto *q = static_cast<__nv_bfloat16 *>(sc.alloc(q_elems * 2));
    void *out = sc.alloc(q_elems * 2);
    const size_t flush_bytes = kFlushBytes;
    void *flush = sc.alloc(flush_bytes);
    if (!src_k || !src_v || !q || !out || !flush) return SA_ERR_WORKSPACE_TOO_SMALL;
    const size_t used_fixed = sc.used;
    fill_uniform_kernel<<<1024, 256, 0, st>>>(src_k, kv_elems, 0x1234567u);
    fill_uniform_kernel<<<1024, 256, 0, st>>>(src_v, kv_elems, 0x89abcdeu);
    fill_uniform_kernel<<<1024, 256, 0, st>>>(q, q_elems, 0x2468aceu);
    if (cudaGetLastError() != cudaSuccess) return SA_ERR_CUDA;

    // decode sessions: shared by every grid point (batch d uses the first d of them)
    std::vector<int32_t> dec_sids;
    for (int j = 0; j < d_max; ++j) {
        int32_t sid = -1;
        int32_t rc = sa_kv_session_open(pool, &sid);
        if (rc != SA_OK) return rc;
        sc.sids.push_back(sid);
        dec_sids.push_back(sid);
        rc = fill_session(pool, sid, ctx[size_t(j)], src_k, src_v, st);
        if (rc != SA_OK) return rc;
    }
    std::vector<int32_t> pre_sids;
    for (int j = 0; j < c_max; ++j) {
        int32_t sid = -1;
        int32_t rc = sa_kv_session_open(pool, &sid);
        if (rc != SA_OK) return rc;
        sc.sids.push_back(sid);
        pre_sids.push_back(sid);
    }

    std::vector<float> times(static_cast<size_t>(iters));
    for (int a = 0; a < n_p; ++a) {
        // chunk sessions for this prefill size: each holds prefix + its own chunk
        const int32_t p = prefill_tokens[a];
        const int32_t n_chunks = (p + sa::kMaxChunkLatency - 1) / sa::kMaxChunkLatency;
        std::vector<int32_t> chunk_len(static_cast<size_t>(n_chunks));
        for (int j = 0; j < n_chunks; ++j) {
            chunk_len[size_t(j)] = std::min<int32_t>(sa::kMaxChunkLatency, p - j * sa::kMaxChunkLatency);
            int32_t rc = sa_kv_session_truncate(pool, pre_sids[size_t(j)], 0);
            if (rc == SA_OK) rc = fill_session(pool, pre_sids[size_t(j)], prefill_prefix_len + chunk_len[size_t(j)], src_k, src_v, st);
            if (rc != SA_OK) return rc;
        }
        for (int b = 0; b < n_d; ++b) {
            const int32_t d = decode_batch[b];
            std::vector<int32_t> sids, indptr;
            point_requests(p, d, pre_sids, dec_sids, &sids, &indptr);
            const int32_t n_req = int32_t(sids.size());
            float *cell = out_ms + size_t(a) * n_d + b;
            int64_t stats[8] = {0};
            if (n_req > 0) {
                int32_t rc = sa_mixed_attention_plan(pool, n_req, sids.data(), indptr.data(), stats);
                if (rc != SA_OK) return rc;
            }
            if (out_sum_kv) {
                out_sum_kv[(size_t(a) * n_d + b) * 2 + 0] = stats[5];
                out_sum_kv[(size_t(a) * n_d + b) * 2 + 1] = stats[6];
            }
            if (n_req == 0) {
                *cell = 0.f;
                continue;
            }
            size_t ws_bytes = 0;
            int32_t rc = sa_mixed_attention_workspace_bytes(pool, n_req, sids.data(), indptr.data(), &ws_bytes);
            if (rc != SA_OK) return rc;
            sc.used = used_fixed;  // every grid point reuses the region after the fixed buffers
            void *ws = sc.alloc(ws_bytes);
            if (!ws) return SA_ERR_WORKSPACE_TOO_SMALL;
            for (int it = 0; it < warmup + iters; ++it) {
                if (cudaMemsetAsync(flush, it & 0xff, flush_bytes, st) != cudaSuccess) return SA_ERR_CUDA;  // evict L2
                cudaEventRecord(sc.e0, st);
                rc = sa_mixed_attention(pool, n_req, sids.data(), indptr.data(), q, out, nullptr, 0.f, ws, ws_bytes, st);
                cudaEventRecord(sc.e1, st);
                if (rc != SA_OK) return rc;
                if (cudaEventSynchronize(sc.e1) != cudaSuccess) return SA_ERR_CUDA;
                float ms = 0.f;
                cudaEventElapsedTime(&ms, sc.e0, sc.e1);
                if (it >= warmup) times[size_t(it - warmup)] = ms;
            }
            std::sort(times.begin(), times.end());
            *cell = (iters & 1) ? times[size_t(iters / 2)] : 0.5f * (times[size_t(iters / 2 - 1)] + times[size_t(iters / 2)]);
        }
    }
    if (cudaStreamSynchronize(st) != cudaSuccess) return SA_ERR_CUDA;
    return SA_OK;
}
