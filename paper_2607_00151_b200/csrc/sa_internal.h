// sa_internal.h -- internal declarations shared by the translation units of libsmoothagent.so.
// Not part of the ABI (that is include/smoothagent.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "smoothagent.h"

namespace sa {

constexpr int kMetaRing = 8;            // per-call metadata slabs in flight
constexpr int kDecodeSplitKeys = 1024;  // split-KV granularity of decode-like rows (logical keys)
constexpr int kLegacyTileM = 64;        // packed rows per CTA of the mma.sync prefill kernel
constexpr int kTc5TileM = 256;          // packed rows per CTA of the tcgen05 prefill kernel
constexpr int kMaxChunkLatency = 2048;  // sa_latency_table prefill chunk size

// One request of a hot call as the kernels see it (device copy lives in the metadata ring).
struct ReqMeta {
    int32_t sid;         // session id -> row of the device block table
    int32_t q_start;     // first row of the request in the packed [T, H, D] arrays
    int32_t q_len;       // query rows (append: tokens appended)
    int32_t kv_len;      // attention: cached tokens incl. own rows; append: position of row 0
    int32_t item_begin;  // first work item (CTA) of this request inside its kernel's grid
    int32_t n_splits;    // decode-like class: number of KV splits
    int32_t part_begin;  // decode-like class: first partial row ([split][token][head])
    int32_t n_tiles;     // prefill class: packed-row tiles per kv head
};

struct Session {
    bool open = false;
    int64_t len = 0;
    std::vector<int32_t> pages;
};

}  // namespace sa

struct sa_kv_pool {
    sa_kv_pool_config cfg;
    int32_t G = 1;
    int32_t log2_page = 0;
    int64_t max_pages_per_session = 0;
    bool host_only = true;

    // device carve-up of the caller's storage
    char *storage = nullptr;
    size_t storage_bytes = 0;
    void *k_base = nullptr;
    void *v_base = nullptr;
    int32_t *block_table = nullptr;  // [max_sessions][max_pages_per_session]
    float2 *rope_tab = nullptr;      // [D/2] (hi, lo) of theta_m / (2 pi)
    char *meta_dev = nullptr;        // [kMetaRing][meta_slab_bytes]
    size_t meta_slab_bytes = 0;
    int64_t stride_page = 0, stride_head = 0, stride_slot = 0;

    // host side
    char *meta_host = nullptr;  // pinned, same shape as meta_dev
    cudaEvent_t meta_event[sa::kMetaRing] = {};
    bool meta_event_used[sa::kMetaRing] = {};
    int meta_next = 0;
    std::vector<int32_t> free_pages;  // stack: back() is handed out next
    std::vector<sa::Session> sessions;
    int32_t last_launches = 0;
    int32_t num_sms = 148;

    // tcgen05 prefill kernel: TMA descriptors over the K and V page arrays (filled at create)
    alignas(64) unsigned char tmap_k[128];
    alignas(64) unsigned char tmap_v[128];
    bool tc5_ready = false;
};

namespace sa {

// Reserve the next metadata slab (host pinned + device twin); waits for the slab's previous
// copy if it is still in flight.  commit_meta enqueues the H2D copy of `bytes` bytes.
int32_t acquire_meta(sa_kv_pool *pool, char **host, char **dev);
int32_t commit_meta(sa_kv_pool *pool, size_t bytes, cudaStream_t stream);

// --- kernel launchers (each returns a cudaError_t from the launch) ---
cudaError_t launch_rope_append(const sa_kv_pool *pool, const ReqMeta *reqs_dev, int32_t n_req,
                               int64_t total_rows, const void *k, const void *v, void *q,
                               cudaStream_t stream, int32_t *launches);

struct AttnPlan {
    int32_t n_dec = 0, n_pre = 0;        // requests per class
    int32_t dec_items = 0, pre_items = 0;  // CTAs per class
    int64_t part_rows = 0;               // decode-like partial rows ([split][token][head])
    int64_t dec_rows = 0;                // decode-like (token, head) rows to merge
};

cudaError_t launch_flash_decode(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const AttnPlan &plan,
                                const void *q, void *out, float *lse, float sm_scale, float *part_o,
                                float *part_lse, cudaStream_t stream, int32_t *launches);
cudaError_t launch_flash_prefill_legacy(const sa_kv_pool *pool, const ReqMeta *reqs_dev,
                                        const AttnPlan &plan, const void *q, void *out, float *lse,
                                        float sm_scale, cudaStream_t stream, int32_t *launches);

// tcgen05 path (sa_prefill_tc5.cu)
int32_t tc5_init(sa_kv_pool *pool);  // builds the TMA descriptors; SA_OK or SA_ERR_CUDA
bool tc5_supported(const sa_kv_pool *pool);
cudaError_t launch_prefill_tc5(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const AttnPlan &plan,
                               int64_t total_q, const void *q, void *out, float *lse, float sm_scale,
                               cudaStream_t stream, int32_t *launches);

}  // namespace sa
