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
constexpr int kTc5TileM = 256;          // packed rows per CTA of the tcgen05 prefill kernel
constexpr int kMaxChunkLatency = 2048;  // sa_latency_table prefill chunk size
constexpr int kTc5KeysPerUnit = 128;    // one schedule unit of the tcgen05 kernel = one 128-key KV tile of an item
constexpr int kTc5FixedCost = 3;        // per-part overhead (Q load, first QK, epilogue) in schedule units
constexpr int kTc5MinPart = 4;          // never cut a part shorter than this many units
// one partial result of a split item: unnormalised O f32 [256][128], then (m * scale_log2, l) f32 [256][2]
constexpr size_t kTc5SlotBytes = size_t(kTc5TileM) * 128 * 4 + size_t(kTc5TileM) * 2 * 4;

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

// Metadata of a small append carried in the kernel parameters (no upload launch, no block-table launch).
constexpr int kInlineReqs = 64;
constexpr int kInlinePages = 384;
struct InlineAppendMeta {
    ReqMeta reqs[kInlineReqs];     // as in the slab: kv_len = position of the first new token, item_begin / n_splits /
    int32_t pages[kInlinePages];   // part_begin = the request's slice of `pages` and the block-table index it starts at
    int32_t n_req, n_list, used, pad;
};

// The requests of a small decode-only attention call, carried in the kernel parameters.
struct InlineReqs {
    ReqMeta reqs[kInlineReqs];
};

// Metadata of a captured decode step (sa_decode_step_*): a pinned host slab the host rewrites between replays and a
// device twin the step's first kernel refreshes.  Layout: [StepHeader][ReqMeta x cap][StepAppend x cap].
struct StepHeader {
    int32_t n_req;    // requests of this step (<= cap)
    int32_t n_items;  // decode work items = sum over requests of Hkv * n_splits
    int32_t pad[6];
};
struct StepAppend {
    int32_t sid, pos, page, pad;  // the request's new token: position in the session, page that holds its slot
};
__host__ __device__ inline size_t step_append_offset(int32_t cap) { return sizeof(StepHeader) + sizeof(ReqMeta) * size_t(cap); }
__host__ __device__ inline size_t step_slab_bytes(int32_t cap) { return step_append_offset(cap) + sizeof(StepAppend) * size_t(cap); }

// tcgen05 prefill kernel: one persistent CTA per SM walks a list of parts.  An item is (request, kv
// head, 256 packed rows); a part is the KV-tile range [u0, u1) of an item.  slot < 0: the part is the
// whole item and writes the output directly; otherwise it writes partial slot `slot` and the merge
// kernel combines the item's parts (consecutive slots, KV order).
struct Tc5Part {
    int32_t req;    // index into the prefill ReqMeta array of the call
    int32_t g;      // kv head
    int32_t tile;   // 256-row tile of the request's packed rows
    int32_t u0, u1; // KV tiles [u0, u1) of the item's n_kv
    int32_t slot;   // partial slot, or -1
    int32_t n_kv;   // KV tiles of the whole item
    int32_t cta;    // CTA that runs it (host-side bookkeeping)
};
struct Tc5Merge {
    int32_t req, g, tile, slot0, n_parts, pad0, pad1, pad2;
};
struct Tc5Schedule {
    std::vector<int32_t> cta_begin;  // [n_cta + 1] into parts
    std::vector<Tc5Part> parts;      // grouped by CTA, execution order
    std::vector<Tc5Merge> merges;
    int32_t n_slots = 0;
    int64_t total_units = 0;         // sum of n_kv over items
    int64_t makespan = 0;            // largest CTA load in units (incl. fixed costs)
    size_t payload_bytes() const {
        return (cta_begin.size() * 4 + 31) / 32 * 32 + parts.size() * sizeof(Tc5Part) + merges.size() * sizeof(Tc5Merge);
    }
};
// Static schedule of the prefill items of a call over n_cta persistent CTAs (sa_tc5_schedule.cu).
void tc5_schedule(const std::vector<ReqMeta> &pre, int G, int Hkv, int n_cta, Tc5Schedule *out);

struct PlanCache;  // last attention plan of a pool (sa_attention.cu)
PlanCache *plan_cache_new();
void plan_cache_delete(PlanCache *pc);

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
    int32_t *tickets = nullptr;      // [max_sessions][Hkv] arrival counters of the split-KV decode kernel (zero between kernels)
    char *meta_dev = nullptr;        // [kMetaRing][meta_slab_bytes]
    size_t meta_slab_bytes = 0;
    int64_t stride_page = 0, stride_head = 0, stride_slot = 0;

    // host side
    char *meta_host = nullptr;  // pinned, same shape as meta_dev
    cudaEvent_t meta_event[sa::kMetaRing] = {};
    bool meta_event_used[sa::kMetaRing] = {};
    int meta_next = 0;
    char *big_host = nullptr;   // pinned, grown on demand: metadata too long for a slab (long tcgen05 schedules)
    size_t big_cap = 0;
    cudaEvent_t big_event = nullptr;
    bool big_event_used = false;
    std::vector<int32_t> free_pages;  // stack: back() is handed out next
    std::vector<int32_t> page_ref;    // sessions holding each page (forked sessions share the retained prefix's pages)
    std::vector<sa::Session> sessions;
    int32_t last_launches = 0;
    int32_t num_sms = 148;
    sa::PlanCache *plan_cache = nullptr;  // owned; the one piece of state the const planning calls update

    // tcgen05 prefill kernel: TMA descriptors over the K and V page arrays (filled at create)
    alignas(64) unsigned char tmap_k[128];
    alignas(64) unsigned char tmap_v[128];
    bool tc5_ready = false;
};

namespace sa {

// Every entry point that touches the device runs on the POOL's device (cfg.device), whatever device is current in the
// calling thread, and leaves the caller's current device as it found it.  Host-only pools and null pools: a no-op.
struct DeviceGuard {
    int prev = -1;
    bool switched = false, ok = true;
    explicit DeviceGuard(const sa_kv_pool *pool) {
        if (pool && !pool->host_only) enter(pool->cfg.device);
    }
    explicit DeviceGuard(int device) { enter(device); }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;

  private:
    void enter(int device) {
        if (cudaGetDevice(&prev) != cudaSuccess) {
            ok = false;
            return;
        }
        if (prev != device) {
            ok = cudaSetDevice(device) == cudaSuccess;
            switched = ok;
        }
    }
};

// Reserve the next metadata slab (host pinned + device twin); waits for the slab's previous
// copy if it is still in flight.  commit_meta enqueues the H2D copy of `bytes` bytes.
// `bytes`: what the caller is about to write into the slab; more than a slab holds is refused (SA_ERR_UNSUPPORTED)
// before anything is touched, never written past the slab's end.
int32_t acquire_meta(sa_kv_pool *pool, size_t bytes, char **host, char **dev);
int32_t commit_meta(sa_kv_pool *pool, size_t bytes, cudaStream_t stream);
// Same slab, but the bytes go to `dev_dst` (a block-table row) instead of the slab's device twin.
int32_t commit_meta_to(sa_kv_pool *pool, void *dev_dst, size_t bytes, cudaStream_t stream);
// commit_meta without the event that frees the slab (dev_dst nullptr: the slab's device twin); the caller records it
// with meta_mark once the kernels that read the metadata are enqueued
int32_t commit_meta_deferred(sa_kv_pool *pool, void *dev_dst, size_t bytes, cudaStream_t stream, int *slot);
int32_t meta_mark(sa_kv_pool *pool, int slot, cudaStream_t stream);
// Page bookkeeping: a page returns to the free list when its last holder lets go of it.
int32_t take_page(sa_kv_pool *pool);
void release_page(sa_kv_pool *pool, int32_t page);
// Device copy of one whole page (K and V, all heads) on `stream`: copy-on-write of a shared partial page.
cudaError_t copy_page_async(const sa_kv_pool *pool, int32_t dst_page, int32_t src_page, cudaStream_t stream);
// Metadata that does not fit a slab: one growable pinned buffer (waits for its previous copy),
// copied to a device address of the caller's workspace.
int32_t acquire_big_meta(sa_kv_pool *pool, size_t bytes, char **host);
int32_t commit_big_meta(sa_kv_pool *pool, void *dev_dst, size_t bytes, cudaStream_t stream);

#ifdef __CUDACC__
// Launch with programmatic stream serialization: the grid may be staged (and run whatever precedes its
// griddepcontrol.wait) while the kernel before it in the stream is still running.  Every kernel launched this way
// executes griddepcontrol.wait before it reads or writes anything that is ordered by the stream.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// (cos, sin) of pos * theta_m from the pool's table u = (hi, lo) of theta_m / (2 pi) (reading R9):
// the position is an exact fp32 integer (< 2^24), the product pos * u is formed error-free, whole
// turns are dropped and sincospif evaluates the fraction.
__device__ __forceinline__ float2 rope_cos_sin(int32_t pos, float2 u) {
    const float p = float(pos);
    const float ph = p * u.x;
    float pl = fmaf(p, u.x, -ph);              // exact error of the product
    pl = fmaf(p, u.y, pl);
    const float fr = (ph - rintf(ph)) + pl;    // turns, |fr| <= 0.5 (+ tiny)
    float sn, cs;
    sincospif(2.0f * fr, &sn, &cs);
    return make_float2(cs, sn);
}
#endif

// Host half of an append: validation, page allocation, metadata upload, block-table update (sa_append.cu).
// im (nullable): if the call is small enough its metadata is returned there (im->used = 1) instead of going to the
// device, and the caller's kernel updates the block table itself.
int32_t append_prepare(sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr,
                       bool have_data, cudaStream_t stream, const ReqMeta **reqs_dev_out, int64_t *total_out,
                       InlineAppendMeta *im = nullptr);

// --- kernel launchers (each returns a cudaError_t from the launch) ---
cudaError_t launch_rope_append(const sa_kv_pool *pool, const ReqMeta *reqs_dev, int32_t n_req,
                               int64_t total_rows, const void *k, const void *v, void *q,
                               cudaStream_t stream, int32_t *launches);

// the step's first kernel: slab_host -> slab_dev, then RoPE + placement of one token per request (sa_append.cu)
cudaError_t launch_step_append(const sa_kv_pool *pool, const void *slab_host, void *slab_dev, int32_t cap, const void *k,
                               const void *v, void *q, cudaStream_t stream, int32_t *launches);
// shared-memory opt-in of the step's decode kernel for the current device (so that nothing but launches happens later)
cudaError_t flash_loop_prepare(const sa_kv_pool *pool);

struct AttnPlan {
    int32_t n_dec = 0, n_pre = 0;        // requests per class
    int32_t dec_items = 0, pre_items = 0;  // CTAs per class
    int64_t part_rows = 0;               // decode-like partial rows ([split][token][head])
    int64_t dec_rows = 0;                // decode-like (token, head) rows to merge
};

cudaError_t launch_flash_decode(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const ReqMeta *reqs_host,
                                const AttnPlan &plan, const void *q, void *out, float *lse, float sm_scale,
                                float *part_o, float *part_lse, cudaStream_t stream, int32_t *launches,
                                int loop_ctas = 0, const int32_t *dyn = nullptr);
// dense operators of the layer (sa_gemm_tc5.cu); each returns an SA_* status
int32_t gemm_plain(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N, int32_t K,
                   void *splitk_ws, size_t splitk_bytes, cudaStream_t stream, int32_t *launches);
int32_t gemm_swiglu(const void *x, const void *w_gate, const void *w_up, void *act, int64_t M, int32_t F, int32_t K,
                    void *splitk_ws, size_t splitk_bytes, cudaStream_t stream, int32_t *launches);
size_t gemm_plain_splitk_bytes(int64_t M, int32_t N, int32_t K);
size_t gemm_swiglu_splitk_bytes(int64_t M, int32_t F, int32_t K);
int32_t rmsnorm(const void *x, const void *w, float eps, void *y, int64_t M, int32_t H, cudaStream_t stream);
size_t qkv_workspace_bytes(const sa_kv_pool *pool, int64_t total);
int32_t qkv_rope_append_device(sa_kv_pool *pool, const ReqMeta *reqs_dev, int32_t n_req, int64_t total, const void *h,
                               const void *w_qkv, int32_t hidden, void *q_out, void *workspace, size_t workspace_bytes,
                               cudaStream_t stream);
// sa_mixed_attention's workspace need for a batch whose q_r tokens are still to be appended (sa_attention.cu)
int32_t attention_workspace_after_append(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                         const int32_t *qo_indptr, size_t *out_bytes);

// cuTensorMapEncodeTiled resolved through the runtime (no link against libcuda); nullptr if unavailable
void *tensor_map_encode_fn();

// tcgen05 path (sa_prefill_tc5.cu)
int32_t tc5_init(sa_kv_pool *pool);  // builds the TMA descriptors; SA_OK or SA_ERR_CUDA
bool tc5_supported(const sa_kv_pool *pool);
// sched_dev: the schedule payload on the device ([cta_begin][parts][merges]); partials: n_slots slots
cudaError_t launch_prefill_tc5(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const AttnPlan &plan,
                               const Tc5Schedule &sched, const char *sched_dev, char *partials,
                               int64_t total_q, const void *q, void *out, float *lse, float sm_scale,
                               cudaStream_t stream, int32_t *launches);

}  // namespace sa
