// sa_layer.cu -- C-ABI entry points of the layer's dense operators (section 4
// "GEMM", L299-303) and of one whole decoder layer over a mixed batch; sa_gemm_table profiles
// T_GEMM(M), the "offline-profiled lookup table" of L303.  The kernels are in sa_gemm_tc5.cu.
#include <cuda_bf16.h>

#include <algorithm>
#include <vector>

#include "sa_internal.h"

namespace {

inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

struct LayerWs {
    size_t off_h, off_q, off_attn, off_x1, off_act, off_qkv, off_attn_ws, off_splitk, splitk_bytes, total;
};

LayerWs layer_ws(const sa_kv_pool *pool, const sa_layer_weights *L, int64_t T, size_t attn_ws) {
    const size_t t = size_t(T), H = size_t(L->hidden), QD = size_t(pool->cfg.num_q_heads) * pool->cfg.head_dim;
    LayerWs w;
    w.off_h = 0;
    w.off_q = w.off_h + up256(t * H * 2);
    w.off_attn = w.off_q + up256(t * QD * 2);
    w.off_x1 = w.off_attn + up256(t * QD * 2);
    w.off_act = w.off_x1 + up256(t * H * 2);
    w.off_qkv = w.off_act + up256(t * size_t(L->ffn) * 2);
    w.off_attn_ws = w.off_qkv + up256(sa::qkv_workspace_bytes(pool, T));
    w.off_splitk = w.off_attn_ws + up256(attn_ws) + 256;
    // split-K scratch of the output projection, the SwiGLU GEMM and the down projection (they run one after the other)
    w.splitk_bytes = std::max(std::max(sa::gemm_plain_splitk_bytes(T, L->hidden, int32_t(QD)), sa::gemm_swiglu_splitk_bytes(T, L->ffn, L->hidden)),
                              sa::gemm_plain_splitk_bytes(T, L->hidden, L->ffn));
    w.total = w.off_splitk + up256(w.splitk_bytes) + 512;
    return w;
}

int32_t check_layer(const sa_kv_pool *pool, const sa_layer_weights *L) {
    if (!pool || !L) return SA_ERR_INVALID_ARG;
    if (L->hidden <= 0 || L->ffn <= 0) return SA_ERR_INVALID_ARG;
    if (pool->cfg.head_dim != 128 || L->hidden % 64 != 0 || L->ffn % 64 != 0) return SA_ERR_UNSUPPORTED;
    return SA_OK;
}

__global__ void fill_small_kernel(__nv_bfloat16 *p, size_t n, uint32_t salt, float amp) {
    for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < n; i += size_t(gridDim.x) * blockDim.x) {
        uint32_t x = uint32_t(i) * 2654435761u + salt;
        x ^= x >> 15;
        x *= 2246822519u;
        x ^= x >> 13;
        p[i] = __float2bfloat16((float(x >> 8) * (1.0f / 16777216.0f) - 0.5f) * amp);
    }
}

}  // namespace

extern "C" int32_t sa_linear(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N,
                             int32_t K, void *stream) {
    return sa::gemm_plain(x, w, residual, y, M, N, K, nullptr, 0, static_cast<cudaStream_t>(stream), nullptr);
}

extern "C" int32_t sa_swiglu(const void *x, const void *w_gate, const void *w_up, void *act, int64_t M, int32_t F,
                             int32_t K, void *stream) {
    return sa::gemm_swiglu(x, w_gate, w_up, act, M, F, K, nullptr, 0, static_cast<cudaStream_t>(stream), nullptr);
}

extern "C" int32_t sa_linear_workspace_bytes(int64_t M, int32_t N, int32_t K, size_t *out_bytes) {
    if (!out_bytes || M < 0 || N <= 0 || K <= 0) return SA_ERR_INVALID_ARG;
    *out_bytes = sa::gemm_plain_splitk_bytes(M, N, K);
    return SA_OK;
}

extern "C" int32_t sa_linear_ws(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N, int32_t K,
                                void *workspace, size_t workspace_bytes, void *stream) {
    return sa::gemm_plain(x, w, residual, y, M, N, K, workspace, workspace_bytes, static_cast<cudaStream_t>(stream), nullptr);
}

extern "C" int32_t sa_swiglu_workspace_bytes(int64_t M, int32_t F, int32_t K, size_t *out_bytes) {
    if (!out_bytes || M < 0 || F <= 0 || K <= 0) return SA_ERR_INVALID_ARG;
    *out_bytes = sa::gemm_swiglu_splitk_bytes(M, F, K);
    return SA_OK;
}

extern "C" int32_t sa_swiglu_ws(const void *x, const void *w_gate, const void *w_up, void *act, int64_t M, int32_t F, int32_t K,
                                void *workspace, size_t workspace_bytes, void *stream) {
    return sa::gemm_swiglu(x, w_gate, w_up, act, M, F, K, workspace, workspace_bytes, static_cast<cudaStream_t>(stream), nullptr);
}

extern "C" int32_t sa_rmsnorm(const void *x, const void *w, float eps, void *y, int64_t M, int32_t H, void *stream) {
    return sa::rmsnorm(x, w, eps, y, M, H, static_cast<cudaStream_t>(stream));
}

extern "C" int32_t sa_qkv_rope_append_workspace_bytes(const sa_kv_pool *pool, int64_t total_tokens, size_t *out_bytes) {
    if (!pool || !out_bytes || total_tokens < 0) return SA_ERR_INVALID_ARG;
    *out_bytes = sa::qkv_workspace_bytes(pool, total_tokens);
    return SA_OK;
}

extern "C" int32_t sa_qkv_rope_append(sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr,
                                      const void *h, const void *w_qkv, int32_t hidden, void *q_out, void *workspace,
                                      size_t workspace_bytes, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    using namespace sa;
    if (!pool || n_req < 0 || hidden <= 0) return SA_ERR_INVALID_ARG;
    if (pool->cfg.head_dim != 128 || hidden % 64 != 0) return SA_ERR_UNSUPPORTED;
    if (n_req > 0 && qo_indptr && !pool->host_only) {
        const int64_t total = qo_indptr[n_req];
        if (total > 0 && (!h || !w_qkv || !q_out || !workspace || workspace_bytes < qkv_workspace_bytes(pool, total)))
            return total > 0 && workspace && workspace_bytes < qkv_workspace_bytes(pool, total) ? SA_ERR_WORKSPACE_TOO_SMALL
                                                                                         : SA_ERR_INVALID_ARG;
        if ((reinterpret_cast<uintptr_t>(h) | reinterpret_cast<uintptr_t>(w_qkv) | reinterpret_cast<uintptr_t>(q_out)) & 15)
            return SA_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const ReqMeta *reqs_dev = nullptr;
    int64_t total = 0;
    const int32_t st = append_prepare(pool, n_req, sids, qo_indptr, h && w_qkv, stream, &reqs_dev, &total);
    if (st != SA_OK || !reqs_dev || total == 0) return st;
    return qkv_rope_append_device(pool, reqs_dev, n_req, total, h, w_qkv, hidden, q_out, workspace, workspace_bytes, stream);
}

extern "C" int32_t sa_layer_workspace_bytes(const sa_kv_pool *pool, const sa_layer_weights *layer, int32_t n_req,
                                            const int32_t *sids, const int32_t *qo_indptr, size_t *out_bytes) {
    if (!out_bytes) return SA_ERR_INVALID_ARG;
    int32_t st = check_layer(pool, layer);
    if (st != SA_OK) return st;
    size_t attn_ws = 0;
    st = sa::attention_workspace_after_append(pool, n_req, sids, qo_indptr, &attn_ws);
    if (st != SA_OK) return st;
    const int64_t T = n_req > 0 ? qo_indptr[n_req] : 0;
    *out_bytes = layer_ws(pool, layer, T, attn_ws).total;
    return SA_OK;
}

extern "C" int32_t sa_layer_forward(sa_kv_pool *pool, const sa_layer_weights *L, int32_t n_req, const int32_t *sids,
                                    const int32_t *qo_indptr, const void *x, void *y, float sm_scale, void *workspace,
                                    size_t workspace_bytes, void *stream_) {
    sa::DeviceGuard device_guard(pool);
    if (!device_guard.ok) return SA_ERR_CUDA;
    using namespace sa;
    int32_t st = check_layer(pool, L);
    if (st != SA_OK) return st;
    if (pool->host_only) return SA_ERR_CUDA;
    size_t attn_ws = 0;
    st = attention_workspace_after_append(pool, n_req, sids, qo_indptr, &attn_ws);
    if (st != SA_OK) return st;
    const int64_t T = n_req > 0 ? qo_indptr[n_req] : 0;
    pool->last_launches = 0;
    if (T == 0) return SA_OK;
    const LayerWs wl = layer_ws(pool, L, T, attn_ws);
    if (!workspace || workspace_bytes < wl.total) return SA_ERR_WORKSPACE_TOO_SMALL;
    if (!x || !y || !L->norm1 || !L->w_qkv || !L->w_o || !L->norm2 || !L->w_gate || !L->w_up || !L->w_down)
        return SA_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    char *w = reinterpret_cast<char *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
    void *h = w + wl.off_h, *q = w + wl.off_q, *attn = w + wl.off_attn, *x1 = w + wl.off_x1, *act = w + wl.off_act;
    const int32_t H = L->hidden, QD = pool->cfg.num_q_heads * pool->cfg.head_dim;
    int32_t launches = 0;

    // h = RMSNorm(x; norm1)
    if ((st = rmsnorm(x, L->norm1, L->rms_eps, h, T, H, stream)) != SA_OK) return st;
    ++launches;
    // q|k|v = h W_qkv^T, RoPE, K'/V into the pages, Q' to q   (all-or-nothing on page exhaustion)
    st = sa_qkv_rope_append(pool, n_req, sids, qo_indptr, h, L->w_qkv, H, q, w + wl.off_qkv, sa::qkv_workspace_bytes(pool, T), stream);
    if (st != SA_OK) return st;
    launches += pool->last_launches;
    // a = attention over the paged cache (prefill chunks and decode rows of the batch together)
    st = sa_mixed_attention(pool, n_req, sids, qo_indptr, q, attn, nullptr, sm_scale, w + wl.off_attn_ws, up256(attn_ws) + 256, stream);
    if (st != SA_OK) return st;
    launches += pool->last_launches;
    // x1 = x + a W_o^T
    void *sk = w + wl.off_splitk;
    const size_t skb = up256(wl.splitk_bytes) + 256;
    if ((st = gemm_plain(attn, L->w_o, x, x1, T, H, QD, sk, skb, stream, &launches)) != SA_OK) return st;
    // h2 = RMSNorm(x1; norm2)  (reuses h)
    if ((st = rmsnorm(x1, L->norm2, L->rms_eps, h, T, H, stream)) != SA_OK) return st;
    ++launches;
    // act = SiLU(h2 W_gate^T) * (h2 W_up^T)
    if ((st = gemm_swiglu(h, L->w_gate, L->w_up, act, T, L->ffn, H, sk, skb, stream, &launches)) != SA_OK) return st;
    // y = x1 + act W_down^T
    if ((st = gemm_plain(act, L->w_down, x1, y, T, H, L->ffn, sk, skb, stream, &launches)) != SA_OK) return st;
    pool->last_launches = launches;
    return SA_OK;
}

namespace {
constexpr size_t kGemmTableFlush = size_t(256) << 20;          // larger than the 126 MB L2
constexpr size_t kGemmTableSplitK = size_t(160) * 128 * 1024;  // split-K scratch: tiles x slices never exceeds the SM count
inline size_t gt_up(size_t b) { return (std::max<size_t>(b, 256) + 255) / 256 * 256; }
int32_t gemm_table_check(int32_t hidden, int32_t ffn, int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                         const int32_t *m_list, int32_t n_m, int32_t *m_max) {
    if (!m_list || n_m <= 0 || hidden <= 0 || ffn <= 0 || num_q_heads <= 0 || num_kv_heads <= 0 || head_dim <= 0)
        return SA_ERR_INVALID_ARG;
    if (hidden % 64 != 0 || ffn % 64 != 0 || (num_q_heads * head_dim) % 64 != 0) return SA_ERR_UNSUPPORTED;
    *m_max = 0;
    for (int i = 0; i < n_m; ++i) {
        if (m_list[i] <= 0) return SA_ERR_INVALID_ARG;
        *m_max = std::max(*m_max, m_list[i]);
    }
    return SA_OK;
}
}  // namespace

extern "C" int32_t sa_gemm_table_workspace_bytes(int32_t hidden, int32_t ffn, int32_t num_q_heads, int32_t num_kv_heads,
                                                 int32_t head_dim, const int32_t *m_list, int32_t n_m, size_t *out_bytes) {
    int32_t m_max = 0;
    const int32_t st = gemm_table_check(hidden, ffn, num_q_heads, num_kv_heads, head_dim, m_list, n_m, &m_max);
    if (st != SA_OK) return st;
    if (!out_bytes) return SA_ERR_INVALID_ARG;
    const size_t H = size_t(hidden), F = size_t(ffn), QD = size_t(num_q_heads) * head_dim;
    const size_t NQKV = size_t(num_q_heads + 2 * num_kv_heads) * head_dim, M = size_t(m_max);
    *out_bytes = gt_up(NQKV * H * 2) + gt_up(H * QD * 2) + 3 * gt_up(F * H * 2) + 2 * gt_up(H * 2) + 4 * gt_up(M * H * 2) +
                 gt_up(M * NQKV * 2) + gt_up(M * F * 2) + gt_up(kGemmTableFlush) + gt_up(kGemmTableSplitK) + 256;
    return SA_OK;
}

extern "C" int32_t sa_gemm_table(int32_t hidden, int32_t ffn, int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                                 const int32_t *m_list, int32_t n_m, int32_t warmup, int32_t iters, float *out_ms,
                                 void *workspace, size_t workspace_bytes, void *stream_) {
    using namespace sa;
    int32_t m_max = 0;
    {
        const int32_t st = gemm_table_check(hidden, ffn, num_q_heads, num_kv_heads, head_dim, m_list, n_m, &m_max);
        if (st != SA_OK) return st;
    }
    if (!out_ms || iters <= 0 || warmup < 0) return SA_ERR_INVALID_ARG;
    size_t need = 0;
    sa_gemm_table_workspace_bytes(hidden, ffn, num_q_heads, num_kv_heads, head_dim, m_list, n_m, &need);
    if (!workspace || workspace_bytes < need) return SA_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t H = size_t(hidden), F = size_t(ffn), QD = size_t(num_q_heads) * head_dim;
    const size_t NQKV = size_t(num_q_heads + 2 * num_kv_heads) * head_dim, M = size_t(m_max);
    // weights and activations of the given shape are carved from the CALLER's workspace (values irrelevant to the timing)
    struct Buf {
        char *base = nullptr;
        size_t used = 0;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        ~Buf() {
            if (e0) cudaEventDestroy(e0);
            if (e1) cudaEventDestroy(e1);
        }
        void *alloc(size_t bytes) {
            void *q = base + used;
            used += gt_up(bytes);
            return q;
        }
    } b;
    b.base = reinterpret_cast<char *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
    const size_t flush_bytes = kGemmTableFlush;
    void *w_qkv = b.alloc(NQKV * H * 2), *w_o = b.alloc(H * QD * 2), *w_g = b.alloc(F * H * 2), *w_u = b.alloc(F * H * 2);
    void *w_d = b.alloc(H * F * 2), *n1 = b.alloc(H * 2), *n2 = b.alloc(H * 2);
    void *x = b.alloc(M * H * 2), *h = b.alloc(M * H * 2), *qkv = b.alloc(M * NQKV * 2), *x1 = b.alloc(M * H * 2);
    void *act = b.alloc(M * F * 2), *y = b.alloc(M * H * 2), *flush = b.alloc(flush_bytes);
    const size_t skb = kGemmTableSplitK;
    void *sk = b.alloc(skb);
    if (cudaEventCreate(&b.e0) != cudaSuccess || cudaEventCreate(&b.e1) != cudaSuccess) return SA_ERR_CUDA;
    struct { void *p; size_t n; float amp; } fills[] = {
        {w_qkv, NQKV * H, 0.05f}, {w_o, H * QD, 0.05f}, {w_g, F * H, 0.05f}, {w_u, F * H, 0.05f}, {w_d, H * F, 0.05f},
        {n1, H, 2.0f}, {n2, H, 2.0f}, {x, M * H, 2.0f}};
    uint32_t salt = 1;
    for (auto &f : fills) fill_small_kernel<<<1184, 256, 0, stream>>>(static_cast<__nv_bfloat16 *>(f.p), f.n, salt++, f.amp);
    if (cudaGetLastError() != cudaSuccess) return SA_ERR_CUDA;

    std::vector<float> times;
    for (int i = 0; i < n_m; ++i) {
        const int64_t m = m_list[i];
        times.clear();
        for (int it = 0; it < warmup + iters; ++it) {
            if (cudaMemsetAsync(flush, it & 0xff, flush_bytes, stream) != cudaSuccess) return SA_ERR_CUDA;
            cudaEventRecord(b.e0, stream);
            int32_t st = rmsnorm(x, n1, 1e-5f, h, m, hidden, stream);
            // the attention output stands in for the o-projection's input: the first Hq*D columns of qkv's buffer
            if (st == SA_OK) st = gemm_plain(h, w_qkv, nullptr, qkv, m, int32_t(NQKV), hidden, sk, skb, stream, nullptr);
            if (st == SA_OK) st = gemm_plain(qkv, w_o, x, x1, m, hidden, int32_t(QD), sk, skb, stream, nullptr);
            if (st == SA_OK) st = rmsnorm(x1, n2, 1e-5f, h, m, hidden, stream);
            if (st == SA_OK) st = gemm_swiglu(h, w_g, w_u, act, m, ffn, hidden, sk, skb, stream, nullptr);
            if (st == SA_OK) st = gemm_plain(act, w_d, x1, y, m, hidden, ffn, sk, skb, stream, nullptr);
            if (st != SA_OK) return st;
            cudaEventRecord(b.e1, stream);
            if (cudaEventSynchronize(b.e1) != cudaSuccess) return SA_ERR_CUDA;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, b.e0, b.e1);
            if (it >= warmup) times.push_back(ms);
        }
        std::sort(times.begin(), times.end());
        out_ms[i] = times[times.size() / 2];
    }
    return SA_OK;
}
