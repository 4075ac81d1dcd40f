// sa_flash_mma.cu -- decode attention over paged KV on the warp-level tensor path (mma.sync m16n8k16):
// decode-like rows (q_len * G <= 16), split-KV, HBM-bound.  One CTA per (request, kv head, 1024-key
// split); the G query heads of the group are the M rows of the MMA so K/V are read once per group;
// 4 warps take 16 keys each of every 64-key tile; cp.async 3-stage ring of page-gathered tiles;
// deterministic merge of the splits ("a single query token that attends to its full
// KV cache of length L_j ... memory-bandwidth bound").  Prefill chunks run on the tcgen05 kernel
// (sa_prefill_tc5.cu) for every supported head_dim.
// Packed rows: row rho of a (request, kv head g) pair is (token rho / G, q head g*G + rho % G).
#include <cuda_bf16.h>
#include <math.h>
#include <string.h>

#include "sa_internal.h"

namespace sa {

namespace {

constexpr int kThreads = 128;
constexpr int kBN = 64;      // keys per tile
constexpr int kStages = 3;   // cp.async ring depth (64 KiB of K/V in flight per CTA)

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&p);
}
// byte offset of 16-byte chunk `chunk` of row `row` in a [rows][D] bf16 tile, XOR-swizzled
template <int D>
__device__ __forceinline__ uint32_t tile_off(int row, int chunk) {
    return uint32_t(row * (D * 2) + ((chunk ^ (row & 7)) << 4));
}

struct KvView {
    const __nv_bfloat16 *k_base, *v_base;
    const int32_t *bt_row;  // block table row of the session
    int64_t stride_page;
    int64_t head_off;  // g * stride_head
    int32_t log2_page;
};

// Gather one 64-key tile of K and V (logical keys kt .. kt+63, kt a multiple of 64 and < kv_len) into
// swizzled smem; rows at or beyond kv_len are zero-filled (src-size 0: nothing is read), so slots the
// session does not own never reach the math.  The block-table reads come first and are branch-free:
// with pages of >= 64 slots a tile lies in one page (one read per thread); smaller pages read one entry
// per row, all independent, so their latencies overlap instead of adding up row by row.
template <int D>
__device__ __forceinline__ void load_kv_tile(const KvView &kv, int kt, int kv_len, uint32_t sK, uint32_t sV, int tid) {
    constexpr int CPR = D / 8;               // 16-byte chunks per row
    constexpr int RPP = kThreads / CPR;      // rows per pass
    constexpr int NP = kBN / RPP;            // passes
    const int chunk = tid % CPR;
    const int r0 = tid / CPR;
    const int last = kv_len - 1;
    if (kv.log2_page >= 6) {
        const int32_t page = __ldg(kv.bt_row + (kt >> kv.log2_page));
        const int slot0 = (kt & ((1 << kv.log2_page) - 1)) + r0;
        const int64_t base = int64_t(page) * kv.stride_page + kv.head_off + int64_t(slot0) * D + chunk * 8;
        const __nv_bfloat16 *kp = kv.k_base + base, *vp = kv.v_base + base;
#pragma unroll
        for (int i = 0; i < NP; ++i) {
            const int row = r0 + i * RPP;
            const int nb = (kt + row <= last) ? 16 : 0;
            const uint32_t so = tile_off<D>(row, chunk);
            cp_async16(sK + so, kp + i * (RPP * D), nb);
            cp_async16(sV + so, vp + i * (RPP * D), nb);
        }
        return;
    }
    const int pmask = (1 << kv.log2_page) - 1;
    int32_t page[NP];
#pragma unroll
    for (int i = 0; i < NP; ++i) page[i] = __ldg(kv.bt_row + (min(kt + r0 + i * RPP, last) >> kv.log2_page));
#pragma unroll
    for (int i = 0; i < NP; ++i) {
        const int row = r0 + i * RPP;
        const int key = kt + row;
        const int64_t off = int64_t(page[i]) * kv.stride_page + kv.head_off + int64_t(min(key, last) & pmask) * D + chunk * 8;
        const uint32_t so = tile_off<D>(row, chunk);
        const int nb = key <= last ? 16 : 0;
        cp_async16(sK + so, kv.k_base + off, nb);
        cp_async16(sV + so, kv.v_base + off, nb);
    }
}

// One online-softmax step of a warp over NKG groups of 16 keys starting at tile row key_off.
template <int D, int NKG>
__device__ __forceinline__ void warp_step(const uint32_t (&qf)[D / 16][4], uint32_t sK, uint32_t sV, int key_off,
                                          int kt_abs, int lim0, int lim1, bool need_mask, float scale_log2,
                                          float (&o)[D / 8][4], float &m0, float &m1, float &l0, float &l1, int lane) {
    float s[NKG * 2][4];
#pragma unroll
    for (int i = 0; i < NKG * 2; ++i) s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f;
    const int mi = lane >> 3, rr = lane & 7;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
#pragma unroll
        for (int kg = 0; kg < NKG; ++kg) {
            const int krow = key_off + kg * 16 + (mi >> 1) * 8 + rr;
            uint32_t b[4];
            ldsm_x4(b, sK + tile_off<D>(krow, ks * 2 + (mi & 1)));
            mma16816(s[kg * 2], qf[ks], b[0], b[1]);
            mma16816(s[kg * 2 + 1], qf[ks], b[2], b[3]);
        }
    }
    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < NKG * 2; ++nt) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            float v = s[nt][e] * scale_log2;
            if (need_mask) {
                const int pos = kt_abs + key_off + nt * 8 + 2 * (lane & 3) + (e & 1);
                if (pos > (e < 2 ? lim0 : lim1)) v = -INFINITY;
            }
            s[nt][e] = v;
            if (e < 2) mx0 = fmaxf(mx0, v); else mx1 = fmaxf(mx1, v);
        }
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
    const float b0 = (mn0 == -INFINITY) ? 0.f : mn0, b1 = (mn1 == -INFINITY) ? 0.f : mn1;
    const float c0 = exp2f(m0 - b0), c1 = exp2f(m1 - b1);
    m0 = mn0;
    m1 = mn1;
    float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
    for (int nt = 0; nt < NKG * 2; ++nt) {
        s[nt][0] = exp2f(s[nt][0] - b0);
        s[nt][1] = exp2f(s[nt][1] - b0);
        s[nt][2] = exp2f(s[nt][2] - b1);
        s[nt][3] = exp2f(s[nt][3] - b1);
        rs0 += s[nt][0] + s[nt][1];
        rs1 += s[nt][2] + s[nt][3];
    }
    l0 = l0 * c0 + rs0;  // per-thread partial sums; reduced across the quad at the end
    l1 = l1 * c1 + rs1;
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt) {
        o[nt][0] *= c0;
        o[nt][1] *= c0;
        o[nt][2] *= c1;
        o[nt][3] *= c1;
    }
#pragma unroll
    for (int kg = 0; kg < NKG; ++kg) {
        uint32_t a[4];
        a[0] = pack_bf16(s[kg * 2][0], s[kg * 2][1]);
        a[1] = pack_bf16(s[kg * 2][2], s[kg * 2][3]);
        a[2] = pack_bf16(s[kg * 2 + 1][0], s[kg * 2 + 1][1]);
        a[3] = pack_bf16(s[kg * 2 + 1][2], s[kg * 2 + 1][3]);
        const int vrow = key_off + kg * 16 + (mi & 1) * 8 + rr;
#pragma unroll
        for (int np = 0; np < D / 16; ++np) {
            uint32_t b[4];
            ldsm_x4_t(b, sV + tile_off<D>(vrow, np * 2 + (mi >> 1)));
            mma16816(o[np * 2], a, b[0], b[1]);
            mma16816(o[np * 2 + 1], a, b[2], b[3]);
        }
    }
}

__device__ __forceinline__ int find_req(const ReqMeta *reqs, int n, int item) {
    int lo = 0, hi = n - 1;  // last request with item_begin <= item (requests with no items never match last)
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (reqs[mid].item_begin <= item) lo = mid; else hi = mid - 1;
    }
    return lo;
}

struct AttnArgs {
    const ReqMeta *reqs;
    int32_t n_reqs;
    const __nv_bfloat16 *q;
    __nv_bfloat16 *out;
    float *lse;
    float *part_o;
    float *part_lse;
    const __nv_bfloat16 *k_base, *v_base;
    const int32_t *block_table;
    int64_t mpps, stride_page, stride_head;
    int32_t log2_page, Hq, Hkv, log2G;
    float scale_log2;
    // Captured launches (sa_decode_step): the grid is sized for the step's capacity and the actual counts are read on the
    // device, dyn = {requests, decode CTAs, ...} in the step's metadata slab; nullptr: counts are the launch's own.
    const int32_t *dyn;
};

// barrier over one 128-thread group of the CTA (id 0 with 128 threads is __syncthreads of a 128-thread CTA)
__device__ __forceinline__ void group_sync(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }

// Load BM packed rows of Q (row base rho0) into swizzled smem; rows beyond n_rows are zero.
template <int D, int BM>
__device__ __forceinline__ void load_q_tile(const AttnArgs &a, const ReqMeta &r, int g, int rho0, int n_rows,
                                            uint32_t sQ, int tid) {
    constexpr int CPR = D / 8;
    for (int e = tid; e < BM * CPR; e += kThreads) {
        const int row = e / CPR, chunk = e % CPR;
        const int rho = rho0 + row;
        uint4 val = make_uint4(0, 0, 0, 0);
        if (rho < n_rows) {
            const int tok = rho >> a.log2G, hq = (g << a.log2G) + (rho & ((1 << a.log2G) - 1));
            val = *reinterpret_cast<const uint4 *>(a.q + (int64_t(r.q_start + tok) * a.Hq + hq) * D + chunk * 8);
        }
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};\n" ::"r"(sQ + tile_off<D>(row, chunk)), "r"(val.x),
                     "r"(val.y), "r"(val.z), "r"(val.w) : "memory");
    }
}

// ------------------------------------------------------------------------------------------
// Decode-like rows: split-KV, partials out.
// One work item = one (request, kv head, 1024-key split), computed by a group of 128 threads over its own ring in
// shared memory.  The arithmetic (and so every bit of the result) depends on the item alone: which kernel, CTA or
// group runs it does not matter.
template <int D>
__device__ __forceinline__ void decode_item(const AttnArgs &a, const ReqMeta *reqs, int n_reqs, int item, unsigned char *smem,
                                            int tid, int bar_id) {
    constexpr int BM = 16;
    constexpr int TILE_BYTES = kBN * D * 2;
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t s_base = smem_u32(smem);
    const uint32_t sQ = s_base + kStages * 2 * TILE_BYTES;

    const int ri = find_req(reqs, n_reqs, item);
    const ReqMeta r = reqs[ri];
    const int local = item - r.item_begin;
    const int G = 1 << a.log2G;
    const int n_rows = r.q_len * G;
    const int g = local / r.n_splits, split = local % r.n_splits;
    constexpr int rho0 = 0;
    const int k_begin = split * kDecodeSplitKeys;
    const int k_end = min(r.kv_len, k_begin + kDecodeSplitKeys);
    KvView kv;
    kv.k_base = a.k_base;
    kv.v_base = a.v_base;
    kv.bt_row = a.block_table + int64_t(r.sid) * a.mpps;
    kv.stride_page = a.stride_page;
    kv.head_off = int64_t(g) * a.stride_head;
    kv.log2_page = a.log2_page;

    const int n_tiles = (k_end - k_begin + kBN - 1) / kBN;
    // prologue of the cp.async ring
#pragma unroll
    for (int s = 0; s < kStages - 1; ++s) {
        if (s < n_tiles)
            load_kv_tile<D>(kv, k_begin + s * kBN, r.kv_len, s_base + s * 2 * TILE_BYTES,
                            s_base + s * 2 * TILE_BYTES + TILE_BYTES, tid);
        cp_async_commit();
    }
    load_q_tile<D, BM>(a, r, g, rho0, n_rows, sQ, tid);
    group_sync(bar_id);
    constexpr int row_base = 0;
    uint32_t qf[D / 16][4];
    {
        const int mi = lane >> 3, rr = lane & 7;
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks)
            ldsm_x4(qf[ks], sQ + tile_off<D>(row_base + (mi & 1) * 8 + rr, ks * 2 + (mi >> 1)));
    }
    // causal limits (inclusive last key) of this thread's two rows
    const int rA = rho0 + row_base + (lane >> 2), rB = rA + 8;
    const int base_lim = r.kv_len - r.q_len;
    const int lim0 = rA < n_rows ? base_lim + (rA >> a.log2G) : -1;
    const int lim1 = rB < n_rows ? base_lim + (rB >> a.log2G) : -1;
    // smallest limit among this warp's rows (warp-uniform): tiles entirely at or below it need no mask
    const int warp_rows_lo = rho0 + row_base;
    const int lim_min = (warp_rows_lo + 15 < n_rows) ? base_lim + (warp_rows_lo >> a.log2G) : -1;

    float o[D / 8][4];
#pragma unroll
    for (int i = 0; i < D / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;

    for (int t = 0; t < n_tiles; ++t) {
        cp_async_wait<kStages - 2>();
        group_sync(bar_id);
        {
            const int tn = t + kStages - 1;
            if (tn < n_tiles) {
                const int sn = tn % kStages;
                load_kv_tile<D>(kv, k_begin + tn * kBN, r.kv_len, s_base + sn * 2 * TILE_BYTES,
                                s_base + sn * 2 * TILE_BYTES + TILE_BYTES, tid);
            }
            cp_async_commit();
        }
        const int st = t % kStages;
        const uint32_t sK = s_base + st * 2 * TILE_BYTES, sV = sK + TILE_BYTES;
        const int kt = k_begin + t * kBN;
        const int key_off = warp * 16;
        if (kt + key_off < k_end) {  // warp-uniform: this warp's 16 keys hold at least one live key
            const bool need_mask = kt + key_off + 15 > lim_min;
            warp_step<D, 1>(qf, sK, sV, key_off, kt, lim0, lim1, need_mask, a.scale_log2, o, m0, m1, l0, l1, lane);
        }
    }
    cp_async_wait<0>();
    l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
    l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 2);

    // ---- merge the four warps' states (each saw a disjoint quarter of every tile)
    group_sync(bar_id);  // everyone is done with the stage buffers
    float *sO = reinterpret_cast<float *>(smem);             // [4][16][D]
    float *sM = sO + 4 * 16 * D;                             // [4][16]
    float *sL = sM + 4 * 16;                                 // [4][16]
    {
        const int r0 = lane >> 2, r1 = r0 + 8;
        float *wo = sO + warp * 16 * D;
#pragma unroll
        for (int nt = 0; nt < D / 8; ++nt) {
            const int col = nt * 8 + 2 * (lane & 3);
            *reinterpret_cast<float2 *>(wo + r0 * D + col) = make_float2(o[nt][0], o[nt][1]);
            *reinterpret_cast<float2 *>(wo + r1 * D + col) = make_float2(o[nt][2], o[nt][3]);
        }
        if ((lane & 3) == 0) {
            sM[warp * 16 + r0] = m0;
            sM[warp * 16 + r1] = m1;
            sL[warp * 16 + r0] = l0;
            sL[warp * 16 + r1] = l1;
        }
    }
    group_sync(bar_id);
    for (int e = tid; e < n_rows * (D / 4); e += kThreads) {
        const int row = e / (D / 4), c4 = e % (D / 4);
        float M = -INFINITY;
#pragma unroll
        for (int w = 0; w < 4; ++w) M = fmaxf(M, sM[w * 16 + row]);
        const float Mb = (M == -INFINITY) ? 0.f : M;
        float L = 0.f;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int w = 0; w < 4; ++w) {  // fixed order: bit-reproducible
            const float wgt = exp2f(sM[w * 16 + row] - Mb);
            L += sL[w * 16 + row] * wgt;
            const float4 ov = *reinterpret_cast<const float4 *>(sO + (w * 16 + row) * D + c4 * 4);
            acc.x += ov.x * wgt;
            acc.y += ov.y * wgt;
            acc.z += ov.z * wgt;
            acc.w += ov.w * wgt;
        }
        const float inv = L > 0.f ? 1.f / L : 0.f;
        const int tok = row >> a.log2G, hq = (g << a.log2G) + (row & (G - 1));
        const int64_t prow = int64_t(r.part_begin) + (int64_t(split) * r.q_len + tok) * a.Hq + hq;
        *reinterpret_cast<float4 *>(a.part_o + prow * D + c4 * 4) = make_float4(acc.x * inv, acc.y * inv, acc.z * inv, acc.w * inv);
        if (c4 == 0) a.part_lse[prow] = L > 0.f ? M + log2f(L) : -INFINITY;  // log2 domain
    }
}

// grid = decode CTAs of the call (one item each).  INLINE: the requests of a small decode-only call ride in the kernel
// parameters (no metadata upload launch).
template <int D, bool INLINE>
__global__ void __launch_bounds__(kThreads) flash_mma_kernel(const __grid_constant__ InlineReqs ir, const AttnArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    int n_reqs = a.n_reqs;
    if (!INLINE && a.dyn) {
        n_reqs = a.dyn[0];
        if (int(blockIdx.x) >= a.dyn[1]) return;
    }
    decode_item<D>(a, INLINE ? ir.reqs : a.reqs, n_reqs, blockIdx.x, smem, threadIdx.x, 0);
}

// The same items on a FIXED number of CTAs, each with two 128-thread groups that walk the item list with their own
// rings (2 x 100 KiB of shared memory: nothing else fits on the SM).  Used by the overlapped mixed call, where the
// decode rows must stay on a subset of the SMs while the tensor-core prefill kernel owns the others.
template <int D>
__global__ void __launch_bounds__(2 * kThreads) flash_mma_persist_kernel(const AttnArgs a, int n_items) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr size_t GROUP_BYTES = size_t(kStages) * 2 * kBN * D * 2 + size_t(16) * D * 2;
    const int grp = threadIdx.x >> 7, tid = threadIdx.x & 127;
    unsigned char *my = smem + size_t(grp) * GROUP_BYTES;
    for (int item = blockIdx.x * 2 + grp; item < n_items; item += gridDim.x * 2) {
        decode_item<D>(a, a.reqs, a.n_reqs, item, my, tid, 1 + grp);
        group_sync(1 + grp);  // the merge scratch of this item lives in the ring the next item fills
    }
}

// Merge of the split partials, fixed split order.  grid = (decode-like requests, Hkv); each warp
// takes packed rows of the group; lanes cover D with float4.
template <int D, bool INLINE>
__global__ void __launch_bounds__(128) merge_splits_kernel(const __grid_constant__ InlineReqs ir, const AttnArgs a) {
    // launched with programmatic stream serialization: the grid is staged while the split kernel drains and waits
    // here until that kernel has completed and its partials are visible (a no-op for an ordinary launch)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (!INLINE && a.dyn && int(blockIdx.x) >= a.dyn[0]) return;
    const ReqMeta r = INLINE ? ir.reqs[blockIdx.x] : a.reqs[blockIdx.x];
    const int g = blockIdx.y;
    const int G = 1 << a.log2G;
    const int n_rows = r.q_len * G;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int LANES = D / 4;
    for (int row = warp; row < n_rows; row += 4) {
        const int tok = row >> a.log2G, hq = (g << a.log2G) + (row & (G - 1));
        const int64_t p0 = int64_t(r.part_begin) + int64_t(tok) * a.Hq + hq;
        const int64_t pstride = int64_t(r.q_len) * a.Hq;
        float M = -INFINITY;
        for (int s = 0; s < r.n_splits; ++s) M = fmaxf(M, a.part_lse[p0 + s * pstride]);
        const float Mb = (M == -INFINITY) ? 0.f : M;
        float W = 0.f;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int s = 0; s < r.n_splits; ++s) {
            const float w = exp2f(a.part_lse[p0 + s * pstride] - Mb);
            W += w;
            if (lane < LANES) {
                const float4 ov = *reinterpret_cast<const float4 *>(a.part_o + (p0 + s * pstride) * D + lane * 4);
                acc.x += ov.x * w;
                acc.y += ov.y * w;
                acc.z += ov.z * w;
                acc.w += ov.w * w;
            }
        }
        const float inv = W > 0.f ? 1.f / W : 0.f;
        const int64_t orow = int64_t(r.q_start + tok) * a.Hq + hq;
        if (lane < LANES) {
            uint2 pk;
            pk.x = pack_bf16(acc.x * inv, acc.y * inv);
            pk.y = pack_bf16(acc.z * inv, acc.w * inv);
            *reinterpret_cast<uint2 *>(a.out + orow * D + lane * 4) = pk;
        }
        if (a.lse && lane == 0) a.lse[orow] = (M + log2f(W)) * 0.6931471805599453f;
    }
}

AttnArgs make_args(const sa_kv_pool *pool, const ReqMeta *reqs, int32_t n, const void *q, void *out, float *lse,
                   float sm_scale, float *part_o, float *part_lse) {
    AttnArgs a;
    a.reqs = reqs;
    a.n_reqs = n;
    a.q = static_cast<const __nv_bfloat16 *>(q);
    a.out = static_cast<__nv_bfloat16 *>(out);
    a.lse = lse;
    a.part_o = part_o;
    a.part_lse = part_lse;
    a.k_base = static_cast<const __nv_bfloat16 *>(pool->k_base);
    a.v_base = static_cast<const __nv_bfloat16 *>(pool->v_base);
    a.block_table = pool->block_table;
    a.mpps = pool->max_pages_per_session;
    a.stride_page = pool->stride_page;
    a.stride_head = pool->stride_head;
    a.log2_page = pool->log2_page;
    a.Hq = pool->cfg.num_q_heads;
    a.Hkv = pool->cfg.num_kv_heads;
    int lg = 0;
    while ((1 << lg) < pool->G) ++lg;
    a.log2G = lg;
    a.scale_log2 = sm_scale * 1.4426950408889634f;
    a.dyn = nullptr;
    return a;
}

// The > 48 KiB dynamic shared memory opt-in is a per-device, per-function attribute: set it once per (function, device).
template <auto kernel>
cudaError_t opt_in_smem(size_t smem) {
    static unsigned long long done = 0;  // bit per device ordinal; one static per kernel (the kernel is the template argument)
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 64 && (done >> dev) & 1ull) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (e == cudaSuccess && dev < 64) done |= 1ull << dev;
    return e;
}

template <int D>
constexpr size_t group_smem() {
    return size_t(kStages) * 2 * kBN * D * 2 + size_t(16) * D * 2;
}

// The merge of the splits is launched with programmatic stream serialization: its grid is set up while the split
// kernel still runs and starts (griddepcontrol.wait at its top) the moment that kernel has completed.
template <int D, bool INLINE>
cudaError_t launch_merge(const InlineReqs &ir, const AttnArgs &a, dim3 grid, cudaStream_t stream) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(128);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, merge_splits_kernel<D, INLINE>, ir, a);
}

template <int D, bool INLINE>
cudaError_t launch_flash(const InlineReqs &ir, const AttnArgs &a, int items, dim3 merge_grid, cudaStream_t stream,
                         int32_t *launches) {
    constexpr size_t smem = group_smem<D>();
    static_assert(smem >= 4 * 16 * D * 4 + 2 * 4 * 16 * 4, "merge scratch must fit in the stage ring");
    cudaError_t e = opt_in_smem<&flash_mma_kernel<D, INLINE>>(smem);
    if (e != cudaSuccess) return e;
    flash_mma_kernel<D, INLINE><<<unsigned(items), kThreads, smem, stream>>>(ir, a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ++*launches;
    e = launch_merge<D, INLINE>(ir, a, merge_grid, stream);
    ++*launches;
    return e;
}

template <int D>
cudaError_t launch_flash_persist(const AttnArgs &a, int items, int n_cta, dim3 merge_grid, cudaStream_t stream, int32_t *launches) {
    constexpr size_t smem = 2 * group_smem<D>();
    cudaError_t e = opt_in_smem<&flash_mma_persist_kernel<D>>(smem);
    if (e != cudaSuccess) return e;
    flash_mma_persist_kernel<D><<<unsigned(n_cta), 2 * kThreads, smem, stream>>>(a, items);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ++*launches;
    static const InlineReqs none{};
    e = launch_merge<D, false>(none, a, merge_grid, stream);
    ++*launches;
    return e;
}

}  // namespace

// reqs_host != nullptr (and plan.n_dec <= kInlineReqs): the requests go in the kernel parameters, reqs_dev is unused.
// persist_ctas > 0: the items run on that many two-group CTAs (one per SM) instead of one CTA each.
// dyn != nullptr (captured step): grid sizes come from `plan` (the step's capacity), the actual counts from dyn.
cudaError_t launch_flash_decode(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const ReqMeta *reqs_host,
                                const AttnPlan &plan, const void *q, void *out, float *lse, float sm_scale,
                                float *part_o, float *part_lse, cudaStream_t stream, int32_t *launches,
                                int persist_ctas, const int32_t *dyn) {
    if (plan.dec_items == 0) return cudaSuccess;
    AttnArgs a = make_args(pool, reqs_dev, plan.n_dec, q, out, lse, sm_scale, part_o, part_lse);
    a.dyn = dyn;
    const dim3 grid(unsigned(plan.n_dec), unsigned(pool->cfg.num_kv_heads));
    const bool d128 = pool->cfg.head_dim == 128;
    if (reqs_host) {
        InlineReqs ir;
        memcpy(ir.reqs, reqs_host, sizeof(ReqMeta) * size_t(plan.n_dec));
        return d128 ? launch_flash<128, true>(ir, a, plan.dec_items, grid, stream, launches)
                    : launch_flash<64, true>(ir, a, plan.dec_items, grid, stream, launches);
    }
    if (persist_ctas > 0)
        return d128 ? launch_flash_persist<128>(a, plan.dec_items, persist_ctas, grid, stream, launches)
                    : launch_flash_persist<64>(a, plan.dec_items, persist_ctas, grid, stream, launches);
    static const InlineReqs none{};  // never read by the slab variants
    return d128 ? launch_flash<128, false>(none, a, plan.dec_items, grid, stream, launches)
                : launch_flash<64, false>(none, a, plan.dec_items, grid, stream, launches);
}

}  // namespace sa
