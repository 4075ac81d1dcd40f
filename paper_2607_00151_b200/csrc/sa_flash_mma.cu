// sa_flash_mma.cu -- decode attention over paged KV on the warp-level tensor path (mma.sync m16n8k16):
// decode-like rows (q_len * G <= 16), split-KV, HBM-bound.  One CTA per (request, kv head, 1024-key
// split); the G query heads of the group are the N columns of the MMA (keys are its M rows: S^T = K Q^T,
// O^T += V^T P^T) so K/V are read once per group and no tensor work is spent on padding rows;
// 4 warps take 16 keys each of every 64-key tile; 3-stage ring of page-gathered tiles filled by TMA (one thread
// issues the page boxes of a tile, an mbarrier per stage counts the bytes);
// deterministic merge of the splits by the last of them to finish ("a single query token that attends to its full
// KV cache of length L_j ... memory-bandwidth bound").  Prefill chunks run on the tcgen05 kernel
// (sa_prefill_tc5.cu) for every supported head_dim.
// Packed rows: row rho of a (request, kv head g) pair is (token rho / G, q head g*G + rho % G).
#include <cuda.h>
#include <cuda_bf16.h>
#include <math.h>
#include <string.h>

#include "sa_internal.h"
#include "sa_tc5_ptx.cuh"

namespace sa {

namespace {

constexpr int kThreads = 128;
constexpr int kBN = 64;      // keys per tile
constexpr int kStages = 3;   // depth of the TMA-filled K/V ring (64 KiB in flight per item)
constexpr int kMaxSplitPages = kDecodeSplitKeys / 16;  // pages a split can span at the smallest page size

using ptx::smem_u32;
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
// Byte offset of 16-byte chunk `chunk` of row `row` in a [ROWS][D] bf16 tile held as D/64 halves of [ROWS][128 B] in
// the 128-byte swizzle (chunk ^ row % 8 inside a 128-byte row): what a TMA box of 64 dims x ROWS slots with
// SWIZZLE_128B writes, and conflict-free for ldmatrix.
template <int ROWS>
__device__ __forceinline__ uint32_t tile_off(int row, int chunk) {
    return uint32_t((chunk >> 3) * (ROWS * 128) + row * 128 + (((chunk & 7) ^ (row & 7)) << 4));
}

constexpr int kLoopReqCache = 128;  // requests a captured step keeps in shared memory (4 KiB)
// shared memory of the 128 threads of an item: the K/V ring, the Q tile, the page ids of the split, a flag, the ring's mbarriers
template <int D>
constexpr size_t group_smem() {
    return size_t(kStages) * 2 * kBN * D * 2 + size_t(16) * D * 2 + kMaxSplitPages * 4 + 16 + 32;
}
constexpr size_t kSmemAlign = 1024;  // TMA destinations in the 128-byte swizzle want 1024-byte aligned tiles

struct KvView {
    const CUtensorMap *tmap_k, *tmap_v;  // 4-D maps over the pool's pages: (64 dims, page slots, 1 head, 1 page) boxes
    const int32_t *pages;   // shared memory: the page ids of the item's split, pages[0] = page of key k_begin
    int32_t page0;          // k_begin >> log2_page
    int32_t n_pages;        // pages of the split that hold session data
    int32_t g;              // kv head
    int32_t log2_page;
};

// One 64-key tile of K and V (logical keys kt .. kt+63, kt a multiple of 64) into a ring stage, by TMA: one elected
// thread issues D/64 boxes per page and operand and the stage's mbarrier counts the bytes.  (Until round 2 every
// thread issued sixteen 16-byte cp.async per tile behind its own address arithmetic, ~100 of the ~400 instructions a warp
// spent per tile; with this and the transposed MMAs the kernel executes 38 % fewer instructions for the same time.)  Only pages the
// session owns are requested; what the rest of the stage holds is dealt with by the caller (zero_v_tail).
template <int D>
__device__ __forceinline__ void issue_kv_tile(const KvView &kv, int kt, uint32_t sK, uint32_t sV, uint32_t bar) {
    constexpr int DH = D / 64;
    constexpr uint32_t HALF = kBN * 128;
    if (kv.log2_page >= 6) {
        const int32_t pg = kv.pages[(kt >> kv.log2_page) - kv.page0];
        ptx::mbar_expect_tx(bar, 2 * DH * HALF);
#pragma unroll
        for (int h = 0; h < DH; ++h) {
            ptx::tma_load_4d(sK + h * HALF, kv.tmap_k, bar, h * 64, 0, kv.g, pg);
            ptx::tma_load_4d(sV + h * HALF, kv.tmap_v, bar, h * 64, 0, kv.g, pg);
        }
        return;
    }
    const int p0 = (kt >> kv.log2_page) - kv.page0;
    const int np = min(kBN >> kv.log2_page, kv.n_pages - p0);
    const uint32_t page_bytes = 128u << kv.log2_page;  // one page, one 64-dim half
    ptx::mbar_expect_tx(bar, uint32_t(np) * 2 * DH * page_bytes);
    for (int u = 0; u < np; ++u) {
        const int32_t pg = kv.pages[p0 + u];
#pragma unroll
        for (int h = 0; h < DH; ++h) {
            ptx::tma_load_4d(sK + h * HALF + u * page_bytes, kv.tmap_k, bar, h * 64, 0, kv.g, pg);
            ptx::tma_load_4d(sV + h * HALF + u * page_bytes, kv.tmap_v, bar, h * 64, 0, kv.g, pg);
        }
    }
}

// Rows [valid, 64) of a V stage hold no session data (slots past the end of the session, pages never requested):
// they must be exactly zero, because P is 0 there and 0 * NaN = NaN.  (K rows past the end only produce scores that
// the mask replaces.)  Generic-proxy stores into a buffer the async proxy writes next: fenced.
template <int D>
__device__ __forceinline__ void zero_v_tail(uint32_t sV, int valid, int tid) {
    constexpr int CPR = D / 8;
    for (int e = valid * CPR + tid; e < kBN * CPR; e += kThreads) {
        const int row = e / CPR, chunk = e % CPR;
        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(sV + tile_off<kBN>(row, chunk)), "r"(0) : "memory");
    }
    ptx::fence_proxy_async_smem();
}

// barrier over the 128 threads that run an item (id 0 with 128 threads is __syncthreads of a 128-thread CTA)
__device__ __forceinline__ void group_sync(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }

__device__ __forceinline__ uint32_t movmatrix_t(uint32_t x) {  // transpose of an 8x8 b16 matrix held one row pair per lane
    uint32_t y;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;\n" : "=r"(y) : "r"(x));
    return y;
}

// Running state of a warp for its NT * 8 query rows.  Everything is held TRANSPOSED: the 16 keys of a step are the M
// rows of the MMA and the query rows its N columns, S^T = K Q^T and O^T += V^T P^T.  A decode batch has G (<= 8) live
// rows per kv head, so one n8 column tile carries them and a step costs D/16 + D/16 HMMAs instead of twice that with
// the rows as M (16 rows, most of them padding); on sm_100a the warp-level HMMA pipe retires one m16n8k16 per ~30 cycles
// per scheduler, and with the rows as M it was busy for two thirds of a lone item's time.  (Measured: the pipe's
// active time halved, issue slots 32 -> 19 % busy on a full batch; the time of a call is set elsewhere -- HBM on a
// full batch, fixed costs at one row -- and did not move.)
// A thread holds query rows qa = nt*8 + 2*(lane%4) and qa + 1 (C-fragment columns); keys / dims run over lane/4.
template <int D, int NT>
struct WarpState {
    float o[D / 16][NT][4];  // O^T: [0],[1] dim = np*16 + lane/4, rows qa, qa+1; [2],[3] dim + 8
    float m[NT][2], l[NT][2];
};

// One online-softmax step of a warp over 16 keys starting at tile row key_off (absolute position kt_abs + key_off).
template <int D, int NT>
__device__ __forceinline__ void warp_step(const uint32_t (&qf)[D / 16][4], uint32_t sK, uint32_t sV, int key_off, int kt_abs,
                                          const int (&lim)[NT][2], bool need_mask, float scale_log2, WarpState<D, NT> &w,
                                          int lane) {
    float s[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
    const int mi = lane >> 3, rr = lane & 7;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
        uint32_t ka[4];  // A = K: keys x dims, row-major as stored
        ldsm_x4(ka, sK + tile_off<kBN>(key_off + (mi & 1) * 8 + rr, ks * 2 + (mi >> 1)));
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) mma16816(s[nt], ka, qf[ks][2 * nt], qf[ks][2 * nt + 1]);
    }
    const int key_lo = kt_abs + key_off + (lane >> 2);  // this thread's keys: key_lo ([0],[1]) and key_lo + 8 ([2],[3])
    float c[NT][2], b[NT][2];
    bool moved = false;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            float v = s[nt][e] * scale_log2;
            if (need_mask && key_lo + (e >> 1) * 8 > lim[nt][e & 1]) v = -INFINITY;
            s[nt][e] = v;
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float mx = fmaxf(s[nt][j], s[nt][2 + j]);
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
            const float mn = fmaxf(w.m[nt][j], mx);
            b[nt][j] = (mn == -INFINITY) ? 0.f : mn;
            c[nt][j] = exp2f(w.m[nt][j] - b[nt][j]);
            moved = moved || c[nt][j] != 1.f;
            w.m[nt][j] = mn;
        }
    }
    uint32_t pb[NT][2];  // B = P^T: keys x rows
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        s[nt][0] = exp2f(s[nt][0] - b[nt][0]);
        s[nt][1] = exp2f(s[nt][1] - b[nt][1]);
        s[nt][2] = exp2f(s[nt][2] - b[nt][0]);
        s[nt][3] = exp2f(s[nt][3] - b[nt][1]);
        // per-thread partial row sums (this thread's two keys); reduced over lane/4 at the end of the item
        w.l[nt][0] = w.l[nt][0] * c[nt][0] + (s[nt][0] + s[nt][2]);
        w.l[nt][1] = w.l[nt][1] * c[nt][1] + (s[nt][1] + s[nt][3]);
        // C fragment (key = lane/4, rows qa, qa+1) -> B fragment (keys 2*(lane%4), +1, row = lane/4): an 8x8 transpose
        pb[nt][0] = movmatrix_t(pack_bf16(s[nt][0], s[nt][1]));
        pb[nt][1] = movmatrix_t(pack_bf16(s[nt][2], s[nt][3]));
    }
    // O needs rescaling only when some row max of the warp moved (c = 1 exactly otherwise: skipping changes no bit)
    if (__any_sync(0xffffffffu, moved)) {
#pragma unroll
        for (int np = 0; np < D / 16; ++np)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                w.o[np][nt][0] *= c[nt][0];
                w.o[np][nt][1] *= c[nt][1];
                w.o[np][nt][2] *= c[nt][0];
                w.o[np][nt][3] *= c[nt][1];
            }
    }
#pragma unroll
    for (int np = 0; np < D / 16; ++np) {
        uint32_t va[4];  // A = V^T: dims x keys, i.e. the stored [key][dim] tile read through the transposing ldmatrix
        ldsm_x4_t(va, sV + tile_off<kBN>(key_off + (mi >> 1) * 8 + rr, np * 2 + (mi & 1)));
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) mma16816(w.o[np][nt], va, pb[nt][0], pb[nt][1]);
    }
}

// The tile loop of one item for NT * 8 query rows; leaves the warp's (unnormalised O^T, m, l) in the merge scratch.
template <int D, int NT>
__device__ __forceinline__ void decode_tiles(const KvView &kv, const ReqMeta &r, int log2G, int n_rows, int k_begin, int k_end,
                                             int n_tiles, float scale_log2, uint32_t s_base, uint32_t sQ, unsigned char *smem,
                                             uint32_t bars, uint32_t &phase, int tid, int bar_id) {
    constexpr int TILE_BYTES = kBN * D * 2;
    const int lane = tid & 31, warp = tid >> 5;
    uint32_t qf[D / 16][4];  // B = Q^T: [ks][2*nt], [2*nt+1] = dims ks*16 + {0..7, 8..15} of rows nt*8 + lane/4
    {
        const int mi = lane >> 3, rr = lane & 7;
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) ldsm_x4(qf[ks], sQ + tile_off<16>((mi >> 1) * 8 + rr, ks * 2 + (mi & 1)));
    }
    // causal limits (inclusive last key) of this thread's rows; rows beyond n_rows are padding whose results are
    // never read (Q is zero there, so they stay finite): no limit, so that they never force a mask
    const int base_lim = r.kv_len - r.q_len;
    int lim[NT][2];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int q = nt * 8 + 2 * (lane & 3) + j;
            lim[nt][j] = q < n_rows ? base_lim + (q >> log2G) : 0x7fffffff;
        }
    const int lim_min = base_lim;  // row 0's limit, the smallest: tiles entirely at or below it need no mask

    WarpState<D, NT> w;
#pragma unroll
    for (int np = 0; np < D / 16; ++np)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) w.o[np][nt][0] = w.o[np][nt][1] = w.o[np][nt][2] = w.o[np][nt][3] = 0.f;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        w.m[nt][0] = w.m[nt][1] = -INFINITY;
        w.l[nt][0] = w.l[nt][1] = 0.f;
    }

    for (int t = 0; t < n_tiles; ++t) {
        const int st = t % kStages;
        ptx::mbar_wait_watched(bars + 8 * st, (phase >> st) & 1u);  // tile t has landed (acquire: its bytes are visible)
        phase ^= 1u << st;
        group_sync(bar_id);                                 // ... and everyone is done with tile t - 1: its stage is free
        {
            const int tn = t + kStages - 1;
            if (tid == 0 && tn < n_tiles) {
                const int sn = tn % kStages;
                issue_kv_tile<D>(kv, k_begin + tn * kBN, s_base + sn * 2 * TILE_BYTES, s_base + sn * 2 * TILE_BYTES + TILE_BYTES,
                                 bars + 8 * sn);
            }
        }
        const uint32_t sK = s_base + st * 2 * TILE_BYTES, sV = sK + TILE_BYTES;
        const int kt = k_begin + t * kBN;
        if (k_end - kt < kBN) {  // the session ends inside this tile (uniform over the item; its last tile only)
            zero_v_tail<D>(sV, k_end - kt, tid);
            group_sync(bar_id);
        }
        const int key_off = warp * 16;
        if (kt + key_off < k_end) {  // warp-uniform: this warp's 16 keys hold at least one live key
            const bool need_mask = kt + key_off + 15 > lim_min;
            warp_step<D, NT>(qf, sK, sV, key_off, kt, lim, need_mask, scale_log2, w, lane);
        }
    }
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            w.l[nt][j] += __shfl_xor_sync(0xffffffffu, w.l[nt][j], 4);
            w.l[nt][j] += __shfl_xor_sync(0xffffffffu, w.l[nt][j], 8);
            w.l[nt][j] += __shfl_xor_sync(0xffffffffu, w.l[nt][j], 16);
        }
    // ---- the warp's state into the merge scratch (each warp saw a disjoint quarter of every tile)
    group_sync(bar_id);  // everyone is done with the stage buffers
    float *sO = reinterpret_cast<float *>(smem);             // [4][16][D]
    float *sM = sO + 4 * 16 * D;                             // [4][16]
    float *sL = sM + 4 * 16;                                 // [4][16]
    float *wo = sO + warp * 16 * D;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        const int qa = nt * 8 + 2 * (lane & 3);
#pragma unroll
        for (int np = 0; np < D / 16; ++np) {
            const int dim = np * 16 + (lane >> 2);
            wo[qa * D + dim] = w.o[np][nt][0];
            wo[(qa + 1) * D + dim] = w.o[np][nt][1];
            wo[qa * D + dim + 8] = w.o[np][nt][2];
            wo[(qa + 1) * D + dim + 8] = w.o[np][nt][3];
        }
        if ((lane >> 2) == 0) {
            sM[warp * 16 + qa] = w.m[nt][0];
            sM[warp * 16 + qa + 1] = w.m[nt][1];
            sL[warp * 16 + qa] = w.l[nt][0];
            sL[warp * 16 + qa + 1] = w.l[nt][1];
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
    const int32_t *block_table;
    int32_t *tickets;  // [requests of the call][Hkv] arrival counters, zero on entry and on exit
    int64_t mpps;
    int32_t log2_page, Hq, Hkv, log2G;
    float scale_log2;
    // Captured launches (sa_decode_step): the grids are fixed and the actual counts are read on the device,
    // dyn = {requests, items} at the head of the step's metadata; nullptr: the counts are the launch's own.
    const int32_t *dyn;
};


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
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};\n" ::"r"(sQ + tile_off<BM>(row, chunk)), "r"(val.x),
                     "r"(val.y), "r"(val.z), "r"(val.w) : "memory");
    }
}

// Merge of the splits of one (request, kv head), run by the LAST of its split items to finish (arrival counter in
// the pool): each warp takes packed rows of the group; lanes cover D with float4.  Every sum has a fixed order that
// depends on the request's split count alone (row max and the weight total: lane-strided, then a butterfly over the
// warp; the output: split order), so a row's bits depend neither on its batch nor on which item arrived last.  The
// partials of 4 splits are requested together and the next 4 before those are summed: one load per loop trip made the
// merge a chain of L2 round trips as long as the streaming of the splits itself.  Loads bypass L1 (other SMs wrote).
template <int D>
__device__ __forceinline__ void merge_rows(const AttnArgs &a, const ReqMeta &r, int g, int tid) {
    const int G = 1 << a.log2G;
    const int n_rows = r.q_len * G;
    const int lane = tid & 31, warp = tid >> 5;
    constexpr int LANES = D / 4;
    constexpr int U = 4;
    const int n = r.n_splits;
    for (int row = warp; row < n_rows; row += 4) {
        const int tok = row >> a.log2G, hq = (g << a.log2G) + (row & (G - 1));
        const int64_t p0 = int64_t(r.part_begin) + int64_t(tok) * a.Hq + hq;
        const int64_t pstride = int64_t(r.q_len) * a.Hq;
        float4 ov[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            ov[u] = (u < n && lane < LANES) ? __ldcg(reinterpret_cast<const float4 *>(a.part_o + (p0 + u * pstride) * D + lane * 4))
                                            : make_float4(0.f, 0.f, 0.f, 0.f);
        float M = -INFINITY;
        for (int s = lane; s < n; s += 32) M = fmaxf(M, __ldcg(a.part_lse + p0 + s * pstride));
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, d));
        const float Mb = (M == -INFINITY) ? 0.f : M;
        float W = 0.f;
        for (int s = lane; s < n; s += 32) W += exp2f(__ldcg(a.part_lse + p0 + s * pstride) - Mb);
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) W += __shfl_xor_sync(0xffffffffu, W, d);
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int s0 = 0; s0 < n; s0 += U) {
            float ls[U];
            float4 nx[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                ls[u] = s0 + u < n ? __ldcg(a.part_lse + p0 + (s0 + u) * pstride) : -INFINITY;
                nx[u] = (s0 + U + u < n && lane < LANES)
                            ? __ldcg(reinterpret_cast<const float4 *>(a.part_o + (p0 + (s0 + U + u) * pstride) * D + lane * 4))
                            : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {  // split order
                if (s0 + u < n) {
                    const float w = exp2f(ls[u] - Mb);
                    acc.x += ov[u].x * w;
                    acc.y += ov[u].y * w;
                    acc.z += ov[u].z * w;
                    acc.w += ov[u].w * w;
                }
                ov[u] = nx[u];
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

// ------------------------------------------------------------------------------------------
// Decode-like rows: split-KV, partials out.
// One work item = one (request, kv head, 1024-key split), computed by a group of 128 threads over its own ring in
// shared memory.  The arithmetic (and so every bit of the result) depends on the item alone: which kernel, CTA or
// group runs it does not matter.
template <int D>
__device__ __forceinline__ void decode_item(const AttnArgs &a, const CUtensorMap *tmap_k, const CUtensorMap *tmap_v,
                                            const ReqMeta *reqs, int n_reqs, int item, unsigned char *smem, uint32_t &phase,
                                            int tid, int bar_id) {
    constexpr int BM = 16;
    constexpr int TILE_BYTES = kBN * D * 2;
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t s_base = smem_u32(smem);
    const uint32_t sQ = s_base + kStages * 2 * TILE_BYTES;
    int32_t *s_pages = reinterpret_cast<int32_t *>(smem + kStages * 2 * TILE_BYTES + BM * D * 2);  // [kMaxSplitPages]
    const uint32_t bars = smem_u32(s_pages + kMaxSplitPages + 4);  // [kStages] mbarriers of the ring (after the flag)

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
    kv.tmap_k = tmap_k;
    kv.tmap_v = tmap_v;
    kv.pages = s_pages;
    kv.page0 = k_begin >> a.log2_page;
    kv.n_pages = ((k_end - 1) >> a.log2_page) - kv.page0 + 1;
    kv.g = g;
    kv.log2_page = a.log2_page;

    const int n_tiles = (k_end - k_begin + kBN - 1) / kBN;
    // the split's slice of the block table (<= 64 entries) and Q: one global round trip, then the ring starts
    if (tid < kv.n_pages) s_pages[tid] = __ldg(a.block_table + int64_t(r.sid) * a.mpps + kv.page0 + tid);
    load_q_tile<D, BM>(a, r, g, rho0, n_rows, sQ, tid);
    group_sync(bar_id);
    if (tid == 0) {  // prologue of the ring
#pragma unroll
        for (int s = 0; s < kStages - 1; ++s)
            if (s < n_tiles)
                issue_kv_tile<D>(kv, k_begin + s * kBN, s_base + s * 2 * TILE_BYTES, s_base + s * 2 * TILE_BYTES + TILE_BYTES, bars + 8 * s);
    }
    // rows as MMA columns: one n8 tile when the group's rows fit (every decode batch with G <= 8), else two
    if (n_rows <= 8)
        decode_tiles<D, 1>(kv, r, a.log2G, n_rows, k_begin, k_end, n_tiles, a.scale_log2, s_base, sQ, smem, bars, phase, tid, bar_id);
    else
        decode_tiles<D, 2>(kv, r, a.log2G, n_rows, k_begin, k_end, n_tiles, a.scale_log2, s_base, sQ, smem, bars, phase, tid, bar_id);
    float *sO = reinterpret_cast<float *>(smem);             // [4][16][D]
    float *sM = sO + 4 * 16 * D;                             // [4][16]
    float *sL = sM + 4 * 16;                                 // [4][16]
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
    // ---- the last split of this (request, kv head) to get here merges them all: no second kernel, no launch gap
    int *s_last = reinterpret_cast<int *>(s_pages + kMaxSplitPages);
    __threadfence();
    group_sync(bar_id);
    if (tid == 0) {
        int *ticket = a.tickets + ri * a.Hkv + g;
        const int arrived = r.n_splits > 1 ? atomicAdd(ticket, 1) : 0;
        const int last = arrived == r.n_splits - 1;
        if (last && r.n_splits > 1) *ticket = 0;  // everyone else has been here: the counter is zero again for the next kernel
        *s_last = last;
    }
    group_sync(bar_id);
    if (*s_last) {
        __threadfence();
        merge_rows<D>(a, r, g, tid);
    }
}

// grid = decode CTAs of the call (one item each).  INLINE: the requests of a small decode-only call ride in the kernel
// parameters (no metadata upload launch).
// The 1024-byte aligned start of the dynamic shared memory, with the ring's mbarriers initialised (count 1: the
// issuing thread's arrive.expect_tx) by the time every thread returns.
template <int D>
__device__ __forceinline__ unsigned char *ring_setup(unsigned char *smem_raw, const CUtensorMap *tmap_k, const CUtensorMap *tmap_v) {
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + kSmemAlign - 1) & ~uintptr_t(kSmemAlign - 1));
    if (threadIdx.x == 0) {
        const uint32_t bars = smem_u32(smem + group_smem<D>() - 32);
#pragma unroll
        for (int s = 0; s < kStages; ++s) ptx::mbar_init(bars + 8 * s, 1);
        ptx::fence_mbar_init();
        ptx::prefetch_tmap(tmap_k);
        ptx::prefetch_tmap(tmap_v);
    }
    __syncthreads();
    return smem;
}

// grid = decode CTAs of the call (one item each).  INLINE: the requests of a small decode-only call ride in the kernel
// parameters (no metadata upload launch).
template <int D, bool INLINE>
__global__ void __launch_bounds__(kThreads)
flash_mma_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v,
                 const __grid_constant__ InlineReqs ir, const AttnArgs a) {
    extern __shared__ unsigned char smem_raw[];
    // programmatic dependent launch: staged behind the kernel before it (the append, the metadata upload), with the
    // prefill kernel of a mixed call staged behind it; the ring is set up, then everything else waits for that kernel
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    unsigned char *smem = ring_setup<D>(smem_raw, &tmap_k, &tmap_v);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    uint32_t phase = 0;
    decode_item<D>(a, &tmap_k, &tmap_v, INLINE ? ir.reqs : a.reqs, a.n_reqs, blockIdx.x, smem, phase, threadIdx.x, 0);
}

// Captured decode step (sa_decode_step_enqueue): the launch is recorded once and replayed on batches whose size and
// lengths change, so the grid is fixed and the counts are read on the device (dyn = {requests, items} in the step's
// metadata); the CTAs stride over the items.  Which CTA runs an item does not enter its arithmetic.
template <int D>
__global__ void __launch_bounds__(kThreads, 3)
flash_mma_loop_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v, const AttnArgs a) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = ring_setup<D>(smem_raw, &tmap_k, &tmap_v);
    // programmatic dependent launch: this grid is staged while the step's append kernel runs and waits here for its
    // results (the metadata twin, the new token in the cache, the rotated q)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // the step's whole request array (a.n_reqs = its capacity; entries past the count are never looked at) comes into
    // shared memory together with the counts: one global round trip instead of a binary search of dependent ones
    ReqMeta *s_reqs = reinterpret_cast<ReqMeta *>(smem + group_smem<D>());
    const bool cached = a.n_reqs <= kLoopReqCache;
    if (cached)
        for (int i = threadIdx.x; i < a.n_reqs * int(sizeof(ReqMeta) / 16); i += kThreads)
            reinterpret_cast<uint4 *>(s_reqs)[i] = reinterpret_cast<const uint4 *>(a.reqs)[i];
    const int n_reqs = a.dyn[0], n_items = a.dyn[1];
    __syncthreads();
    uint32_t phase = 0;  // parity each ring stage's mbarrier completes with next; carried from item to item
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        decode_item<D>(a, &tmap_k, &tmap_v, cached ? s_reqs : a.reqs, n_reqs, item, smem, phase, threadIdx.x, 0);
        // the merge scratch, the page list and the zeroed V rows of this item live where the next item's ring goes:
        // generic-proxy stores before the async proxy's
        ptx::fence_proxy_async_smem();
        group_sync(0);
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
    a.block_table = pool->block_table;
    a.tickets = pool->tickets;
    a.mpps = pool->max_pages_per_session;
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


template <int D, bool INLINE>
cudaError_t launch_flash(const sa_kv_pool *pool, const InlineReqs &ir, const AttnArgs &a, int items, cudaStream_t stream,
                         int32_t *launches) {
    constexpr size_t smem = group_smem<D>() + kSmemAlign;
    const CUtensorMap &tk = *reinterpret_cast<const CUtensorMap *>(pool->tmap_k);
    const CUtensorMap &tv = *reinterpret_cast<const CUtensorMap *>(pool->tmap_v);
    static_assert(size_t(kStages) * 2 * kBN * D * 2 >= 4 * 16 * D * 4 + 2 * 4 * 16 * 4, "merge scratch must fit in the stage ring");
    cudaError_t e = opt_in_smem<&flash_mma_kernel<D, INLINE>>(smem);
    if (e != cudaSuccess) return e;
    e = launch_pdl(flash_mma_kernel<D, INLINE>, dim3(unsigned(items)), dim3(kThreads), smem, stream, tk, tv, ir, a);
    if (e != cudaSuccess) return e;
    ++*launches;
    return e;
}

template <int D>
cudaError_t launch_flash_loop(const sa_kv_pool *pool, const AttnArgs &a, int n_cta, cudaStream_t stream, int32_t *launches) {
    constexpr size_t smem = group_smem<D>() + kLoopReqCache * sizeof(ReqMeta) + kSmemAlign;
    const CUtensorMap &tk = *reinterpret_cast<const CUtensorMap *>(pool->tmap_k);
    const CUtensorMap &tv = *reinterpret_cast<const CUtensorMap *>(pool->tmap_v);
    cudaError_t e = opt_in_smem<&flash_mma_loop_kernel<D>>(smem);
    if (e != cudaSuccess) return e;
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(unsigned(n_cta));
        cfg.blockDim = dim3(kThreads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, flash_mma_loop_kernel<D>, tk, tv, a);
    }
    if (e != cudaSuccess) return e;
    ++*launches;
    return e;
}

}  // namespace

cudaError_t flash_loop_prepare(const sa_kv_pool *pool) {
    return pool->cfg.head_dim == 128
               ? opt_in_smem<&flash_mma_loop_kernel<128>>(group_smem<128>() + kLoopReqCache * sizeof(ReqMeta) + kSmemAlign)
               : opt_in_smem<&flash_mma_loop_kernel<64>>(group_smem<64>() + kLoopReqCache * sizeof(ReqMeta) + kSmemAlign);
}

// reqs_host != nullptr (and plan.n_dec <= kInlineReqs): the requests go in the kernel parameters, reqs_dev is unused.
// dyn != nullptr (captured step): loop_ctas CTAs stride over the items, plan.n_dec is the capacity of the step's
// request array, the actual counts come from dyn.
cudaError_t launch_flash_decode(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const ReqMeta *reqs_host,
                                const AttnPlan &plan, const void *q, void *out, float *lse, float sm_scale,
                                float *part_o, float *part_lse, cudaStream_t stream, int32_t *launches,
                                int loop_ctas, const int32_t *dyn) {
    if (plan.dec_items == 0 && !dyn) return cudaSuccess;
    if (!pool->tc5_ready) return cudaErrorNotSupported;  // the TMA descriptors over the pages are built with the pool
    AttnArgs a = make_args(pool, reqs_dev, plan.n_dec, q, out, lse, sm_scale, part_o, part_lse);
    a.dyn = dyn;
    const bool d128 = pool->cfg.head_dim == 128;
    if (reqs_host) {
        InlineReqs ir;
        memcpy(ir.reqs, reqs_host, sizeof(ReqMeta) * size_t(plan.n_dec));
        return d128 ? launch_flash<128, true>(pool, ir, a, plan.dec_items, stream, launches)
                    : launch_flash<64, true>(pool, ir, a, plan.dec_items, stream, launches);
    }
    if (dyn)
        return d128 ? launch_flash_loop<128>(pool, a, loop_ctas, stream, launches)
                    : launch_flash_loop<64>(pool, a, loop_ctas, stream, launches);
    static const InlineReqs none{};  // never read by the slab variants
    return d128 ? launch_flash<128, false>(pool, none, a, plan.dec_items, stream, launches)
                : launch_flash<64, false>(pool, none, a, plan.dec_items, stream, launches);
}

}  // namespace sa
