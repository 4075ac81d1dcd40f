// sa_prefill_tc5.cu -- prefill-chunk attention over paged KV on the 5th-generation tensor cores
// (chunk j has q_j query tokens over prefix_j cached
// tokens, "the i-th query token attends to prefix_j + i + 1 tokens"; compute-bound, cost ~ A_j).
//
// An item = one (request, kv head, 256 packed rows); packed row rho is (token rho / G, q head
// g*G + rho % G), so the G query heads of a group share every K/V tile.  The kernel is persistent:
// one CTA per SM walks the list of parts (KV-tile ranges of items) that the host schedule
// (sa_tc5_schedule.cu) gave it; a part that is a whole item writes the output, a part of a split
// item writes an fp32 partial and tc5_merge_kernel combines the item's parts in KV order.
// The 256 rows are two 128-row Q tiles that ping-pong: while the softmax warps of one tile work
// on S, the tensor core runs the other tile's MMAs.  Warp roles (384 threads):
//   warp 0      TMA producer (one lane): Q tiles of the part, then page-gathered K and V tiles
//               (2-stage rings); runs ahead across part boundaries
//   warp 1      MMA issuer: S_t = Q_t K_j^T (SS), O_t += P_t V_j (P from TMEM, V MN-major); zeroes
//               the V rows past the end of the session in an item's last tile
//   warp 2      TMEM allocator
//   warps 4-7   softmax of Q tile 0 (thread = row): S from TMEM, mask, lazy-rescaled online
//   warps 8-11  softmax of Q tile 1   softmax, P (bf16) back into the S columns in three pieces (64 + 32 + 32
//               keys, so that only two PV k-steps are left after the last exponential), epilogue
// TMEM (512 columns): S0/P0 [0,128)  S1/P1 [128,256)  O0 [256,384)  O1 [384,512).
#include <cuda.h>
#include <cuda_bf16.h>
#include <math.h>

#include "sa_internal.h"
#include "sa_tc5_ptx.cuh"

namespace sa {

namespace {

using namespace ptx;

constexpr int DMAX = 128;         // largest head_dim; the kernels are instantiated for DH = 1 or 2 halves of 64 dims
constexpr int BM = 128;           // rows per Q tile
constexpr int BN = 128;           // keys per KV tile
constexpr int kThreadsTc5 = 384;
constexpr int TILE_BYTES = BN * DMAX * 2;   // 32 KiB: two 64-wide halves of 128 rows x 128 B (head_dim 64 uses the first)
constexpr int HALF_BYTES = TILE_BYTES / 2;
constexpr int KV_STAGES = 2;
constexpr int kPolyShare = 2;  // of every 8 column pairs, this many take exp2 as a packed cubic on the FMA pipe, the rest the MUFU
constexpr float kRescaleThreshold = 8.0f;  // log2 units: rescale O only when the row max grows by > 2^8


struct Tc5Args {
    const ReqMeta *reqs;
    const int32_t *cta_begin;  // [gridDim.x + 1] into parts
    const Tc5Part *parts;
    const Tc5Merge *merges;
    char *partials;            // [n_slots] x kTc5SlotBytes
    const int32_t *block_table;
    int64_t mpps;
    __nv_bfloat16 *out;
    float *lse;
    int32_t Hq, Hkv, log2G;
    float scale_log2;
};

enum Bar {
    BAR_Q_FULL = 0,
    BAR_Q_EMPTY = 1,
    BAR_K_FULL = 2,   // [2]
    BAR_K_EMPTY = 4,  // [2]
    BAR_V_FULL = 6,   // [2]
    BAR_V_EMPTY = 8,  // [2]
    BAR_S_FULL = 10,  // [2] per Q tile
    BAR_P_A = 12,     // [2] P columns of keys 0..63 of the tile are in TMEM
    BAR_P_B = 14,     // [2] ... keys 64..95
    BAR_P_C = 16,     // [2] ... keys 96..127
    BAR_O_FULL = 18,  // [2] all PV products of the part have landed in O_t
    BAR_O_EMPTY = 20, // [2] the epilogue has read O_t out of TMEM
    BAR_COUNT = 22
};

// Everything a role needs to know about one part; every role derives the same values.
struct PartGeom {
    ReqMeta r;
    int g, rho0, base_lim, u0, u1, slot, pages_needed, valid_last;
    bool fix_last;  // the part ends on the item's last KV tile and that tile has rows past the session end
};

template <int LOG2B>
__device__ __forceinline__ PartGeom load_part(const Tc5Args &a, int p) {
    constexpr int B = 1 << LOG2B;
    constexpr int PAGES_PER_TILE = BN / B;
    const Tc5Part pt = a.parts[p];
    PartGeom gm;
    gm.r = a.reqs[pt.req];
    gm.g = pt.g;
    gm.u0 = pt.u0;
    gm.u1 = pt.u1;
    gm.slot = pt.slot;
    gm.rho0 = pt.tile * (2 * BM);
    gm.base_lim = gm.r.kv_len - gm.r.q_len;
    const int tok_max = min(gm.r.q_len - 1, (gm.rho0 + 2 * BM - 1) >> a.log2G);
    const int k_end = gm.base_lim + tok_max + 1;                   // keys [0, k_end) are needed
    const int n_kv = (k_end + BN - 1) / BN;
    gm.pages_needed = (k_end + B - 1) >> LOG2B;
    // last tile: rows at or past `valid_last` hold no session data (unloaded pages or slots >= kv_len)
    const int last_pages = min(PAGES_PER_TILE, gm.pages_needed - (n_kv - 1) * PAGES_PER_TILE);
    gm.valid_last = min(gm.r.kv_len - (n_kv - 1) * BN, last_pages * B);
    gm.fix_last = pt.u1 == n_kv && gm.valid_last < BN;
    return gm;
}

// ---- per-chunk pieces of the softmax (a chunk = 32 of the 128 S columns of a row, in registers)
__device__ __forceinline__ void chunk_mask(uint32_t (&s)[32], int key0, int lim) {
#pragma unroll
    for (int i = 0; i < 32; ++i)
        if (key0 + i > lim) s[i] = 0xff800000u;  // -inf: selected, never added
}
__device__ __forceinline__ float max3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }  // one FMNMX3
// max of the 32 columns of a chunk as a tree of depth 4 (a serial chain would expose the FMNMX3 latency 16 times)
__device__ __forceinline__ float chunk_max(const uint32_t (&s)[32]) {
    float l1[10];
#pragma unroll
    for (int i = 0; i < 10; ++i)
        l1[i] = max3(__uint_as_float(s[3 * i]), __uint_as_float(s[3 * i + 1]), __uint_as_float(s[3 * i + 2]));
    const float a0 = max3(l1[0], l1[1], l1[2]), a1 = max3(l1[3], l1[4], l1[5]), a2 = max3(l1[6], l1[7], l1[8]);
    const float a3 = max3(l1[9], __uint_as_float(s[30]), __uint_as_float(s[31]));
    return fmaxf(max3(a0, a1, a2), a3);
}
// exp2 of column pairs [I0, I1) of one chunk, row sums, bf16 P packed into pk.  kPolyShare of every eight column
// pairs take the packed cubic on the FMA pipe (never on masked tiles: -inf must give exactly 0).
template <bool MASKED, int I0, int I1>
__device__ __forceinline__ void chunk_exp(const uint32_t (&s)[32], uint64_t sl2_2, uint64_t neg_2, uint64_t (&lsum)[4],
                                          uint32_t (&pk)[16]) {
#pragma unroll
    for (int i = I0; i < I1; ++i) {
        // x = s * scale_log2 - m * scale_log2 for two columns at once (FFMA2)
        float x0, x1;
        unpack_f32x2(ffma2(pack_f32x2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), sl2_2, neg_2), x0, x1);
        float p0, p1;
        if (!MASKED && (i & 7) < kPolyShare) {
            ex2_poly3_x2(x0, x1, p0, p1);
        } else {
            p0 = ex2_approx(x0);
            p1 = ex2_approx(x1);
        }
        lsum[i & 3] = fadd2(lsum[i & 3], pack_f32x2(p0, p1));
        __nv_bfloat162 pb = __floats2bfloat162_rn(p0, p1);
        pk[i] = *reinterpret_cast<uint32_t *>(&pb);
    }
}
// a whole chunk into 16 TMEM columns
template <bool MASKED>
__device__ __forceinline__ void chunk_exp_store(const uint32_t (&s)[32], uint64_t sl2_2, uint64_t neg_2, uint64_t (&lsum)[4],
                                                uint32_t taddr) {
    uint32_t pk[16];
    chunk_exp<MASKED, 0, 16>(s, sl2_2, neg_2, lsum, pk);
    tmem_st16(taddr, pk);
}
// P of the chunks stored so far is in TMEM: tell the MMA warp
__device__ __forceinline__ void publish_p(uint32_t bar_addr) {
    tmem_wait_st();
    tc_fence_before();
    mbar_arrive(bar_addr);
}

template <int LOG2B, int DH>
__global__ void __launch_bounds__(kThreadsTc5, 1)
prefill_tc5_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
                   const __grid_constant__ CUtensorMap tmap_v, const Tc5Args a) {
    constexpr int B = 1 << LOG2B;
    constexpr int D = DH * 64;                     // head_dim: DH halves of 64 dims (one SWIZZLE_128B atom each)
    constexpr int PAGES_PER_TILE = BN / B;
    constexpr uint32_t PAGE_HALF_BYTES = B * 128;  // one page, one 64-wide half: B rows x 128 B

    // Programmatic dependent launch: the grid is staged while the kernel before it in the stream (the metadata upload,
    // or the decode rows' kernel of a mixed call) still runs; barriers and TMEM are set up, then everything that the
    // stream orders -- the schedule, the requests, K/V, Q -- waits for that kernel.  The merge kernel is staged behind.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t sQ = smem_u32(smem);                 // 2 tiles x 32 KiB
    const uint32_t sK = sQ + 2 * TILE_BYTES;            // KV_STAGES x 32 KiB
    const uint32_t sV = sK + KV_STAGES * TILE_BYTES;    // KV_STAGES x 32 KiB
    __shared__ uint64_t bars[BAR_COUNT];
    __shared__ uint32_t tmem_base_smem;
    const uint32_t bar0 = smem_u32(&bars[0]);
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * uint32_t(i); };

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    if (tid == 0) {
        mbar_init(bar(BAR_Q_FULL), 1);
        mbar_init(bar(BAR_Q_EMPTY), 1);
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(BAR_K_FULL + s), 1);
            mbar_init(bar(BAR_K_EMPTY + s), 1);
            mbar_init(bar(BAR_V_FULL + s), 1);
            mbar_init(bar(BAR_V_EMPTY + s), 1);
            mbar_init(bar(BAR_S_FULL + s), 1);
            mbar_init(bar(BAR_P_A + s), BM);
            mbar_init(bar(BAR_P_B + s), BM);
            mbar_init(bar(BAR_P_C + s), BM);
            mbar_init(bar(BAR_O_FULL + s), 1);
            mbar_init(bar(BAR_O_EMPTY + s), BM);
        }
        fence_mbar_init();
    }
    if (warp == 2) tmem_alloc<512>(smem_u32(&tmem_base_smem));
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_smem;
    asm volatile("griddepcontrol.wait;" ::: "memory");

    // ---- the parts of this persistent CTA (uniform over the CTA: an idle CTA gives its TMEM back and leaves)
    const int pb = a.cta_begin[blockIdx.x], pe = a.cta_begin[blockIdx.x + 1];
    if (pb == pe) {
        if (warp == 2) tmem_dealloc<512>(tmem);
        return;
    }

    // Phase bookkeeping shared by all roles: kc counts the KV tiles this CTA has gone through (K/V
    // ring stage kc & 1, ring phase (kc >> 1) & 1; S/P barriers complete once per tile: phase
    // kc & 1), pc = p - pb counts its parts (Q, O barriers: phase pc & 1).
    // (setmaxnreg sits inside each role branch so that no control-flow merge follows it)

    if (warp == 0) {
        // =========================== TMA producer ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
        if (lane == 0) {
            prefetch_tmap(&tmap_q);
            prefetch_tmap(&tmap_k);
            prefetch_tmap(&tmap_v);
            int kc = 0;
            for (int p = pb; p < pe; ++p) {
                const PartGeom gm = load_part<LOG2B>(a, p);
                // Q of this part may land once every QK product of the previous part has read its Q
                if (p > pb) mbar_wait_watched(bar(BAR_Q_EMPTY), (p - pb - 1) & 1);
                mbar_expect_tx(bar(BAR_Q_FULL), 2 * DH * HALF_BYTES);
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const int tok0 = gm.r.q_start + ((gm.rho0 + t * BM) >> a.log2G);
#pragma unroll
                    for (int h = 0; h < DH; ++h)
                        tma_load_3d(sQ + t * TILE_BYTES + h * HALF_BYTES, &tmap_q, bar(BAR_Q_FULL), h * 64, gm.g << a.log2G, tok0);
                }
                const int32_t *bt = a.block_table + int64_t(gm.r.sid) * a.mpps;
                for (int j = gm.u0; j < gm.u1; ++j, ++kc) {
                    const int s = kc & 1, ph = (kc >> 1) & 1;
                    const int p0 = j * PAGES_PER_TILE;
                    const int np = min(PAGES_PER_TILE, gm.pages_needed - p0);
                    int32_t pg[PAGES_PER_TILE];
#pragma unroll
                    for (int u = 0; u < PAGES_PER_TILE; ++u) pg[u] = u < np ? __ldg(bt + p0 + u) : 0;
                    mbar_wait_watched(bar(BAR_K_EMPTY + s), ph ^ 1);
                    mbar_expect_tx(bar(BAR_K_FULL + s), uint32_t(np) * DH * PAGE_HALF_BYTES);
#pragma unroll
                    for (int u = 0; u < PAGES_PER_TILE; ++u)
                        if (u < np) {
                            tma_load_4d(sK + s * TILE_BYTES + u * PAGE_HALF_BYTES, &tmap_k, bar(BAR_K_FULL + s), 0, 0, gm.g, pg[u]);
                            if (DH == 2) tma_load_4d(sK + s * TILE_BYTES + HALF_BYTES + u * PAGE_HALF_BYTES, &tmap_k, bar(BAR_K_FULL + s), 64, 0, gm.g, pg[u]);
                        }
                    mbar_wait_watched(bar(BAR_V_EMPTY + s), ph ^ 1);
                    mbar_expect_tx(bar(BAR_V_FULL + s), uint32_t(np) * DH * PAGE_HALF_BYTES);
#pragma unroll
                    for (int u = 0; u < PAGES_PER_TILE; ++u)
                        if (u < np) {
                            tma_load_4d(sV + s * TILE_BYTES + u * PAGE_HALF_BYTES, &tmap_v, bar(BAR_V_FULL + s), 0, 0, gm.g, pg[u]);
                            if (DH == 2) tma_load_4d(sV + s * TILE_BYTES + HALF_BYTES + u * PAGE_HALF_BYTES, &tmap_v, bar(BAR_V_FULL + s), 64, 0, gm.g, pg[u]);
                        }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        // The whole warp walks the loop and waits on the barriers; lane 0 issues.  (All lanes are
        // needed once per item: V rows past the session end must be zeroed, see fix_last.)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
        constexpr uint32_t idesc_qk = umma_idesc_bf16(BM, BN, false, false);
        constexpr uint32_t idesc_pv = umma_idesc_bf16(BM, D, false, true);
        // descriptors are built once; an operand at a fixed offset is one 64-bit add away
        const uint64_t dq0 = umma_desc(sQ, 16, 1024), dk0 = umma_desc(sK, 16, 1024), dv0 = umma_desc(sV, HALF_BYTES, 1024);
        auto issue_qk = [&](int t, int s) {
            const uint64_t dq = umma_desc_adv(dq0, t * TILE_BYTES), dk = umma_desc_adv(dk0, s * TILE_BYTES);
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const uint32_t off = (ks >> 2) * HALF_BYTES + (ks & 3) * 32;
                umma_ss(tmem + t * BN, umma_desc_adv(dq, off), umma_desc_adv(dk, off), idesc_qk, ks > 0);
            }
        };
        auto issue_pv = [&](int t, int s, int ks0, int nks, bool acc) {  // nks k-steps of 16 keys from k-step ks0
            const uint64_t dv = umma_desc_adv(dv0, s * TILE_BYTES);
#pragma unroll
            for (int ks = ks0; ks < ks0 + nks; ++ks)
                umma_ts(tmem + 2 * BN + t * DMAX, tmem + t * BN + ks * 8, umma_desc_adv(dv, ks * 2048), idesc_pv, acc || ks > ks0);
        };
        // S_t of the first KV tile of a part; `single`: that tile is also the part's last, so its
        // second QK product is the last reader of the part's Q
        auto issue_first_qk = [&](int t, int s, bool single) {
            if (elect_one()) {
                issue_qk(t, s);
                umma_commit(bar(BAR_S_FULL + t));
                if (t == 1) {
                    umma_commit(bar(BAR_K_EMPTY + s));
                    if (single) umma_commit(bar(BAR_Q_EMPTY));
                }
            }
            __syncwarp();
        };
        int kc = 0;
        PartGeom gm = load_part<LOG2B>(a, pb);
        mbar_wait(bar(BAR_Q_FULL), 0);
        mbar_wait(bar(BAR_K_FULL + 0), 0);
        tc_fence_after();
        issue_first_qk(0, 0, gm.u1 - gm.u0 == 1);
        issue_first_qk(1, 0, gm.u1 - gm.u0 == 1);
        for (int p = pb; p < pe; ++p) {
            const bool has_next_part = p + 1 < pe;
            PartGeom gn = gm;
            if (has_next_part) gn = load_part<LOG2B>(a, p + 1);
            for (int j = gm.u0; j < gm.u1; ++j, ++kc) {
                const int s = kc & 1, ph = (kc >> 1) & 1;
                const int sn = s ^ 1, phn = ((kc + 1) >> 1) & 1;
                const bool last = j == gm.u1 - 1;
                mbar_wait(bar(BAR_V_FULL + s), ph);
                if (last && gm.fix_last) {
                    // V rows that hold no session data must be exactly zero: P is 0 there, and 0 * NaN = NaN
                    const int n_zero = BN - gm.valid_last;  // rows [valid_last, 128), DH halves x 8 chunks of 16 B each
                    for (int e = lane; e < n_zero * (8 * DH); e += 32) {
                        const int row = gm.valid_last + e / (8 * DH), hc = e % (8 * DH);
                        const uint32_t addr = sV + s * TILE_BYTES + (hc >> 3) * HALF_BYTES + row * 128 + (hc & 7) * 16;
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(addr), "r"(0) : "memory");
                    }
                    fence_proxy_async_smem();
                    __syncwarp();
                }
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    // the first PV product of a part overwrites O_t: the previous part's epilogue must have read it
                    if (j == gm.u0 && p > pb) mbar_wait(bar(BAR_O_EMPTY + t), (p - pb - 1) & 1);
                    // P arrives in three pieces (64 + 32 + 32 keys): the products of the first 96 keys run under
                    // the remaining exponentials and only two k-steps are left after the last one
                    mbar_wait(bar(BAR_P_A + t), kc & 1);
                    tc_fence_after();
                    if (elect_one()) issue_pv(t, s, 0, 4, j > gm.u0);
                    __syncwarp();
                    mbar_wait(bar(BAR_P_B + t), kc & 1);
                    tc_fence_after();
                    if (elect_one()) issue_pv(t, s, 4, 2, true);
                    __syncwarp();
                    mbar_wait(bar(BAR_P_C + t), kc & 1);
                    tc_fence_after();
                    if (elect_one()) {
                        issue_pv(t, s, 6, 2, true);
                        if (t == 1) umma_commit(bar(BAR_V_EMPTY + s));
                    }
                    __syncwarp();
                    if (!last) {
                        if (t == 0) {
                            mbar_wait(bar(BAR_K_FULL + sn), phn);
                            tc_fence_after();
                        }
                        issue_first_qk(t, sn, j + 1 == gm.u1 - 1);
                    } else {
                        if (elect_one()) umma_commit(bar(BAR_O_FULL + t));
                        __syncwarp();
                        if (has_next_part) {  // keep the tensor pipe fed across the part boundary
                            if (t == 0) {
                                mbar_wait(bar(BAR_Q_FULL), (p + 1 - pb) & 1);
                                mbar_wait(bar(BAR_K_FULL + sn), phn);
                                tc_fence_after();
                            }
                            issue_first_qk(t, sn, gn.u1 - gn.u0 == 1);
                        }
                    }
                }
            }
            gm = gn;
        }
    } else if (warp < 4) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
    } else {
        // =========================== softmax + epilogue ===========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
        const int t = (warp - 4) >> 2;                 // Q tile of this warpgroup
        const int row = ((warp & 3) << 5) + lane;      // TMEM lane == row of the tile
        const uint32_t lane_addr = tmem + (uint32_t((warp & 3) << 5) << 16);
        const uint32_t tS = lane_addr + t * BN, tO = lane_addr + 2 * BN + t * DMAX;
        const float sl2 = a.scale_log2;
        const uint64_t sl2_2 = pack_f32x2(sl2, sl2);
        const int G = 1 << a.log2G;
        int kc = 0;
        for (int p = pb; p < pe; ++p) {
            const PartGeom gm = load_part<LOG2B>(a, p);
            const int n_rows = gm.r.q_len * G;
            const int rho = gm.rho0 + t * BM + row;
            const bool valid = rho < n_rows;
            const int lim = valid ? gm.base_lim + (rho >> a.log2G) : -1;
            const int lim_min = gm.base_lim + ((gm.rho0 + t * BM) >> a.log2G);  // smallest limit among the tile's rows
            float m_used = -INFINITY;
            uint64_t lsum[4] = {0ull, 0ull, 0ull, 0ull};  // 4 x f32x2 independent partial row sums
            for (int j = gm.u0; j < gm.u1; ++j, ++kc) {
                mbar_wait(bar(BAR_S_FULL + t), kc & 1);
                tc_fence_after();
                uint32_t s0[32], s1[32], s2[32], s3[32];
                tmem_ld32(tS, s0);
                tmem_ld32(tS + 32, s1);
                tmem_ld32(tS + 64, s2);
                tmem_ld32(tS + 96, s3);
                tmem_wait_ld();
                const int kt = j * BN;
                const bool masked = kt + BN - 1 > lim_min;  // uniform over the warpgroup: diagonal / last tiles only
                if (masked) {
                    chunk_mask(s0, kt, lim);
                    chunk_mask(s1, kt + 32, lim);
                    chunk_mask(s2, kt + 64, lim);
                    chunk_mask(s3, kt + 96, lim);
                }
                const float mx = fmaxf(fmaxf(chunk_max(s0), chunk_max(s1)), fmaxf(chunk_max(s2), chunk_max(s3)));
                const float m_new = fmaxf(m_used, mx);
                const bool need = (m_new - m_used) * sl2 > kRescaleThreshold;  // true on the first live tile
                if (__any_sync(0xffffffffu, need)) {
                    const float f = need ? ex2_approx((m_used - m_new) * sl2) : 1.0f;
                    if (need) {
                        const uint64_t f2 = pack_f32x2(f, f);
#pragma unroll
                        for (int c = 0; c < 4; ++c) lsum[c] = fmul2(lsum[c], f2);
                        m_used = m_new;
                    }
                    if (j > gm.u0) {  // PV(t, j-1) has completed (it precedes QK(t, j) in the pipe); PV(t, j) waits for P
#pragma unroll
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t rr[32];
                            tmem_ld32(tO + c * 32, rr);
                            tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i) rr[i] = __float_as_uint(__uint_as_float(rr[i]) * f);
                            tmem_st32(tO + c * 32, rr);
                        }
                    }
                }
                const float neg = (m_used == -INFINITY) ? 0.f : -m_used * sl2;
                const uint64_t neg_2 = pack_f32x2(neg, neg);
                // A piece of P is published half a chunk late: by then its tcgen05.st has long landed, so
                // tcgen05.wait::st does not stall the exponentials, and its PV product still has the rest of the tile
                // to run under.  Only the last piece waits for its own store.
                if (masked) {
                    uint32_t pk[16];
                    chunk_exp_store<true>(s0, sl2_2, neg_2, lsum, tS);
                    chunk_exp_store<true>(s1, sl2_2, neg_2, lsum, tS + 16);
                    chunk_exp<true, 0, 8>(s2, sl2_2, neg_2, lsum, pk);
                    publish_p(bar(BAR_P_A + t));
                    chunk_exp<true, 8, 16>(s2, sl2_2, neg_2, lsum, pk);
                    tmem_st16(tS + 32, pk);
                    chunk_exp<true, 0, 8>(s3, sl2_2, neg_2, lsum, pk);
                    publish_p(bar(BAR_P_B + t));
                    chunk_exp<true, 8, 16>(s3, sl2_2, neg_2, lsum, pk);
                    tmem_st16(tS + 48, pk);
                } else {
                    uint32_t pk[16];
                    chunk_exp_store<false>(s0, sl2_2, neg_2, lsum, tS);
                    chunk_exp_store<false>(s1, sl2_2, neg_2, lsum, tS + 16);
                    chunk_exp<false, 0, 8>(s2, sl2_2, neg_2, lsum, pk);
                    publish_p(bar(BAR_P_A + t));
                    chunk_exp<false, 8, 16>(s2, sl2_2, neg_2, lsum, pk);
                    tmem_st16(tS + 32, pk);
                    chunk_exp<false, 0, 8>(s3, sl2_2, neg_2, lsum, pk);
                    publish_p(bar(BAR_P_B + t));
                    chunk_exp<false, 8, 16>(s3, sl2_2, neg_2, lsum, pk);
                    tmem_st16(tS + 48, pk);
                }
                publish_p(bar(BAR_P_C + t));
            }
            float l;
            {
                float a0, a1;
                unpack_f32x2(fadd2(fadd2(lsum[0], lsum[1]), fadd2(lsum[2], lsum[3])), a0, a1);
                l = a0 + a1;
            }
            // ---- epilogue of the part
            mbar_wait_watched(bar(BAR_O_FULL + t), (p - pb) & 1);
            tc_fence_after();
            if (gm.slot < 0) {
                // whole item: O / l -> bf16 -> out
                const float inv = l > 0.f ? 1.0f / l : 0.f;
                const int tok = rho >> a.log2G, hq = (gm.g << a.log2G) + (rho & (G - 1));
                const int64_t orow = int64_t(gm.r.q_start + tok) * a.Hq + hq;
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t rr[32];
                    tmem_ld32(tO + c * 32, rr);
                    tmem_wait_ld();
                    if (c == D / 32 - 1) {  // O_t is in registers: the next part's PV products may overwrite it
                        tc_fence_before();
                        mbar_arrive(bar(BAR_O_EMPTY + t));
                    }
                    if (valid) {
                        uint4 *dst = reinterpret_cast<uint4 *>(a.out + orow * D + c * 32);
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            uint32_t w[4];
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                __nv_bfloat162 pb2 = __floats2bfloat162_rn(__uint_as_float(rr[i * 8 + 2 * e]) * inv,
                                                                           __uint_as_float(rr[i * 8 + 2 * e + 1]) * inv);
                                w[e] = *reinterpret_cast<uint32_t *>(&pb2);
                            }
                            dst[i] = make_uint4(w[0], w[1], w[2], w[3]);
                        }
                    }
                }
                if (valid && a.lse) a.lse[orow] = (m_used * sl2 + log2f(l)) * 0.6931471805599453f;
            } else {
                // part of a split item: unnormalised O, running max (log2 domain) and row sum to the partial slot
                char *slot = a.partials + size_t(gm.slot) * kTc5SlotBytes;
                float *po = reinterpret_cast<float *>(slot) + size_t(t * BM + row) * DMAX;   // slot layout is head_dim-independent
                float2 *pml = reinterpret_cast<float2 *>(slot + size_t(2 * BM) * DMAX * 4) + (t * BM + row);
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t rr[32];
                    tmem_ld32(tO + c * 32, rr);
                    tmem_wait_ld();
                    if (c == D / 32 - 1) {
                        tc_fence_before();
                        mbar_arrive(bar(BAR_O_EMPTY + t));
                    }
                    if (valid) {
                        uint4 *dst = reinterpret_cast<uint4 *>(po + c * 32);
#pragma unroll
                        for (int i = 0; i < 8; ++i) dst[i] = make_uint4(rr[4 * i], rr[4 * i + 1], rr[4 * i + 2], rr[4 * i + 3]);
                    }
                }
                if (valid) *pml = make_float2(m_used * sl2, l);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc<512>(tmem);
}

// Merge of the parts of split items, in KV order (fixed, so bit-reproducible).  grid = (split
// items, 32): each CTA takes 8 of the item's 256 rows, one row per warp, lanes cover D with float4;
// the loads of up to four parts are issued together (the kernel is latency-bound otherwise).
template <int DH>
__global__ void __launch_bounds__(256) tc5_merge_kernel(const Tc5Args a) {
    asm volatile("griddepcontrol.wait;" ::: "memory");  // staged behind the prefill kernel: its partials must be complete
    constexpr int D = DH * 64;
    const Tc5Merge mg = a.merges[blockIdx.x];
    const ReqMeta r = a.reqs[mg.req];
    const int G = 1 << a.log2G;
    const int n_rows = r.q_len * G;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const char *slot0 = a.partials + size_t(mg.slot0) * kTc5SlotBytes;
    const int lrow = blockIdx.y * 8 + warp;
    const int rho = mg.tile * (2 * BM) + lrow;
    if (rho >= n_rows) return;
    auto ml_of = [&](int s) { return reinterpret_cast<const float2 *>(slot0 + size_t(s) * kTc5SlotBytes + size_t(2 * BM) * DMAX * 4)[lrow]; };
    auto o_of = [&](int s) { return reinterpret_cast<const float4 *>(slot0 + size_t(s) * kTc5SlotBytes + size_t(lrow) * DMAX * 4)[lane]; };
    float M = -INFINITY;
    for (int s = 0; s < mg.n_parts; ++s) M = fmaxf(M, ml_of(s).x);
    const float Mb = (M == -INFINITY) ? 0.f : M;
    float L = 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s0 = 0; s0 < mg.n_parts; s0 += 4) {
        float2 ml[4];
        float4 ov[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (s0 + u < mg.n_parts) {
                ml[u] = ml_of(s0 + u);
                ov[u] = lane < D / 4 ? o_of(s0 + u) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
        for (int u = 0; u < 4; ++u)  // KV order
            if (s0 + u < mg.n_parts && ml[u].x != -INFINITY) {  // -inf: the part saw no live key of this row
                const float w = exp2f(ml[u].x - Mb);
                L += ml[u].y * w;
                acc.x += ov[u].x * w;
                acc.y += ov[u].y * w;
                acc.z += ov[u].z * w;
                acc.w += ov[u].w * w;
            }
    }
    const float inv = L > 0.f ? 1.f / L : 0.f;
    const int tok = rho >> a.log2G, hq = (mg.g << a.log2G) + (rho & (G - 1));
    const int64_t orow = int64_t(r.q_start + tok) * a.Hq + hq;
    __nv_bfloat162 lo = __floats2bfloat162_rn(acc.x * inv, acc.y * inv), hi = __floats2bfloat162_rn(acc.z * inv, acc.w * inv);
    uint2 pk;
    pk.x = *reinterpret_cast<uint32_t *>(&lo);
    pk.y = *reinterpret_cast<uint32_t *>(&hi);
    if (lane < D / 4) *reinterpret_cast<uint2 *>(a.out + orow * D + lane * 4) = pk;
    if (a.lse && lane == 0) a.lse[orow] = (M + log2f(L)) * 0.6931471805599453f;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        (void)cudaGetLastError();
    }
    return fn;
}

constexpr size_t kSmemTc5 = size_t(2 + 2 * KV_STAGES) * TILE_BYTES + 1024;

}  // namespace


void *tensor_map_encode_fn() { return reinterpret_cast<void *>(get_encode()); }

// the instantiation for a (page size, head_dim) pair; nullptr if there is none
static const void *tc5_kernel_of(int page_size, int head_dim) {
    if (page_size == 64) return head_dim == 128 ? (const void *)prefill_tc5_kernel<6, 2> : (const void *)prefill_tc5_kernel<6, 1>;
    if (page_size == 16) return head_dim == 128 ? (const void *)prefill_tc5_kernel<4, 2> : (const void *)prefill_tc5_kernel<4, 1>;
    return nullptr;
}

int32_t tc5_init(sa_kv_pool *pool) {
    pool->tc5_ready = false;
    if (pool->cfg.head_dim != 64 && pool->cfg.head_dim != 128) return SA_OK;
    EncodeTiledFn enc = get_encode();
    if (!enc) return SA_ERR_CUDA;
    const sa_kv_pool_config &c = pool->cfg;
    const cuuint64_t D = cuuint64_t(c.head_dim);
    cuuint64_t dims[4] = {cuuint64_t(D), cuuint64_t(c.page_size), cuuint64_t(c.num_kv_heads), cuuint64_t(c.num_pages)};
    cuuint64_t strides[3] = {cuuint64_t(D) * 2, cuuint64_t(c.page_size) * D * 2,
                             cuuint64_t(c.num_kv_heads) * c.page_size * D * 2};
    cuuint32_t box[4] = {64, cuuint32_t(c.page_size), 1, 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    for (int w = 0; w < 2; ++w) {
        CUresult rc = enc(reinterpret_cast<CUtensorMap *>(w ? pool->tmap_v : pool->tmap_k), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
                          4, w ? pool->v_base : pool->k_base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (rc != CUDA_SUCCESS) return SA_ERR_CUDA;
    }
    const void *fn = tc5_kernel_of(c.page_size, c.head_dim);
    if (!fn || cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemTc5)) != cudaSuccess) return SA_ERR_CUDA;
    pool->tc5_ready = true;
    return SA_OK;
}

// Host-only pools (no device) report the same routing a device pool of this shape would use, so
// the planner can be tested without a GPU.
bool tc5_supported(const sa_kv_pool *pool) {
    return pool->host_only ? (pool->cfg.head_dim == 64 || pool->cfg.head_dim == 128) : pool->tc5_ready;
}

cudaError_t launch_prefill_tc5(const sa_kv_pool *pool, const ReqMeta *reqs_dev, const AttnPlan &plan,
                               const Tc5Schedule &sched, const char *sched_dev, char *partials,
                               int64_t total_q, const void *q, void *out, float *lse, float sm_scale,
                               cudaStream_t stream, int32_t *launches) {
    if (plan.n_pre == 0 || sched.parts.empty()) return cudaSuccess;
    EncodeTiledFn enc = get_encode();
    if (!enc) return cudaErrorNotSupported;
    const sa_kv_pool_config &c = pool->cfg;
    // Q as [T][Hq][D]; one box = 64 dims x G heads x 128/G tokens = a 128-row packed tile half
    alignas(64) CUtensorMap tq;
    const cuuint64_t D = cuuint64_t(c.head_dim);
    cuuint64_t dims[3] = {cuuint64_t(D), cuuint64_t(c.num_q_heads), cuuint64_t(total_q)};
    cuuint64_t strides[2] = {cuuint64_t(D) * 2, cuuint64_t(c.num_q_heads) * D * 2};
    cuuint32_t box[3] = {64, cuuint32_t(pool->G), cuuint32_t(BM / pool->G)};
    cuuint32_t es[3] = {1, 1, 1};
    if (enc(&tq, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(q), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorInvalidValue;
    const int n_cta = int(sched.cta_begin.size()) - 1;
    Tc5Args a;
    a.reqs = reqs_dev;
    a.cta_begin = reinterpret_cast<const int32_t *>(sched_dev);
    const size_t off_parts = (sched.cta_begin.size() * 4 + 31) / 32 * 32;
    a.parts = reinterpret_cast<const Tc5Part *>(sched_dev + off_parts);
    a.merges = reinterpret_cast<const Tc5Merge *>(sched_dev + off_parts + sched.parts.size() * sizeof(Tc5Part));
    a.partials = partials;
    a.block_table = pool->block_table;
    a.mpps = pool->max_pages_per_session;
    a.out = static_cast<__nv_bfloat16 *>(out);
    a.lse = lse;
    a.Hq = c.num_q_heads;
    a.Hkv = c.num_kv_heads;
    int lg = 0;
    while ((1 << lg) < pool->G) ++lg;
    a.log2G = lg;
    a.scale_log2 = sm_scale * 1.4426950408889634f;
    const CUtensorMap &tk = *reinterpret_cast<const CUtensorMap *>(pool->tmap_k);
    const CUtensorMap &tv = *reinterpret_cast<const CUtensorMap *>(pool->tmap_v);
    cudaError_t e;
    const dim3 grid{unsigned(n_cta), 1, 1}, block{unsigned(kThreadsTc5), 1, 1};
    if (c.page_size == 64 && c.head_dim == 128)
        e = launch_pdl(prefill_tc5_kernel<6, 2>, grid, block, kSmemTc5, stream, tq, tk, tv, a);
    else if (c.page_size == 64)
        e = launch_pdl(prefill_tc5_kernel<6, 1>, grid, block, kSmemTc5, stream, tq, tk, tv, a);
    else if (c.head_dim == 128)
        e = launch_pdl(prefill_tc5_kernel<4, 2>, grid, block, kSmemTc5, stream, tq, tk, tv, a);
    else
        e = launch_pdl(prefill_tc5_kernel<4, 1>, grid, block, kSmemTc5, stream, tq, tk, tv, a);
    ++*launches;
    if (e != cudaSuccess) return e;
    if (!sched.merges.empty()) {
        const dim3 mgrid(unsigned(sched.merges.size()), 32);
        e = c.head_dim == 128 ? launch_pdl(tc5_merge_kernel<2>, mgrid, dim3(256), 0, stream, a)
                              : launch_pdl(tc5_merge_kernel<1>, mgrid, dim3(256), 0, stream, a);
        ++*launches;
    }
    return e;
}

}  // namespace sa
