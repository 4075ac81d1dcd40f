// sa_gemm_tc5.cu -- the dense operators of the layer on the tcgen05 tensor cores (
// PAPER.md section 4 "GEMM", L299-303: "the projection matrices in attention (QKV and output
// projections) and the FFN layers", whose cost T_GEMM(M) depends on the forward tokens M only).
//
// One persistent warp-specialised kernel, y = x W^T with x [M, K] and W [N, K] both K-major bf16:
//   warp 0      TMA producer: a 4-stage ring of (A 128 x 64, B 256 x 64) SWIZZLE_128B tiles
//   warp 1      one lane issues tcgen05.mma 128 x 256 x 16 (cta_group::1), fp32 accumulators in TMEM
//   warp 2      TMEM allocator (all 512 columns = two 128 x 256 accumulators)
//   warps 4-7   epilogue: thread = output row, tcgen05.ld of the accumulator while the MMA warp is
//               already filling the other accumulator with the next tile
// and three epilogues (template EPI):
//   EPI_PLAIN   y = acc (+ residual), bf16                            (output / down projection)
//   EPI_SWIGLU  B tile = 128 gate rows + 128 up rows of the same FFN units:
//               act = SiLU(acc_gate) * acc_up                         (sa_swiglu)
//   EPI_QKV     a tile is two heads of the fused QKV projection: Q and K heads are rotated (RoPE,
//               half-split pairs m / m+64 sit in the same thread's row), K' and V are scattered
//               into the pool pages through the per-token slot table, Q' goes to q_out
//               (sa_qkv_rope_append: "KV cache construction", L168)
#include <cuda.h>
#include <cuda_bf16.h>

#include <algorithm>
#include <mutex>
#include <vector>

#include "sa_internal.h"
#include "sa_tc5_ptx.cuh"

namespace sa {

using namespace ptx;

namespace {

constexpr int GBM = 128, GBN = 256, GBK = 64, GSTAGES = 4;
constexpr uint32_t A_STAGE = GBM * GBK * 2;   // 16 KiB
constexpr uint32_t B_HALF = 128 * GBK * 2;    // 16 KiB: 128 rows of W
constexpr uint32_t B_STAGE = 2 * B_HALF;      // 32 KiB
constexpr uint32_t STAGE_BYTES = A_STAGE + B_STAGE;
constexpr int kGemmThreads = 256;
constexpr size_t kSmemGemm = size_t(GSTAGES) * STAGE_BYTES + 1024;
constexpr int M_GROUP = 16;  // m-tiles walked fastest, so that concurrently running CTAs share W tiles in L2

enum { EPI_PLAIN = 0, EPI_SWIGLU = 1, EPI_QKV = 2 };

struct GemmArgs {
    int64_t M;
    int32_t N;        // output features (EPI_SWIGLU: FFN units F)
    int32_t K;
    int32_t m_tiles, n_tiles;
    __nv_bfloat16 *y;
    const __nv_bfloat16 *residual;
    int64_t ldy;
    // EPI_QKV
    const float2 *cs;          // [T][64] (cos, sin) at the token's absolute position
    const int64_t *tok_off;    // [T] element offset of (page, head 0, slot, 0) in the K / V page arrays
    __nv_bfloat16 *k_base, *v_base, *q_out;
    int64_t stride_head;
    int32_t Hq, Hkv;
    // split-K (small M: too few tiles to stream the weights at HBM rate): a work unit is (tile, k slice)
    int32_t k_splits;          // >= 1
    float *partial;            // [tiles * k_splits][128 rows][256 columns] fp32 when k_splits > 1
};
constexpr size_t kPartialFloats = size_t(GBN) * GBM;  // per work unit

__device__ __forceinline__ void tile_coords(const GemmArgs &a, int t, int &mt, int &nt) {
    const int per_group = M_GROUP * a.n_tiles;
    const int g = t / per_group, r = t - g * per_group;
    const int gm = min(M_GROUP, a.m_tiles - g * M_GROUP);
    mt = g * M_GROUP + r % gm;
    nt = r / gm;
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&p);
}

// 32 fp32 accumulator values of one row -> 32 bf16 = 64 bytes at dst (16-byte aligned)
__device__ __forceinline__ void store_row32(__nv_bfloat16 *dst, const float (&f)[32], int n_valid = 32) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (8 * i >= n_valid) break;  // ragged last columns: N is a multiple of 8
        uint4 u;
        u.x = pack_bf16x2(f[8 * i + 0], f[8 * i + 1]);
        u.y = pack_bf16x2(f[8 * i + 2], f[8 * i + 3]);
        u.z = pack_bf16x2(f[8 * i + 4], f[8 * i + 5]);
        u.w = pack_bf16x2(f[8 * i + 6], f[8 * i + 7]);
        *reinterpret_cast<uint4 *>(dst + 8 * i) = u;
    }
}

__device__ __forceinline__ void ld_row32(uint32_t taddr, float (&f)[32]) {
    uint32_t r[32];
    tmem_ld32(taddr, r);
    tmem_wait_ld();
#pragma unroll
    for (int i = 0; i < 32; ++i) f[i] = __uint_as_float(r[i]);
}

// One chunk of one output row, from 32-column pieces of the fp32 accumulator row that `ld(column, f)` supplies
// (TMEM in the GEMM kernel, the sum of the k-slice partials in the split-K reduction).
//   EPI_PLAIN : chunk c in 0..7 = columns 32c..32c+31          y = acc (+ residual)
//   EPI_SWIGLU: chunk c in 0..3 = FFN units 32c..32c+31         act = SiLU(acc[gate]) * acc[128 + up]
//   EPI_QKV   : chunk c in 0..3 = head c>>1, dims m0..m0+31 and 64+m0.. with m0 = 32 (c & 1): RoPE, scatter
template <int EPI> constexpr int epi_chunks() { return EPI == EPI_PLAIN ? 8 : 4; }

template <int EPI, class Load>
__device__ __forceinline__ void epi_chunk(const GemmArgs &a, int nt, int64_t row, bool live, int c, Load ld) {
    if (EPI == EPI_PLAIN) {
        const int col = nt * GBN + c * 32;
        if (col >= a.N) return;  // uniform over the CTA
        float f[32];
        ld(c * 32, f);
        if (live) {
            __nv_bfloat16 *dst = a.y + row * a.ldy + col;
            if (a.residual) {
                const __nv_bfloat16 *rs = a.residual + row * a.ldy + col;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (col + 8 * i >= a.N) break;
                    const uint4 u = *reinterpret_cast<const uint4 *>(rs + 8 * i);
                    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        f[8 * i + 2 * j] += __uint_as_float(w[j] << 16);
                        f[8 * i + 2 * j + 1] += __uint_as_float(w[j] & 0xffff0000u);
                    }
                }
            }
            store_row32(dst, f, a.N - col);
        }
    } else if (EPI == EPI_SWIGLU) {
        const int col = nt * 128 + c * 32;
        if (col >= a.N) return;
        float g[32], u[32];
        ld(c * 32, g);
        ld(128 + c * 32, u);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const float e = ex2_approx(-1.4426950408889634f * g[i]);
            g[i] = __fdividef(g[i], 1.0f + e) * u[i];
        }
        if (live) store_row32(a.y + row * a.ldy + col, g, a.N - col);
    } else {  // EPI_QKV: two heads of 128 dims per tile
        const int hh = c >> 1, m0 = (c & 1) * 32;
        const int head = nt * 2 + hh;
        if (head >= a.Hq + 2 * a.Hkv) return;
        const bool rot = head < a.Hq + a.Hkv;
        const int64_t off = live ? a.tok_off[row] : 0;
        __nv_bfloat16 *dst;
        if (head < a.Hq)
            dst = a.q_out + (row * a.Hq + head) * 128;
        else if (head < a.Hq + a.Hkv)
            dst = a.k_base + off + int64_t(head - a.Hq) * a.stride_head;
        else
            dst = a.v_base + off + int64_t(head - a.Hq - a.Hkv) * a.stride_head;
        float lo[32], hi[32];
        ld(hh * 128 + m0, lo);
        ld(hh * 128 + 64 + m0, hi);
        if (live) {
            if (rot) {
                const float4 *csp = reinterpret_cast<const float4 *>(a.cs + row * 64 + m0);
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float4 c2 = __ldg(csp + i);  // (cos, sin) of dims 2i, 2i+1
                    const float x0 = lo[2 * i], x1 = hi[2 * i];
                    lo[2 * i] = fmaf(x0, c2.x, -(x1 * c2.y));
                    hi[2 * i] = fmaf(x1, c2.x, x0 * c2.y);
                    const float z0 = lo[2 * i + 1], z1 = hi[2 * i + 1];
                    lo[2 * i + 1] = fmaf(z0, c2.z, -(z1 * c2.w));
                    hi[2 * i + 1] = fmaf(z1, c2.z, z0 * c2.w);
                }
            }
            store_row32(dst + m0, lo);
            store_row32(dst + 64 + m0, hi);
        }
    }
}

template <int EPI>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_tc5_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b0,
                const __grid_constant__ CUtensorMap tmap_b1, const GemmArgs a) {
    extern __shared__ unsigned char smem_raw[];
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the next kernel of the stream may be staged behind this one
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t s0 = smem_u32(smem);
    __shared__ uint64_t bars[2 * GSTAGES + 4];
    __shared__ uint32_t tmem_base_smem;
    const uint32_t bar0 = smem_u32(&bars[0]);
    auto bar_full = [&](int s) -> uint32_t { return bar0 + 8u * uint32_t(s); };
    auto bar_empty = [&](int s) -> uint32_t { return bar0 + 8u * uint32_t(GSTAGES + s); };
    auto bar_acc_full = [&](int b) -> uint32_t { return bar0 + 8u * uint32_t(2 * GSTAGES + b); };
    auto bar_acc_empty = [&](int b) -> uint32_t { return bar0 + 8u * uint32_t(2 * GSTAGES + 2 + b); };

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int k_steps = a.K / GBK;
    const int KS = a.k_splits;
    const int n_units = a.m_tiles * a.n_tiles * KS;  // unit u = (tile u / KS, k slice u % KS)
    auto k_range = [&](int u, int &t, int &k0, int &k1) {
        t = u / KS;
        const int sl = u - t * KS;
        k0 = int(int64_t(sl) * k_steps / KS);
        k1 = int(int64_t(sl + 1) * k_steps / KS);
    };

    if (tid == 0) {
        for (int s = 0; s < GSTAGES; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_empty(s), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_acc_full(b), 1);
            mbar_init(bar_acc_empty(b), 128);
        }
        fence_mbar_init();
    }
    if (warp == 2) tmem_alloc<512>(smem_u32(&tmem_base_smem));
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_smem;

    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            prefetch_tmap(&tmap_a);
            prefetch_tmap(&tmap_b0);
            prefetch_tmap(&tmap_b1);
            // Programmatic dependent launch: this grid may be staged while the kernel before it in the stream still runs.
            // The weights (B) depend on nothing, so the B halves of the first GSTAGES stages are requested at once;
            // the activations (A) are what the previous kernel wrote: they wait for it.
            auto walk = [&](int phase) {  // 0: B of the first GSTAGES k-steps; 1: their A, then every later k-step whole
                int kc = 0;
                for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
                    int t, k0, k1, mt, nt;
                    k_range(u, t, k0, k1);
                    tile_coords(a, t, mt, nt);
                    const int m0 = mt * GBM;
                    const int r0 = EPI == EPI_SWIGLU ? nt * 128 : nt * GBN;        // rows of W (b0)
                    const int r1 = EPI == EPI_SWIGLU ? nt * 128 : nt * GBN + 128;  // rows of the second half (b1)
                    for (int ks = k0; ks < k1; ++ks, ++kc) {
                        const bool early = kc < GSTAGES;
                        if (phase == 0 && !early) return;
                        const int s = kc % GSTAGES, ph = (kc / GSTAGES) & 1;
                        const uint32_t sA = s0 + s * STAGE_BYTES, sB = sA + A_STAGE;
                        if (!early) mbar_wait_watched(bar_empty(s), ph ^ 1);
                        if (phase == 0 || !early) {
                            mbar_expect_tx(bar_full(s), STAGE_BYTES);
                            tma_load_2d(sB, &tmap_b0, bar_full(s), ks * GBK, r0);
                            tma_load_2d(sB + B_HALF, &tmap_b1, bar_full(s), ks * GBK, r1);
                        }
                        if (phase == 1) tma_load_2d(sA, &tmap_a, bar_full(s), ks * GBK, m0);
                    }
                }
            };
            walk(0);
            asm volatile("griddepcontrol.wait;" ::: "memory");
            walk(1);
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        constexpr uint32_t idesc = umma_idesc_bf16(GBM, GBN, false, false);
        const uint64_t dA0 = umma_desc(s0, 16, 1024), dB0 = umma_desc(s0 + A_STAGE, 16, 1024);
        int kc = 0, tc = 0;
        for (int u = blockIdx.x; u < n_units; u += gridDim.x, ++tc) {
            int t, k0, k1;
            k_range(u, t, k0, k1);
            const int b = tc & 1;
            mbar_wait(bar_acc_empty(b), ((tc >> 1) & 1) ^ 1);  // the epilogue has drained this accumulator
            tc_fence_after();
            for (int ks = k0; ks < k1; ++ks, ++kc) {
                const int s = kc % GSTAGES, ph = (kc / GSTAGES) & 1;
                mbar_wait(bar_full(s), ph);
                tc_fence_after();
                if (elect_one()) {  // one lane, known to the compiler: the four tcgen05.mma go out back to back
                    const uint64_t dA = umma_desc_adv(dA0, s * STAGE_BYTES), dB = umma_desc_adv(dB0, s * STAGE_BYTES);
#pragma unroll
                    for (int kk = 0; kk < GBK / 16; ++kk)
                        umma_ss(tmem + b * GBN, umma_desc_adv(dA, kk * 32), umma_desc_adv(dB, kk * 32), idesc, ks > k0 || kk > 0);
                    umma_commit(bar_empty(s));
                    if (ks == k1 - 1) umma_commit(bar_acc_full(b));
                }
                __syncwarp();
            }
        }
    } else if (warp >= 4) {
        // =========================== epilogue ===========================
        asm volatile("griddepcontrol.wait;" ::: "memory");  // everything these warps read and write belongs to the stream's order
        const int q4 = warp & 3;                 // TMEM lane quarter this warp may read
        const int row_in_tile = q4 * 32 + lane;
        const uint32_t lane_addr = uint32_t(q4 * 32) << 16;
        int tc = 0;
        for (int u = blockIdx.x; u < n_units; u += gridDim.x, ++tc) {
            const int b = tc & 1;
            int t, k0, k1, mt, nt;
            k_range(u, t, k0, k1);
            tile_coords(a, t, mt, nt);
            const int64_t row = int64_t(mt) * GBM + row_in_tile;
            const bool live = row < a.M;
            mbar_wait(bar_acc_full(b), (tc >> 1) & 1);
            tc_fence_after();
            const uint32_t acc = tmem + lane_addr + b * GBN;
            if (a.k_splits > 1) {
                // a k slice of the tile: the raw fp32 accumulator row goes to this unit's partial [128 rows][256 columns]
                float4 *dstp = reinterpret_cast<float4 *>(a.partial + size_t(u) * kPartialFloats + size_t(row_in_tile) * GBN);
#pragma unroll 1
                for (int c = 0; c < GBN / 32; ++c) {
                    float f[32];
                    ld_row32(acc + c * 32, f);
                    if (live) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) dstp[c * 8 + i] = make_float4(f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3]);
                    }
                }
            } else {
#pragma unroll 1
                for (int c = 0; c < epi_chunks<EPI>(); ++c)
                    epi_chunk<EPI>(a, nt, row, live, c, [&](int col_off, float (&f)[32]) { ld_row32(acc + col_off, f); });
            }
            tc_fence_before();
            mbar_arrive(bar_acc_empty(b));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc<512>(tmem);
}

// inverse of tile_coords
__device__ __forceinline__ int tile_index(const GemmArgs &a, int mt, int nt) {
    const int g = mt / M_GROUP;
    const int gm = min(M_GROUP, a.m_tiles - g * M_GROUP);
    return g * M_GROUP * a.n_tiles + nt * gm + (mt - g * M_GROUP);
}

// sum over the k slices, in slice order, of four consecutive accumulator columns of one row; the loads of eight
// slices go out together (one load per loop trip made the sum a chain of L2 round trips: 7 us for nine slices)
__device__ __forceinline__ float4 splitk_sum4(const GemmArgs &a, int t, int row_in_tile, int col) {
    const float4 *p = reinterpret_cast<const float4 *>(a.partial + size_t(t) * a.k_splits * kPartialFloats + size_t(row_in_tile) * GBN + col);
    float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s0 = 0; s0 < a.k_splits; s0 += 8) {
        float4 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u)
            v[u] = s0 + u < a.k_splits ? p[size_t(s0 + u) * (kPartialFloats / 4)] : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (s0 + u < a.k_splits) {
                s.x += v[u].x;
                s.y += v[u].y;
                s.z += v[u].z;
                s.w += v[u].w;
            }
    }
    return s;
}

__device__ __forceinline__ uint2 pack4(float a, float b, float c, float d) { return make_uint2(pack_bf16x2(a, b), pack_bf16x2(c, d)); }

// Split-K reduction + epilogue, elementwise: one thread = one row and four consecutive output columns (PLAIN: of
// y; SWIGLU: four FFN units; QKV: dims m..m+3 and 64+m..64+m+3 of one head).  Slices are summed in slice order,
// fixed, so the bits do not depend on which CTA ran which slice.
template <int EPI>
__global__ void __launch_bounds__(256) gemm_splitk_reduce_kernel(const GemmArgs a, int64_t n_items, int32_t items_per_row) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (e >= n_items) return;
    const int64_t row = e / items_per_row;
    const int j = int(e - row * items_per_row);
    const int mt = int(row / GBM), rit = int(row - int64_t(mt) * GBM);
    if (EPI == EPI_PLAIN) {
        const int n = j * 4, nt = n / GBN, col = n - nt * GBN;
        float4 v = splitk_sum4(a, tile_index(a, mt, nt), rit, col);
        if (a.residual) {
            const uint2 r = *reinterpret_cast<const uint2 *>(a.residual + row * a.ldy + n);
            v.x += __uint_as_float(r.x << 16);
            v.y += __uint_as_float(r.x & 0xffff0000u);
            v.z += __uint_as_float(r.y << 16);
            v.w += __uint_as_float(r.y & 0xffff0000u);
        }
        *reinterpret_cast<uint2 *>(a.y + row * a.ldy + n) = pack4(v.x, v.y, v.z, v.w);
    } else if (EPI == EPI_SWIGLU) {
        const int f = j * 4, nt = f / 128, col = f - nt * 128;
        const int t = tile_index(a, mt, nt);
        const float4 g = splitk_sum4(a, t, rit, col), u = splitk_sum4(a, t, rit, 128 + col);
        const float gg[4] = {g.x, g.y, g.z, g.w}, uu[4] = {u.x, u.y, u.z, u.w};
        float o[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float ex = ex2_approx(-1.4426950408889634f * gg[i]);
            o[i] = __fdividef(gg[i], 1.0f + ex) * uu[i];
        }
        *reinterpret_cast<uint2 *>(a.y + row * a.ldy + f) = pack4(o[0], o[1], o[2], o[3]);
    } else {
        const int head = j / 16, m = (j - head * 16) * 4;   // 16 items of 4 + 4 dims per head
        const int nt = head >> 1, hh = head & 1;
        const int t = tile_index(a, mt, nt);
        float4 lo = splitk_sum4(a, t, rit, hh * 128 + m), hi = splitk_sum4(a, t, rit, hh * 128 + 64 + m);
        __nv_bfloat16 *dst;
        if (head < a.Hq)
            dst = a.q_out + (row * a.Hq + head) * 128;
        else if (head < a.Hq + a.Hkv)
            dst = a.k_base + a.tok_off[row] + int64_t(head - a.Hq) * a.stride_head;
        else
            dst = a.v_base + a.tok_off[row] + int64_t(head - a.Hq - a.Hkv) * a.stride_head;
        if (head < a.Hq + a.Hkv) {
            const float4 *csp = reinterpret_cast<const float4 *>(a.cs + row * 64 + m);
            const float4 c01 = __ldg(csp), c23 = __ldg(csp + 1);  // (cos, sin) of dims m, m+1 | m+2, m+3
            float x0, x1;
            x0 = lo.x, x1 = hi.x, lo.x = fmaf(x0, c01.x, -(x1 * c01.y)), hi.x = fmaf(x1, c01.x, x0 * c01.y);
            x0 = lo.y, x1 = hi.y, lo.y = fmaf(x0, c01.z, -(x1 * c01.w)), hi.y = fmaf(x1, c01.z, x0 * c01.w);
            x0 = lo.z, x1 = hi.z, lo.z = fmaf(x0, c23.x, -(x1 * c23.y)), hi.z = fmaf(x1, c23.x, x0 * c23.y);
            x0 = lo.w, x1 = hi.w, lo.w = fmaf(x0, c23.z, -(x1 * c23.w)), hi.w = fmaf(x1, c23.z, x0 * c23.w);
        }
        *reinterpret_cast<uint2 *>(dst + m) = pack4(lo.x, lo.y, lo.z, lo.w);
        *reinterpret_cast<uint2 *>(dst + 64 + m) = pack4(hi.x, hi.y, hi.z, hi.w);
    }
}

// Per token of a fused QKV append: the slot it lands in and (cos, sin) of its absolute position.
__global__ void __launch_bounds__(256)
qkv_token_table_kernel(const ReqMeta *__restrict__ reqs, int32_t n_req, int64_t total_rows,
                       const int32_t *__restrict__ block_table, int64_t mpps, int32_t log2_page, int64_t stride_page,
                       const float2 *__restrict__ rope_tab, float2 *__restrict__ cs, int64_t *__restrict__ tok_off) {
    __shared__ int32_t s_pos[4];
    const int64_t t0 = int64_t(blockIdx.x) * 4;
    const int tid = threadIdx.x;
    if (tid < 4 && t0 + tid < total_rows) {
        const int64_t t = t0 + tid;
        int lo = 0, hi = n_req - 1;  // last request with q_start <= t
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (reqs[mid].q_start <= t) lo = mid; else hi = mid - 1;
        }
        const ReqMeta r = reqs[lo];
        const int32_t pos = r.kv_len + int32_t(t - r.q_start);
        const int32_t page = block_table[int64_t(r.sid) * mpps + (pos >> log2_page)];
        const int32_t slot = pos & ((1 << log2_page) - 1);
        s_pos[tid] = pos;
        tok_off[t] = int64_t(page) * stride_page + int64_t(slot) * 128;
    }
    __syncthreads();
    const int tl = tid >> 6, m = tid & 63;
    if (t0 + tl < total_rows) cs[(t0 + tl) * 64 + m] = rope_cos_sin(s_pos[tl], rope_tab[m]);
}

// RMSNorm (reading R22): one CTA per row, fp32; the row is read once (up to 8192 columns stay in registers: every
// load of a thread is in flight at the same time; a row per warp with a 16-trip load loop made the kernel a chain of
// sixteen memory round trips, 10 us for 64 rows) and the eight warps' sums of squares are combined in a fixed order.
__global__ void __launch_bounds__(256)
rmsnorm_kernel(const __nv_bfloat16 *__restrict__ x, const __nv_bfloat16 *__restrict__ w, float eps,
               __nv_bfloat16 *__restrict__ y, int64_t M, int32_t H) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __shared__ float s_part[8];
    const int64_t row = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint4 *wr = reinterpret_cast<const uint4 *>(w);
    const int nv = H / 8;
    constexpr int R = 4;  // 16-byte vectors a thread keeps (R * 256 * 8 = 8192 columns)
    uint4 g[R];
#pragma unroll
    for (int i = 0; i < R; ++i)
        if (tid + i * 256 < nv) g[i] = __ldg(wr + tid + i * 256);  // the weight depends on no earlier kernel
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint4 *xr = reinterpret_cast<const uint4 *>(x + row * H);
    uint4 *yr = reinterpret_cast<uint4 *>(y + row * H);
    uint4 u[R];
#pragma unroll
    for (int i = 0; i < R; ++i)
        if (tid + i * 256 < nv) u[i] = xr[tid + i * 256];
    auto sq = [](const uint4 &q, float ss) {
        const uint32_t v[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float a0 = __uint_as_float(v[j] << 16), a1 = __uint_as_float(v[j] & 0xffff0000u);
            ss = fmaf(a0, a0, ss);
            ss = fmaf(a1, a1, ss);
        }
        return ss;
    };
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < R; ++i)
        if (tid + i * 256 < nv) ss = sq(u[i], ss);
    for (int i = tid + R * 256; i < nv; i += 256) ss = sq(xr[i], ss);  // rows longer than 8192 columns
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if (lane == 0) s_part[warp] = ss;
    __syncthreads();
    float tot = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) tot += s_part[i];
    const float inv = rsqrtf(tot / float(H) + eps);
    auto scale = [inv](const uint4 &q, const uint4 &gq) {
        const uint32_t v[4] = {q.x, q.y, q.z, q.w}, gw[4] = {gq.x, gq.y, gq.z, gq.w};
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float a0 = __uint_as_float(v[j] << 16) * inv * __uint_as_float(gw[j] << 16);
            const float a1 = __uint_as_float(v[j] & 0xffff0000u) * inv * __uint_as_float(gw[j] & 0xffff0000u);
            o[j] = pack_bf16x2(a0, a1);
        }
        return make_uint4(o[0], o[1], o[2], o[3]);
    };
#pragma unroll
    for (int i = 0; i < R; ++i)
        if (tid + i * 256 < nv) yr[tid + i * 256] = scale(u[i], g[i]);
    for (int i = tid + R * 256; i < nv; i += 256) yr[i] = scale(xr[i], wr[i]);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// [rows][K] bf16 row-major, box = 64 columns x 128 rows, SWIZZLE_128B (rows past the end read as zeros)
bool make_tmap_2d(CUtensorMap *tm, const void *base, int64_t rows, int32_t K) {
    EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(tensor_map_encode_fn());
    if (!enc) return false;
    cuuint64_t dims[2] = {cuuint64_t(K), cuuint64_t(rows > 0 ? rows : 1)};
    cuuint64_t strides[1] = {cuuint64_t(K) * 2};
    cuuint32_t box[2] = {64, 128};
    cuuint32_t es[2] = {1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int device_sms() {
    static int sms[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 0;
    if (sms[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
        sms[dev] = n;
    }
    return sms[dev];
}

// Split-K pays when the tiles alone cannot keep the SMs streaming weights (small M: decode batches, L301
// "near-constant latency" regime): k slices per tile so that tiles x slices is about one wave.
int choose_splits(int tiles, int k_steps, int sms) {
    if (tiles <= 0 || tiles * 2 > sms) return 1;
    const int s = std::min(std::min(sms / tiles, k_steps / 2), 32);
    return s >= 2 ? s : 1;
}

template <int EPI>
cudaError_t launch_gemm(const CUtensorMap &ta, const CUtensorMap &tb0, const CUtensorMap &tb1, GemmArgs a, void *splitk_ws,
                        size_t splitk_bytes, cudaStream_t stream, int32_t *launches) {
    static bool attr_done = false;  // (per process; the attribute is set again on every device change below)
    static int attr_dev = -1;
    int dev = 0;
    cudaGetDevice(&dev);
    if (!attr_done || attr_dev != dev) {
        cudaError_t e = cudaFuncSetAttribute(gemm_tc5_kernel<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemGemm));
        if (e != cudaSuccess) return e;
        attr_done = true;
        attr_dev = dev;
    }
    const int sms = device_sms();
    if (sms <= 0) return cudaErrorNoDevice;
    const int tiles = a.m_tiles * a.n_tiles;
    int ks = choose_splits(tiles, a.K / GBK, sms);
    uintptr_t w = (reinterpret_cast<uintptr_t>(splitk_ws) + 255) & ~uintptr_t(255);
    const size_t need = size_t(tiles) * ks * kPartialFloats * sizeof(float) + 256;
    if (ks > 1 && (!splitk_ws || splitk_bytes < need)) ks = 1;  // no scratch: the unsplit kernel is always correct
    a.k_splits = ks;
    a.partial = ks > 1 ? reinterpret_cast<float *>(w) : nullptr;
    cudaError_t e = launch_pdl(gemm_tc5_kernel<EPI>, dim3(unsigned(std::min(tiles * ks, sms))), dim3(kGemmThreads), kSmemGemm, stream,
                               ta, tb0, tb1, a);
    if (launches) ++*launches;
    if (e != cudaSuccess || ks == 1) return e;
    // items of four output columns per row: PLAIN N/4 (N is a multiple of 8), SWIGLU F/4, QKV 16 per head
    const int32_t per_row = EPI == EPI_QKV ? (a.Hq + 2 * a.Hkv) * 16 : a.N / 4;
    const int64_t n_items = a.M * per_row;
    e = launch_pdl(gemm_splitk_reduce_kernel<EPI>, dim3(unsigned((n_items + 255) / 256)), dim3(256), 0, stream, a, n_items, per_row);
    if (launches) ++*launches;
    return e;
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

}  // namespace

// scratch a GEMM of M rows and `n_tiles` column tiles over K wants for split-K (0: it will not split)
size_t gemm_splitk_bytes(int64_t M, int32_t n_tiles, int32_t K) {
    const int sms = device_sms();
    if (M <= 0 || n_tiles <= 0 || K < GBK || sms <= 0) return 0;
    const int64_t tiles = (M + GBM - 1) / GBM * n_tiles;
    if (tiles * 2 > sms) return 0;
    const int ks = choose_splits(int(tiles), K / GBK, sms);
    return ks > 1 ? size_t(tiles) * ks * kPartialFloats * sizeof(float) + 512 : 0;
}
size_t gemm_plain_splitk_bytes(int64_t M, int32_t N, int32_t K) { return gemm_splitk_bytes(M, (N + GBN - 1) / GBN, K); }
size_t gemm_swiglu_splitk_bytes(int64_t M, int32_t F, int32_t K) { return gemm_splitk_bytes(M, (F + 127) / 128, K); }

// y[M, N] = x W^T (+ residual): shared by sa_linear and sa_layer_forward
int32_t gemm_plain(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N, int32_t K,
                   void *splitk_ws, size_t splitk_bytes, cudaStream_t stream, int32_t *launches) {
    if (M < 0 || N <= 0 || K <= 0) return SA_ERR_INVALID_ARG;
    if (K % GBK != 0 || N % 8 != 0 || M > (int64_t(1) << 30)) return SA_ERR_UNSUPPORTED;
    if (M == 0) return SA_OK;
    if (!x || !w || !y || !aligned16(x) || !aligned16(w) || !aligned16(y) || !aligned16(residual)) return SA_ERR_INVALID_ARG;
    alignas(64) CUtensorMap ta, tb;
    if (!make_tmap_2d(&ta, x, M, K) || !make_tmap_2d(&tb, w, N, K)) return SA_ERR_CUDA;
    GemmArgs a{};
    a.M = M;
    a.N = N;
    a.K = K;
    a.m_tiles = int32_t((M + GBM - 1) / GBM);
    a.n_tiles = (N + GBN - 1) / GBN;
    a.y = static_cast<__nv_bfloat16 *>(y);
    a.residual = static_cast<const __nv_bfloat16 *>(residual);
    a.ldy = N;
    return launch_gemm<EPI_PLAIN>(ta, tb, tb, a, splitk_ws, splitk_bytes, stream, launches) == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}

int32_t gemm_swiglu(const void *x, const void *w_gate, const void *w_up, void *act, int64_t M, int32_t F, int32_t K,
                    void *splitk_ws, size_t splitk_bytes, cudaStream_t stream, int32_t *launches) {
    if (M < 0 || F <= 0 || K <= 0) return SA_ERR_INVALID_ARG;
    if (K % GBK != 0 || F % 8 != 0 || M > (int64_t(1) << 30)) return SA_ERR_UNSUPPORTED;
    if (M == 0) return SA_OK;
    if (!x || !w_gate || !w_up || !act || !aligned16(x) || !aligned16(w_gate) || !aligned16(w_up) || !aligned16(act))
        return SA_ERR_INVALID_ARG;
    alignas(64) CUtensorMap ta, tg, tu;
    if (!make_tmap_2d(&ta, x, M, K) || !make_tmap_2d(&tg, w_gate, F, K) || !make_tmap_2d(&tu, w_up, F, K)) return SA_ERR_CUDA;
    GemmArgs a{};
    a.M = M;
    a.N = F;
    a.K = K;
    a.m_tiles = int32_t((M + GBM - 1) / GBM);
    a.n_tiles = (F + 127) / 128;
    a.y = static_cast<__nv_bfloat16 *>(act);
    a.ldy = F;
    return launch_gemm<EPI_SWIGLU>(ta, tg, tu, a, splitk_ws, splitk_bytes, stream, launches) == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}

int32_t rmsnorm(const void *x, const void *w, float eps, void *y, int64_t M, int32_t H, cudaStream_t stream) {
    if (M < 0 || H <= 0) return SA_ERR_INVALID_ARG;
    if (H % 8 != 0) return SA_ERR_UNSUPPORTED;
    if (M == 0) return SA_OK;
    if (!x || !w || !y || !aligned16(x) || !aligned16(w) || !aligned16(y)) return SA_ERR_INVALID_ARG;
    const cudaError_t e = launch_pdl(rmsnorm_kernel, dim3(unsigned(M)), dim3(256), 0, stream, static_cast<const __nv_bfloat16 *>(x),
                                     static_cast<const __nv_bfloat16 *>(w), eps, static_cast<__nv_bfloat16 *>(y), M, H);
    return e == cudaSuccess ? SA_OK : SA_ERR_CUDA;
}

static size_t qkv_tables_bytes(int64_t total) {
    const size_t T = size_t(std::max<int64_t>(total, 0));
    return (T * 64 * sizeof(float2) + 255) / 256 * 256 + (T * sizeof(int64_t) + 255) / 256 * 256 + 256;
}
// per-token tables + split-K scratch; the hidden size is not known here, so the scratch is sized for the most
// slices any K can ask for (tiles x slices never exceeds the SM count)
size_t qkv_workspace_bytes(const sa_kv_pool *pool, int64_t total) {
    const int sms = device_sms();
    const int64_t n_tiles = ((pool->cfg.num_q_heads + 2 * pool->cfg.num_kv_heads) * 128 + GBN - 1) / GBN;
    const int64_t tiles = (std::max<int64_t>(total, 0) + GBM - 1) / GBM * n_tiles;
    const size_t scratch = (sms > 0 && tiles > 0 && tiles * 2 <= sms) ? size_t(sms) * kPartialFloats * sizeof(float) + 512 : 0;
    return qkv_tables_bytes(total) + scratch;
}

// the device half of sa_qkv_rope_append, after append_prepare has placed the tokens
int32_t qkv_rope_append_device(sa_kv_pool *pool, const ReqMeta *reqs_dev, int32_t n_req, int64_t total, const void *h,
                               const void *w_qkv, int32_t hidden, void *q_out, void *workspace, size_t workspace_bytes,
                               cudaStream_t stream) {
    const sa_kv_pool_config &c = pool->cfg;
    const int32_t N = (c.num_q_heads + 2 * c.num_kv_heads) * 128;
    uintptr_t w = (reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255);
    float2 *cs = reinterpret_cast<float2 *>(w);
    int64_t *tok_off = reinterpret_cast<int64_t *>(w + (size_t(total) * 64 * sizeof(float2) + 255) / 256 * 256);
    qkv_token_table_kernel<<<unsigned((total + 3) / 4), 256, 0, stream>>>(reqs_dev, n_req, total, pool->block_table,
                                                                          pool->max_pages_per_session, pool->log2_page,
                                                                          pool->stride_page, pool->rope_tab, cs, tok_off);
    if (cudaGetLastError() != cudaSuccess) return SA_ERR_CUDA;
    ++pool->last_launches;
    alignas(64) CUtensorMap ta, tb;
    if (!make_tmap_2d(&ta, h, total, hidden) || !make_tmap_2d(&tb, w_qkv, N, hidden)) return SA_ERR_CUDA;
    GemmArgs a{};
    a.M = total;
    a.N = N;
    a.K = hidden;
    a.m_tiles = int32_t((total + GBM - 1) / GBM);
    a.n_tiles = (N + GBN - 1) / GBN;
    a.cs = cs;
    a.tok_off = tok_off;
    a.k_base = static_cast<__nv_bfloat16 *>(pool->k_base);
    a.v_base = static_cast<__nv_bfloat16 *>(pool->v_base);
    a.q_out = static_cast<__nv_bfloat16 *>(q_out);
    a.stride_head = pool->stride_head;
    a.Hq = c.num_q_heads;
    a.Hkv = c.num_kv_heads;
    const size_t tables = qkv_tables_bytes(total);
    char *scratch = reinterpret_cast<char *>(w) + tables;
    const size_t used = size_t(scratch - static_cast<char *>(workspace));
    if (launch_gemm<EPI_QKV>(ta, tb, tb, a, scratch, workspace_bytes > used ? workspace_bytes - used : 0, stream,
                             &pool->last_launches) != cudaSuccess)
        return SA_ERR_CUDA;
    return SA_OK;
}

}  // namespace sa


// ---------------------------------------------------------------------------------------------------------------
// sa_linear_noalloc: the split-K linear for callers that have no way to get device scratch.
//
// Who that is: code that is handed its input and output tensors by something else and has no allocator of its
// own to turn to -- an operator plugged into a serving engine whose memory plan was fixed at start-up, a worker
// whose whole HBM share was given to the KV pool and the weights (the normal state of a serving process: the
// pool takes what is left, so a later cudaMalloc of even a few MiB fails), or a latency-critical loop that must
// not call cudaMalloc / cudaFree because both may synchronise the whole device.  Such a caller can run sa_linear
// (no scratch) but not sa_linear_ws, and at decode sizes sa_linear leaves most SMs without work.
//
// The scratch of this variant is part of the library image: a file-scope device array below.  The driver reserves it
// on every GPU on which this library's device code gets loaded and keeps it until the process ends; nothing in this
// file allocates or frees anything.  Its size covers every shape the split-K planner can produce on a GPU of up to
// 160 SMs (tiles x k slices never exceeds the SM count; one work unit writes a 128 x 256 fp32 partial = 128 KiB).
//
// `g_noalloc_scratch` names the array in DEVICE code only.  In host code the same identifier is a handle of the
// host-side shadow the runtime registers, not an address on the GPU: handing it to a kernel as a pointer is a fault
// (or, on systems where the GPU can reach host memory, a silent write to the wrong place).  Host code gets the real
// address from cudaGetSymbolAddress, per device, with that device current -- noalloc_scratch_ptr() below.
namespace sa {
namespace {

constexpr size_t kNoallocUnits = 160;
constexpr size_t kNoallocBytes = kNoallocUnits * kPartialFloats * sizeof(float) + 512;
static_assert(kNoallocBytes == SA_LINEAR_NOALLOC_SCRATCH_BYTES, "smoothagent.h states the size of the built-in scratch");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
void *g_noalloc_ptr[kNoallocMaxDevices] = {};  // device address of g_noalloc_scratch on device i; null = not looked up yet

// Device address of the scratch on the CURRENT device.  The first call on a device asks the runtime (which may load
// this library's device code onto that GPU: not something to do inside a stream capture); later calls read the table.
cudaError_t noalloc_scratch_ptr(void **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNoallocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

}  // namespace
}  // namespace sa

extern "C" int32_t sa_linear_noalloc(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N,
                                     int32_t K, void *stream) {
    if (M < 0 || N <= 0 || K <= 0) return SA_ERR_INVALID_ARG;
    if (K % sa::GBK != 0 || N % 8 != 0 || M > (int64_t(1) << 30)) return SA_ERR_UNSUPPORTED;
    if (M == 0) return SA_OK;
    if (sa::device_sms() <= 0) return SA_ERR_CUDA;
    // the same sizing sa_linear_workspace_bytes reports: 0 = the planner would not split this shape (it has enough
    // tiles to fill the GPU, or K is a single k-step): no scratch is involved and sa_linear is the call to make
    const size_t need = sa::gemm_plain_splitk_bytes(M, N, K);
    if (need == 0) return SA_ERR_UNSUPPORTED;
    if (need > sa::kNoallocBytes) return SA_ERR_WORKSPACE_TOO_SMALL;  // never silently unsplit: the bits would change
    void *scratch = nullptr;
    if (sa::noalloc_scratch_ptr(&scratch) != cudaSuccess) return SA_ERR_CUDA;
    // Nothing in the scratch has to start at zero: every partial word the reduction kernel reads (rows < M, all 256
    // columns of each k slice of each tile) is written by the GEMM kernel of this same call, in stream order before it.
    return sa::gemm_plain(x, w, residual, y, M, N, K, scratch, sa::kNoallocBytes, static_cast<cudaStream_t>(stream), nullptr);
}
