// dgrad_kernel.cuh -- the input-gradient GEMM of Algorithm 1 line 1: dX[T,in] = dY[T,out] . W[out,in]
// from the PRE-update weights ("the kernel issues that GEMM first and applies the optimizer afterwards";
// PAPER.md:296 Remark 2).  forge_layer_backward_grouped launches it for all projections of a layer ahead of the fused
// weight-gradient + AdamW launch on the same stream.
//
// GEMM view: M = T (tokens), N = in, K = out.  A = dY is K-major (out contiguous), B = W is MN-major (in contiguous),
// D = dX bf16 row-major, fp32 accumulation in tensor memory.  Same machinery as fused_kernel.cuh: persistent CTA
// pairs (tcgen05 cta_group::2, a pair owns a 256 x 256 tile of dX), warp 0 = TMA producer, warp 1 = single-thread MMA
// issuer, accumulators double-buffered in TMEM, warps 4-11 = epilogue (TMEM -> bf16 -> swizzled staging -> TMA store).
//
// Scheduling: at T = 512 a layer has only 304 pair-tiles of very different depth (K = out = 1024 .. 14336), so a
// linear tile order leaves a tail of more than one deep tile.  The host sorts the tiles by depth and assigns them
// longest-first to the least-loaded pair (LPT); the kernel walks its pair's slice of that list.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "adamw_math.cuh"   // pack_bf16
#include "ptx.cuh"

namespace forge {

constexpr int kDgMaxProblems = 8;
constexpr int kDgMaxTiles = 2048;   // tiles in the host-built LPT list; larger launches use the linear order
constexpr int kDgMaxPairs = 128;
constexpr int DG_BM = 128;          // rows of dX (tokens) per CTA = TMEM lanes; 256 per pair
constexpr int DG_BN = 256;          // columns of dX (in) per tile = TMEM columns
constexpr int DG_BK = 64;           // depth (out) per ring stage: one 128-byte swizzle span of A
constexpr int kDgThreads = 384;

struct alignas(64) DgradProblem {
    CUtensorMap map_dY;   // [T, out] bf16, box {64 (out), 128 (tokens)}, SWIZZLE_128B  -- A, K-major
    CUtensorMap map_W;    // [out, in] bf16, box {64 (in), 64 (out)}, SWIZZLE_128B      -- B, MN-major
    CUtensorMap map_dX;   // [T, in] bf16, box {64 (in), 32 (tokens)}, SWIZZLE_128B     -- D, stored from staging
    int32_t T, out, in;
    int32_t tiles_n;      // ceil(in / 256)
    int32_t tile_begin;   // first linear tile index of this problem
};

struct alignas(64) DgradParams {
    DgradProblem prob[kDgMaxProblems];
    int32_t num_problems, total_tiles;
    int32_t use_list;                      // 1: pair g walks order[pair_begin[g] .. pair_begin[g + 1])
    uint16_t pair_begin[kDgMaxPairs + 1];
    uint16_t order[kDgMaxTiles];
};

// K-major, 128B-swizzled operand: rows of 128 B (64 bf16 along K), 8-row core groups 1024 B apart (SBO); the leading
// byte offset is unused in this mode.  Advancing K by 16 elements moves the start address by 32 B inside the span.
__device__ __forceinline__ uint64_t make_smem_desc_k_sw128(uint32_t saddr) {
    uint64_t d = 0;
    d |= static_cast<uint64_t>((saddr & 0x3FFFFu) >> 4);
    d |= static_cast<uint64_t>(1) << 16;                 // LBO (ignored for swizzled K-major)
    d |= static_cast<uint64_t>(1024 >> 4) << 32;         // SBO
    d |= 1ull << 46;                                     // descriptor version for sm_100
    d |= 2ull << 61;                                     // SWIZZLE_128B
    return d;
}
// kind::f16 instruction descriptor: bf16 x bf16 -> fp32, A K-major, B MN-major
__host__ __device__ constexpr uint32_t make_idesc_bf16_f32_kmn(uint32_t M, uint32_t N) {
    return (1u << 4) | (1u << 7) | (1u << 10) | (0u << 15) | (1u << 16) | ((N >> 3) << 17) | ((M >> 4) << 24);
}

template <int kStages>
struct DgradCfg {
    static constexpr int A_STAGE = DG_BM * DG_BK * 2;               // 16 KB: this CTA's 128 token rows x 64 deep
    static constexpr int B_STAGE = DG_BK * (DG_BN / 2) * 2;         // 16 KB: this CTA's half of the 256 columns
    static constexpr int STAGE = A_STAGE + B_STAGE;
    static constexpr int OUT_BOX = 32 * 128;                        // 32 rows x 64 bf16 columns
    static constexpr int OUT_BYTES = 8 * 2 * OUT_BOX;               // two boxes per epilogue warp
    static constexpr int kNumBars = 2 * kStages + 4;
    static constexpr int SMEM_BYTES = 1024 + kStages * STAGE + OUT_BYTES + kNumBars * 8 + 16;
    static_assert(SMEM_BYTES <= 232448, "shared memory budget exceeded");
};

struct DgTile {
    int p, tm, tn;   // problem, 128-row token block of THIS CTA, 256-column block
};
__device__ __forceinline__ DgTile dg_decode(const DgradParams &P, int tile, uint32_t rank) {
    int p = 0;
#pragma unroll 1
    for (int i = 1; i < P.num_problems; ++i)
        if (tile >= P.prob[i].tile_begin) p = i;
    const int local = tile - P.prob[p].tile_begin;
    const int tn_count = P.prob[p].tiles_n;
    return DgTile{p, (local / tn_count) * 2 + static_cast<int>(rank), local % tn_count};
}

// iteration over this pair's tiles: either its slice of the LPT list or the strided linear order
struct DgWalk {
    int i, end, step;
    bool list;
    __device__ __forceinline__ DgWalk(const DgradParams &P, int pair, int npairs) {
        list = P.use_list != 0;
        if (list) { i = P.pair_begin[pair]; end = P.pair_begin[pair + 1]; step = 1; }
        else { i = pair; end = P.total_tiles; step = npairs; }
    }
    __device__ __forceinline__ bool valid() const { return i < end; }
    __device__ __forceinline__ int tile(const DgradParams &P) const { return list ? static_cast<int>(P.order[i]) : i; }
    __device__ __forceinline__ void next() { i += step; }
};

template <int kStages>
__global__ void __launch_bounds__(kDgThreads, 1)
forge_dgrad_kernel(const __grid_constant__ DgradParams P) {
    using Cfg = DgradCfg<kStages>;
    const uint32_t rank = cluster_ctarank();
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sML = smem_base;
    const uint32_t sOUT = sML + kStages * Cfg::STAGE;
    const uint32_t sBAR = sOUT + Cfg::OUT_BYTES;
    const uint32_t bar_full = sBAR;
    const uint32_t bar_empty = bar_full + 8 * kStages;
    const uint32_t bar_tm_full = bar_empty + 8 * kStages;   // [2]
    const uint32_t bar_tm_empty = bar_tm_full + 16;         // [2]
    const uint32_t s_tmem_ptr = bar_tm_empty + 16;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        for (int i = 0; i < kStages; ++i) {
            mbar_init(bar_full + 8 * i, 1);
            mbar_init(bar_empty + 8 * i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar_tm_full + 8 * i, 1);
            mbar_init(bar_tm_empty + 8 * i, 8 * 2);          // one arrival per epilogue warp of the pair
        }
        mbar_fence_init();
    }
    if (warp == 2) tmem_alloc_cg2(s_tmem_ptr, 512);
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];\n" : "=r"(tmem_base) : "r"(s_tmem_ptr));

    const int pair = blockIdx.x / 2, npairs = gridDim.x / 2;

    if (warp == 0) {
        // ================= operand producer: dY (A) and W (B) depth chunks ========================
        if (lane == 0) {
            uint32_t it = 0;
            for (DgWalk w(P, pair, npairs); w.valid(); w.next()) {
                const DgTile tc = dg_decode(P, w.tile(P), rank);
                const DgradProblem &pd = P.prob[tc.p];
                const int num_kb = (pd.out + DG_BK - 1) / DG_BK;
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const uint32_t s = it % kStages, ph = (it / kStages) & 1u;
                    mbar_wait(bar_empty + 8 * s, ph ^ 1u);
                    const uint32_t a = sML + s * Cfg::STAGE, b = a + Cfg::A_STAGE;
                    if (rank == 0) mbar_expect_tx(bar_full + 8 * s, 2 * Cfg::STAGE);   // both CTAs' bytes on the leader
                    const uint32_t full = mapa_shared(bar_full + 8 * s, 0);
                    tma_load_2d_cg2(a, &pd.map_dY, full, kb * DG_BK, tc.tm * DG_BM, kEvictLast);
#pragma unroll
                    for (int i = 0; i < DG_BN / 128; ++i)      // this CTA's half of the 256 columns, 64 at a time
                        tma_load_2d_cg2(b + i * DG_BK * 128, &pd.map_W, full,
                                        tc.tn * DG_BN + static_cast<int>(rank) * (DG_BN / 2) + i * 64, kb * DG_BK, kEvictLast);
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (leader CTA) =================================================
        if (lane == 0 && rank == 0) {
            constexpr uint32_t idesc = make_idesc_bf16_f32_kmn(DG_BM * 2, DG_BN);
            uint32_t it = 0, titer = 0;
            for (DgWalk w(P, pair, npairs); w.valid(); w.next(), ++titer) {
                const DgTile tc = dg_decode(P, w.tile(P), rank);
                const int num_kb = (P.prob[tc.p].out + DG_BK - 1) / DG_BK;
                const uint32_t as = titer & 1u, aph = (titer >> 1) & 1u;
                mbar_wait(bar_tm_empty + 8 * as, aph ^ 1u);
                tc_fence_after();
                const uint32_t tmem_d = tmem_base + as * DG_BN;
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const uint32_t s = it % kStages, ph = (it / kStages) & 1u;
                    mbar_wait(bar_full + 8 * s, ph);
                    tc_fence_after();
                    const uint32_t a = sML + s * Cfg::STAGE, b = a + Cfg::A_STAGE;
#pragma unroll
                    for (int k = 0; k < DG_BK / 16; ++k) {
                        const uint64_t ad = make_smem_desc_k_sw128(a + k * 32);                       // 16 deep = 32 B along the span
                        const uint64_t bd = make_smem_desc_mn_sw128(b + k * 2048, DG_BK * 128, 1024);  // 16 deep = 16 rows of 128 B
                        umma_bf16_cg2(tmem_d, ad, bd, idesc, (kb | k) != 0 ? 1u : 0u);
                    }
                    umma_commit_cg2(bar_empty + 8 * s, 3);
                }
                umma_commit_cg2(bar_tm_full + 8 * as, 3);
            }
        }
    } else if (warp >= 4) {
        // ================= epilogue: TMEM -> bf16 -> staging -> TMA store ============================
        const int wg = (warp - 4) >> 2;                 // warpgroup: columns [128 wg, 128 wg + 128)
        const uint32_t quad = warp & 3;                 // TMEM lane quadrant = token rows 32 quad ..
        const uint32_t stage0 = sOUT + static_cast<uint32_t>(warp - 4) * 2 * Cfg::OUT_BOX;
        uint32_t titer = 0, nstore = 0;
        for (DgWalk w(P, pair, npairs); w.valid(); w.next(), ++titer) {
            const DgTile tc = dg_decode(P, w.tile(P), rank);
            const DgradProblem &pd = P.prob[tc.p];
            const uint32_t as = titer & 1u, aph = (titer >> 1) & 1u;
            mbar_wait(bar_tm_full + 8 * as, aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((quad * 32u) << 16) + as * DG_BN + wg * (DG_BN / 2);
#pragma unroll 1
            for (int box = 0; box < 2; ++box, ++nstore) {
                const uint32_t buf = stage0 + (nstore & 1u) * Cfg::OUT_BOX;
                // the store issued two boxes ago from this buffer has been read
                if (lane == 0) tma_store_wait_read<1>();
                __syncwarp();
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    uint32_t g[32];
                    tmem_ld_32x32b_x32(taddr + box * 64 + h * 32, g);
                    tmem_ld_wait();
#pragma unroll
                    for (int j = 0; j < 4; ++j) {       // 8 columns = one 16-byte piece
                        uint4 q;
                        q.x = pack_bf16(__uint_as_float(g[8 * j + 0]), __uint_as_float(g[8 * j + 1]));
                        q.y = pack_bf16(__uint_as_float(g[8 * j + 2]), __uint_as_float(g[8 * j + 3]));
                        q.z = pack_bf16(__uint_as_float(g[8 * j + 4]), __uint_as_float(g[8 * j + 5]));
                        q.w = pack_bf16(__uint_as_float(g[8 * j + 6]), __uint_as_float(g[8 * j + 7]));
                        const uint32_t piece = static_cast<uint32_t>(h * 4 + j);
                        sts128(buf + lane * 128u + ((piece ^ (lane & 7u)) << 4), q);
                    }
                }
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) {
                    tma_store_2d(&pd.map_dX, buf, tc.tn * DG_BN + wg * (DG_BN / 2) + box * 64,
                                 tc.tm * DG_BM + static_cast<int>(quad) * 32, kEvictNormal);
                    tma_store_commit();
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(mapa_shared(bar_tm_empty + 8 * as, 0));
        }
        if (lane == 0) tma_store_wait_all<0>();
    }

    __syncwarp();
    tc_fence_before();
    cluster_sync_all();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc_cg2(tmem_base, 512);
    }
}

}  // namespace forge
