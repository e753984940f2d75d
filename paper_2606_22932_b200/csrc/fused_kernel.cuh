// fused_kernel.cuh -- the persistent, warp-specialised sm_100a kernel of forge-b200.
//
// Per weight tile (128 rows of `out` x 256 columns of `in`), Algorithm 1:
//   lines 2-5  G_ij = sum_k dY_k,i^T X_k,j      tcgen05.mma, bf16 x bf16 -> fp32 in tensor memory
//   line  6    load W_ij, m_ij, v_ij            TMA, 128 x 32-column chunks into a smem ring
//   lines 7-10 AdamW in fp32 registers          adamw_math.cuh
//   line  11   store W_ij, m_ij, v_ij           in place in the smem chunk, then TMA store
// G never leaves the SM.  One CTA owns a tile for the whole token loop, so a
// partial-K update can never be applied.
//
// Warp roles (384 threads, one CTA per SM, persistent over a static tile list):
//   warp 0      operand producer: TMA loads of dY / X token chunks into the mainloop ring
//   warp 1      MMA issuer: one thread issues tcgen05.mma; accumulators double-buffered in TMEM
//   warp 2      TMEM allocator + state loader: TMA loads of W/m/v chunks (independent of G, so
//               they run ahead of the mainloop and across tile boundaries)
//   warp 3      state storer: TMA stores of finished chunks, recycles ring slots
//   warps 4-11  two epilogue warpgroups; warp w reads TMEM lanes 32*(w%4).., one W row per thread,
//               warpgroup g takes chunks g, g+2, ...
//
// Both GEMM operands are MN-major: A = dY^T has `out` contiguous, B = X has `in` contiguous, and
// the token axis (K) is the slow axis of both.  A token chunk is staged as 64-element (128 B)
// swizzled rows: smem[mn_block][k][64], which is the canonical MN-major SWIZZLE_128B UMMA layout
// with LBO = kBlockK*128 B between 64-wide MN blocks and SBO = 1024 B between 8-token groups.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "adamw_math.cuh"
#include "ptx.cuh"

namespace forge {

constexpr int kMaxProblems = 8;
constexpr int BLOCK_M = 128;   // tile rows  (out)  = TMEM lanes
constexpr int BLOCK_N = 256;   // tile cols  (in)   = TMEM columns = one int8 block per row
constexpr int CHUNK_N = 32;    // state chunk columns
constexpr int CHUNKS = BLOCK_N / CHUNK_N;
constexpr int kCtrlWarps = 4;
constexpr int kEpiWarps = 8;
constexpr int kThreads = (kCtrlWarps + kEpiWarps) * 32;
constexpr int kTmemCols = 512;  // 2 accumulator buffers x 256 fp32 columns

enum : int { MDT_FP32 = 0, MDT_BF16 = 1, MDT_INT8 = 2 };
enum : int { MODE_ADAMW = 0, MODE_STORE_G = 1 };

struct alignas(64) ProblemDesc {
    CUtensorMap map_dY;  // [T, out] bf16, box {64, kBlockK}, SWIZZLE_128B
    CUtensorMap map_X;   // [T, in]  bf16, box {64, kBlockK}, SWIZZLE_128B
    CUtensorMap map_W;   // [out, in] bf16, box {32, 128}, SWIZZLE_64B
    CUtensorMap map_m;   // [out, in] moment dtype, box {32, 128}, swizzle = row bytes
    CUtensorMap map_v;   //   (MODE_STORE_G: map_m is the fp32 G output)
    float *m_scale;      // INT8 only: [out, in/256]
    float *v_scale;
    int32_t T, out, in;
    int32_t tiles_n;     // ceil(in / 256)
    int32_t tile_begin;  // first linear tile index of this problem
    int32_t pad_;
};

struct alignas(64) KernelParams {
    ProblemDesc prob[kMaxProblems];
    AdamWScalars hp;
    int32_t num_problems;
    int32_t total_tiles;
    int32_t pf_chunks;   // state chunks prefetched into L2 ahead of the shared-memory ring
    int32_t debug;       // ablation switches for profiling ONLY (results are wrong when set):
                         // 1 = no operand loads / MMA, 2 = no state loads / stores, 4 = no epilogue math
};
enum : int { DBG_NO_MAINLOOP = 1, DBG_NO_STATE = 2, DBG_NO_EPILOGUE = 4 };

// CG = 1: one CTA per 128x256 tile.  CG = 2: a CTA pair (cluster of 2, tcgen05 cta_group::2) shares
// a 256x256 tile: each CTA stages its own 128 rows of A = dY^T and only HALF of B = X (128 of the
// 256 columns), the pair's leader issues one M=256 MMA that reads both CTAs' shared memory, and
// each CTA's TMEM receives its own 128 x 256 accumulator.  Operand bytes per CTA fall by a third
// (L2 -> SM traffic and smem per stage), the state path stays CTA-local.
template <int MDT, int kBlockK, int kStages, int kStateStages, int CG = 1>
struct KernelCfg {
    static constexpr int kMomBytes = (MDT == MDT_FP32) ? 4 : (MDT == MDT_BF16 ? 2 : 1);
    static constexpr int A_STAGE = kBlockK * 128 * (BLOCK_M / 64);
    static constexpr int B_STAGE = kBlockK * 128 * (BLOCK_N / 64) / CG;
    static constexpr int ML_STAGE = A_STAGE + B_STAGE;
    static constexpr int W_ROW = CHUNK_N * 2;
    static constexpr int M_ROW = CHUNK_N * kMomBytes;
    static constexpr int W_CHUNK = BLOCK_M * W_ROW;
    static constexpr int M_CHUNK = (BLOCK_M * M_ROW + 1023) / 1024 * 1024;
    static constexpr int ST_STAGE = W_CHUNK + 2 * M_CHUNK;
    static constexpr int ST_TX_BYTES = BLOCK_M * (W_ROW + 2 * M_ROW);
    static constexpr int kNumBars = 2 * kStages + 4 + 3 * kStateStages;
    static constexpr int XCHG_BYTES = (MDT == MDT_INT8) ? 4096 : 0;   // absmax exchange, 2 buffers
    static constexpr int SMEM_BYTES = 1024 /*align slack*/ + kStages * ML_STAGE +
                                      kStateStages * ST_STAGE + kNumBars * 8 + 16 + XCHG_BYTES;
    static_assert(SMEM_BYTES <= 232448, "shared memory budget exceeded");
    static_assert(kBlockK % 16 == 0 && kBlockK >= 16, "kBlockK must be a multiple of UMMA_K");
    static_assert(CG == 1 || CG == 2, "CTA group is 1 or 2");
    static_assert(MDT != MDT_INT8 || kStateStages >= CHUNKS + 1, "int8 needs a whole tile resident");
    // Chunk ci lives in ring slot ci % kStateStages and is consumed by epilogue warpgroup ci % 2.
    // With an even ring every slot always belongs to the same warpgroup, so a warpgroup observes
    // every phase of the slot barriers it waits on; with an odd ring it would skip the other
    // warpgroup's phases and an mbarrier parity wait could alias to a phase two steps back.
    static_assert(kStateStages % 2 == 0, "state ring must be even (one consumer warpgroup per slot)");
};

struct TileCoord {
    int p, tm, tn;   // problem, 128-row block of THIS CTA, 256-column block
};
// `tile` indexes (128*CG) x 256 work units; rank is this CTA's rank in its pair (0 when CG = 1)
template <int CG>
__device__ __forceinline__ TileCoord decode_tile(const KernelParams &P, int tile, uint32_t rank) {
    int p = 0;
#pragma unroll 1
    for (int i = 1; i < P.num_problems; ++i)
        if (tile >= P.prob[i].tile_begin) p = i;
    const int local = tile - P.prob[p].tile_begin;
    const int tn_count = P.prob[p].tiles_n;
    return TileCoord{p, (local / tn_count) * CG + static_cast<int>(rank), local % tn_count};
}

// byte offset of 16-byte chunk j of row r in a TMA-swizzled box whose rows are ROW bytes long
template <int ROW>
__device__ __forceinline__ uint32_t swz(uint32_t r, uint32_t j) {
    if constexpr (ROW == 128) return r * 128u + ((j ^ (r & 7u)) << 4);
    else if constexpr (ROW == 64) return r * 64u + ((j ^ ((r >> 1) & 3u)) << 4);
    else return r * 32u + ((j ^ ((r >> 2) & 1u)) << 4);
}

// ---------------------------------------------------------------------------------------------
// epilogue bodies: one thread = one W row of the tile, 32 columns of chunk `c` at a time
// ---------------------------------------------------------------------------------------------
template <int MDT>
__device__ __forceinline__ void epi_chunk_fp(const AdamWScalars &hp, const uint32_t (&g)[32],
                                             uint32_t sW, uint32_t sM, uint32_t sV, uint32_t row) {
    // 4 groups of 8 columns: one 16 B piece of W (8 bf16) + matching moments
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t aw = sW + swz<64>(row, j);
        uint4 wq = lds128(aw);
        float w[8] = {bf16lo(wq.x), bf16hi(wq.x), bf16lo(wq.y), bf16hi(wq.y),
                      bf16lo(wq.z), bf16hi(wq.z), bf16lo(wq.w), bf16hi(wq.w)};
        float m[8], v[8];
        if constexpr (MDT == MDT_FP32) {
            const uint32_t am0 = sM + swz<128>(row, 2 * j), am1 = sM + swz<128>(row, 2 * j + 1);
            const uint32_t av0 = sV + swz<128>(row, 2 * j), av1 = sV + swz<128>(row, 2 * j + 1);
            uint4 a = lds128(am0), b = lds128(am1), c = lds128(av0), d = lds128(av1);
            m[0] = __uint_as_float(a.x); m[1] = __uint_as_float(a.y); m[2] = __uint_as_float(a.z); m[3] = __uint_as_float(a.w);
            m[4] = __uint_as_float(b.x); m[5] = __uint_as_float(b.y); m[6] = __uint_as_float(b.z); m[7] = __uint_as_float(b.w);
            v[0] = __uint_as_float(c.x); v[1] = __uint_as_float(c.y); v[2] = __uint_as_float(c.z); v[3] = __uint_as_float(c.w);
            v[4] = __uint_as_float(d.x); v[5] = __uint_as_float(d.y); v[6] = __uint_as_float(d.z); v[7] = __uint_as_float(d.w);
#pragma unroll
            for (int e = 0; e < 8; ++e) adamw_update(hp, __uint_as_float(g[8 * j + e]), w[e], m[e], v[e]);
            sts128(am0, make_uint4(__float_as_uint(m[0]), __float_as_uint(m[1]), __float_as_uint(m[2]), __float_as_uint(m[3])));
            sts128(am1, make_uint4(__float_as_uint(m[4]), __float_as_uint(m[5]), __float_as_uint(m[6]), __float_as_uint(m[7])));
            sts128(av0, make_uint4(__float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]), __float_as_uint(v[3])));
            sts128(av1, make_uint4(__float_as_uint(v[4]), __float_as_uint(v[5]), __float_as_uint(v[6]), __float_as_uint(v[7])));
        } else {
            const uint32_t am = sM + swz<64>(row, j), av = sV + swz<64>(row, j);
            uint4 a = lds128(am), c = lds128(av);
            m[0] = bf16lo(a.x); m[1] = bf16hi(a.x); m[2] = bf16lo(a.y); m[3] = bf16hi(a.y);
            m[4] = bf16lo(a.z); m[5] = bf16hi(a.z); m[6] = bf16lo(a.w); m[7] = bf16hi(a.w);
            v[0] = bf16lo(c.x); v[1] = bf16hi(c.x); v[2] = bf16lo(c.y); v[3] = bf16hi(c.y);
            v[4] = bf16lo(c.z); v[5] = bf16hi(c.z); v[6] = bf16lo(c.w); v[7] = bf16hi(c.w);
#pragma unroll
            for (int e = 0; e < 8; ++e) adamw_update(hp, __uint_as_float(g[8 * j + e]), w[e], m[e], v[e]);
            sts128(am, make_uint4(pack_bf16(m[0], m[1]), pack_bf16(m[2], m[3]), pack_bf16(m[4], m[5]), pack_bf16(m[6], m[7])));
            sts128(av, make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7])));
        }
        sts128(aw, make_uint4(pack_bf16(w[0], w[1]), pack_bf16(w[2], w[3]), pack_bf16(w[4], w[5]), pack_bf16(w[6], w[7])));
    }
}

// store-G twin: the fp32 tile chunk goes to the smem chunk buffer unchanged
__device__ __forceinline__ void epi_chunk_store_g(const uint32_t (&g)[32], uint32_t sG, uint32_t row) {
#pragma unroll
    for (int j = 0; j < 8; ++j)
        sts128(sG + swz<128>(row, j), make_uint4(g[4 * j], g[4 * j + 1], g[4 * j + 2], g[4 * j + 3]));
}


// int8 blockwise moments (App. B; 256-element blocks along `in` == one block per tile
// row).  The new block absmax is only known once all 256 m', v' of the row exist, so the tile is
// walked twice over the TMEM accumulator and the smem-resident codes: pass 1 finds max|m'|, max v',
// pass 2 recomputes the identical m', v' (same instructions, same operands), forms W', and emits
// the codes.  A row is owned by one thread of each warpgroup (even / odd chunks); the two partial
// maxima are combined through shared memory.
__device__ __forceinline__ void unpack_codes(const uint4 &q, int (&c)[16], bool is_signed) {
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const uint32_t b = (w[i >> 2] >> (8 * (i & 3))) & 0xFFu;
        c[i] = is_signed ? static_cast<int>(static_cast<int8_t>(b)) : static_cast<int>(b);
    }
}
__device__ __forceinline__ uint4 pack_codes(const int (&c)[16]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
        w[i] = (static_cast<uint32_t>(c[4 * i]) & 0xFFu) | ((static_cast<uint32_t>(c[4 * i + 1]) & 0xFFu) << 8) |
               ((static_cast<uint32_t>(c[4 * i + 2]) & 0xFFu) << 16) | ((static_cast<uint32_t>(c[4 * i + 3]) & 0xFFu) << 24);
    return make_uint4(w[0], w[1], w[2], w[3]);
}

template <class Cfg, int kStateStages, int CG>
__device__ __forceinline__ void epi_tile_int8(const KernelParams &P, const AdamWScalars &hp, int tile, uint32_t rank,
                                              uint32_t titer, uint32_t taddr, uint32_t sST,
                                              uint32_t bar_st_full, uint32_t bar_st_done, uint32_t row,
                                              int wg, uint32_t s_xchg) {
    const TileCoord tc = decode_tile<CG>(P, tile, rank);
    const ProblemDesc &pd = P.prob[tc.p];
    const int row_g = tc.tm * BLOCK_M + static_cast<int>(row);
    const bool valid = row_g < pd.out;
    const size_t sidx = static_cast<size_t>(valid ? row_g : 0) * static_cast<size_t>(pd.in / BLOCK_N) + tc.tn;
    const float a_m_old = valid ? pd.m_scale[sidx] : 0.0f;
    const float a_v_old = valid ? pd.v_scale[sidx] : 0.0f;
    const float dm = dequant_step(a_m_old, 127.0f), dv = dequant_step(a_v_old, 255.0f);

    // ---- pass 1: block absmax of m', v'
    float pm = 0.0f, pv = 0.0f;
    for (int c = wg; c < CHUNKS; c += 2) {
        const uint32_t ci = titer * CHUNKS + c;
        const uint32_t s = ci % kStateStages, ph = (ci / kStateStages) & 1u;
        uint32_t g[32];
        tmem_ld_32x32b_x32(taddr + c * CHUNK_N, g);
        const uint32_t sM = sST + s * Cfg::ST_STAGE + Cfg::W_CHUNK, sV = sM + Cfg::M_CHUNK;
        mbar_wait(bar_st_full + 8 * s, ph);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            int mc[16], vc[16];
            unpack_codes(lds128(sM + swz<32>(row, j)), mc, true);
            unpack_codes(lds128(sV + swz<32>(row, j)), vc, false);
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                float w = 0.0f, m = __fmul_rn(static_cast<float>(mc[e]), dm), v = __fmul_rn(static_cast<float>(vc[e]), dv);
                adamw_update(hp, __uint_as_float(g[16 * j + e]), w, m, v);
                pm = fmaxf(pm, fabsf(m));
                pv = fmaxf(pv, fabsf(v));
            }
        }
    }
    // ---- combine the two half-rows
    const uint32_t xb = s_xchg + (titer & 1u) * 2048u;
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};\n" ::"r"(xb + (wg * 128u + row) * 8u), "f"(pm), "f"(pv) : "memory");
    asm volatile("bar.sync 1, 256;\n" ::: "memory");
    float om, ov;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(om), "=f"(ov) : "r"(xb + ((wg ^ 1) * 128u + row) * 8u));
    const float a_m = fmaxf(pm, om), a_v = fmaxf(pv, ov);
    const float inv_m = quant_inv_scale(a_m, 127.0f), inv_v = quant_inv_scale(a_v, 255.0f);

    // ---- pass 2: recompute, update W, requantise
    for (int c = wg; c < CHUNKS; c += 2) {
        const uint32_t ci = titer * CHUNKS + c;
        const uint32_t s = ci % kStateStages;
        uint32_t g[32];
        tmem_ld_32x32b_x32(taddr + c * CHUNK_N, g);
        const uint32_t sW = sST + s * Cfg::ST_STAGE, sM = sW + Cfg::W_CHUNK, sV = sM + Cfg::M_CHUNK;
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            int mc[16], vc[16];
            const uint32_t am = sM + swz<32>(row, j), av = sV + swz<32>(row, j);
            unpack_codes(lds128(am), mc, true);
            unpack_codes(lds128(av), vc, false);
            const uint32_t aw0 = sW + swz<64>(row, 2 * j), aw1 = sW + swz<64>(row, 2 * j + 1);
            const uint4 w0 = lds128(aw0), w1 = lds128(aw1);
            float w[16] = {bf16lo(w0.x), bf16hi(w0.x), bf16lo(w0.y), bf16hi(w0.y), bf16lo(w0.z), bf16hi(w0.z),
                           bf16lo(w0.w), bf16hi(w0.w), bf16lo(w1.x), bf16hi(w1.x), bf16lo(w1.y), bf16hi(w1.y),
                           bf16lo(w1.z), bf16hi(w1.z), bf16lo(w1.w), bf16hi(w1.w)};
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                float m = __fmul_rn(static_cast<float>(mc[e]), dm), v = __fmul_rn(static_cast<float>(vc[e]), dv);
                adamw_update(hp, __uint_as_float(g[16 * j + e]), w[e], m, v);
                mc[e] = quant_m_code(m, inv_m);
                vc[e] = quant_v_code(v, inv_v);
            }
            sts128(am, pack_codes(mc));
            sts128(av, pack_codes(vc));
            sts128(aw0, make_uint4(pack_bf16(w[0], w[1]), pack_bf16(w[2], w[3]), pack_bf16(w[4], w[5]), pack_bf16(w[6], w[7])));
            sts128(aw1, make_uint4(pack_bf16(w[8], w[9]), pack_bf16(w[10], w[11]), pack_bf16(w[12], w[13]), pack_bf16(w[14], w[15])));
        }
        fence_proxy_async_smem();
        mbar_arrive(bar_st_done + 8 * s);
    }
    if (wg == 0 && valid) {
        pd.m_scale[sidx] = a_m;
        pd.v_scale[sidx] = a_v;
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <int MDT, int MODE, int kBlockK, int kStages, int kStateStages, int CG>
__global__ void __launch_bounds__(kThreads, 1)
forge_fused_kernel(const __grid_constant__ KernelParams P) {
    using Cfg = KernelCfg<MDT, kBlockK, kStages, kStateStages, CG>;
    const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;   // rank 0 = the pair's leader
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sML = smem_base;                                   // mainloop ring
    const uint32_t sST = sML + kStages * Cfg::ML_STAGE;               // state ring
    const uint32_t sBAR = sST + kStateStages * Cfg::ST_STAGE;         // mbarriers
    // barrier map
    const uint32_t bar_ml_full = sBAR;
    const uint32_t bar_ml_empty = bar_ml_full + 8 * kStages;
    const uint32_t bar_tm_full = bar_ml_empty + 8 * kStages;          // [2]
    const uint32_t bar_tm_empty = bar_tm_full + 16;                   // [2]
    const uint32_t bar_st_full = bar_tm_empty + 16;
    const uint32_t bar_st_done = bar_st_full + 8 * kStateStages;
    const uint32_t bar_st_empty = bar_st_done + 8 * kStateStages;
    const uint32_t s_tmem_ptr = bar_st_empty + 8 * kStateStages;
    const uint32_t s_xchg = s_tmem_ptr + 16;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        for (int i = 0; i < kStages; ++i) {
            mbar_init(bar_ml_full + 8 * i, 1);
            mbar_init(bar_ml_empty + 8 * i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar_tm_full + 8 * i, 1);
            mbar_init(bar_tm_empty + 8 * i, kEpiWarps * CG);   // one arrival per epilogue warp of the pair
        }
        for (int i = 0; i < kStateStages; ++i) {
            mbar_init(bar_st_full + 8 * i, 1);
            mbar_init(bar_st_done + 8 * i, 128);
            mbar_init(bar_st_empty + 8 * i, 1);
        }
        mbar_fence_init();
    }
    if (warp == 2) {
        if constexpr (CG == 2) tmem_alloc_cg2(s_tmem_ptr, kTmemCols);
        else tmem_alloc(s_tmem_ptr, kTmemCols);
    }
    tc_fence_before();
    if constexpr (CG == 2) cluster_sync_all();   // the peer's barriers exist before any remote signal
    else __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];\n" : "=r"(tmem_base) : "r"(s_tmem_ptr));

    const int first_tile = blockIdx.x / CG, tile_step = gridDim.x / CG;

    if (warp == 0) {
        // ================= operand producer (Alg. 1 lines 3-5: stream dY_k,i and X_k,j) ==========
        if (lane == 0 && !(P.debug & DBG_NO_MAINLOOP)) {
            uint32_t it = 0;  // running k-block counter over all tiles of this CTA
            for (int tile = first_tile; tile < P.total_tiles; tile += tile_step) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const ProblemDesc &pd = P.prob[tc.p];
                const int num_kb = (pd.T + kBlockK - 1) / kBlockK;
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const uint32_t s = it % kStages, ph = (it / kStages) & 1u;
                    mbar_wait(bar_ml_empty + 8 * s, ph ^ 1u);
                    const uint32_t a = sML + s * Cfg::ML_STAGE, b = a + Cfg::A_STAGE;
                    if constexpr (CG == 1) {
                        const uint32_t full = bar_ml_full + 8 * s;
                        mbar_expect_tx(full, Cfg::ML_STAGE);
#pragma unroll
                        for (int i = 0; i < BLOCK_M / 64; ++i)
                            tma_load_2d(a + i * kBlockK * 128, &pd.map_dY, full, tc.tm * BLOCK_M + i * 64,
                                        kb * kBlockK, kEvictLast);
#pragma unroll
                        for (int i = 0; i < BLOCK_N / 64; ++i)
                            tma_load_2d(b + i * kBlockK * 128, &pd.map_X, full, tc.tn * BLOCK_N + i * 64,
                                        kb * kBlockK, kEvictLast);
                    } else {
                        // both CTAs' bytes are counted on the LEADER's full barrier
                        if (rank == 0) mbar_expect_tx(bar_ml_full + 8 * s, 2 * Cfg::ML_STAGE);
                        const uint32_t full = mapa_shared(bar_ml_full + 8 * s, 0);
#pragma unroll
                        for (int i = 0; i < BLOCK_M / 64; ++i)
                            tma_load_2d_cg2(a + i * kBlockK * 128, &pd.map_dY, full, tc.tm * BLOCK_M + i * 64,
                                            kb * kBlockK, kEvictLast);
#pragma unroll
                        for (int i = 0; i < BLOCK_N / 128; ++i)   // this CTA's half of the 256 columns
                            tma_load_2d_cg2(b + i * kBlockK * 128, &pd.map_X, full,
                                            tc.tn * BLOCK_N + static_cast<int>(rank) * (BLOCK_N / 2) + i * 64,
                                            kb * kBlockK, kEvictLast);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (Alg. 1 line 4: G_ij += dY_k,i^T X_k,j) =====================
        if (lane == 0 && rank == 0 && !(P.debug & DBG_NO_MAINLOOP)) {
            constexpr uint32_t idesc = make_idesc_bf16_f32_mnmn(BLOCK_M * CG, BLOCK_N);
            uint32_t it = 0, titer = 0;
            for (int tile = first_tile; tile < P.total_tiles; tile += tile_step, ++titer) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const int num_kb = (P.prob[tc.p].T + kBlockK - 1) / kBlockK;
                const uint32_t as = titer & 1u, aph = (titer >> 1) & 1u;
                mbar_wait(bar_tm_empty + 8 * as, aph ^ 1u);   // epilogue has drained this buffer
                tc_fence_after();
                const uint32_t tmem_d = tmem_base + as * BLOCK_N;
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const uint32_t s = it % kStages, ph = (it / kStages) & 1u;
                    mbar_wait(bar_ml_full + 8 * s, ph);
                    tc_fence_after();
                    const uint32_t a = sML + s * Cfg::ML_STAGE, b = a + Cfg::A_STAGE;
#pragma unroll
                    for (int k = 0; k < kBlockK / 16; ++k) {
                        // 16 tokens further = 16 rows of 128 B inside every 64-wide MN block
                        const uint64_t ad = make_smem_desc_mn_sw128(a + k * 2048, kBlockK * 128, 1024);
                        const uint64_t bd = make_smem_desc_mn_sw128(b + k * 2048, kBlockK * 128, 1024);
                        if constexpr (CG == 2) umma_bf16_cg2(tmem_d, ad, bd, idesc, (kb | k) != 0 ? 1u : 0u);
                        else umma_bf16(tmem_d, ad, bd, idesc, (kb | k) != 0 ? 1u : 0u);
                    }
                    // smem slot free (in both CTAs of a pair) once these MMAs retire
                    if constexpr (CG == 2) umma_commit_cg2(bar_ml_empty + 8 * s, 3);
                    else umma_commit(bar_ml_empty + 8 * s);
                }
                // G_ij complete (all of T, exactly once) -- signalled to each CTA's epilogue
                if constexpr (CG == 2) umma_commit_cg2(bar_tm_full + 8 * as, 3);
                else umma_commit(bar_tm_full + 8 * as);
            }
        }
    } else if (warp == 2) {
        // ================= state loader (Alg. 1 line 6: load W_ij, m_ij, v_ij) ===================
        if (MODE == MODE_ADAMW && lane == 0 && !(P.debug & DBG_NO_STATE)) {
            // The ring holds only kStateStages chunks, and a slot stays busy through load latency,
            // epilogue and store read; an L2 prefetch cursor runs pf_chunks further ahead so that
            // the DRAM requests in flight are not bounded by shared memory (126 MB of L2 absorb it).
            int pf_tile = first_tile, pf_c = 0;
            TileCoord pf_tc = decode_tile<CG>(P, pf_tile < P.total_tiles ? pf_tile : first_tile, rank);
            auto prefetch_next = [&]() {
                if (pf_tile >= P.total_tiles) return;
                const ProblemDesc &pd = P.prob[pf_tc.p];
                const int x = pf_tc.tn * BLOCK_N + pf_c * CHUNK_N, y = pf_tc.tm * BLOCK_M;
                tma_prefetch_l2_2d(&pd.map_W, x, y);
                tma_prefetch_l2_2d(&pd.map_m, x, y);
                tma_prefetch_l2_2d(&pd.map_v, x, y);
                if (++pf_c == CHUNKS) {
                    pf_c = 0;
                    pf_tile += tile_step;
                    if (pf_tile < P.total_tiles) pf_tc = decode_tile<CG>(P, pf_tile, rank);
                }
            };
            for (int i = 0; i < P.pf_chunks + kStateStages; ++i) {
                if (i >= kStateStages) prefetch_next();
                else if (P.pf_chunks > 0) {   // the first ring fill is loaded directly: skip, do not prefetch
                    if (++pf_c == CHUNKS) {
                        pf_c = 0;
                        pf_tile += tile_step;
                        if (pf_tile < P.total_tiles) pf_tc = decode_tile<CG>(P, pf_tile, rank);
                    }
                }
            }
            uint32_t ci = 0;  // running chunk counter
            for (int tile = first_tile; tile < P.total_tiles; tile += tile_step) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const ProblemDesc &pd = P.prob[tc.p];
                for (int c = 0; c < CHUNKS; ++c, ++ci) {
                    if (P.pf_chunks > 0) prefetch_next();
                    const uint32_t s = ci % kStateStages, ph = (ci / kStateStages) & 1u;
                    mbar_wait(bar_st_empty + 8 * s, ph ^ 1u);
                    const uint32_t full = bar_st_full + 8 * s;
                    mbar_expect_tx(full, Cfg::ST_TX_BYTES);
                    const uint32_t base = sST + s * Cfg::ST_STAGE;
                    const int x = tc.tn * BLOCK_N + c * CHUNK_N, y = tc.tm * BLOCK_M;
                    tma_load_2d(base, &pd.map_W, full, x, y, kEvictFirst);
                    tma_load_2d(base + Cfg::W_CHUNK, &pd.map_m, full, x, y, kEvictFirst);
                    tma_load_2d(base + Cfg::W_CHUNK + Cfg::M_CHUNK, &pd.map_v, full, x, y, kEvictFirst);
                }
            }
        }
    } else if (warp == 3) {
        // ================= state storer (Alg. 1 line 11: store W_ij, m_ij, v_ij) ================
        if (lane == 0) {
            // One store group may stay in flight while the next chunk is stored (look-ahead 1): the
            // ~0.8 us a TMA store needs before its shared-memory source is reusable is then hidden
            // behind the next chunk instead of serialising the ring.  A slot is released as soon as
            // its own group has been read; if no further chunk is ready the storer drains at once.
            uint32_t ci = 0;
            int held = -1;                                 // slot whose store group is still unreleased
            for (int tile = first_tile; tile < P.total_tiles; tile += tile_step) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const ProblemDesc &pd = P.prob[tc.p];
                for (int c = 0; c < CHUNKS; ++c, ++ci) {
                    const uint32_t s = ci % kStateStages, ph = (ci / kStateStages) & 1u;
                    if (held >= 0 && !mbar_test_wait(bar_st_done + 8 * s, ph)) {
                        tma_store_wait_read<0>();
                        mbar_arrive(bar_st_empty + 8 * held);
                        held = -1;
                    }
                    mbar_wait(bar_st_done + 8 * s, ph);
                    const uint32_t base = sST + s * Cfg::ST_STAGE;
                    const int x = tc.tn * BLOCK_N + c * CHUNK_N, y = tc.tm * BLOCK_M;
                    if (P.debug & DBG_NO_STATE) {
                    } else if constexpr (MODE == MODE_ADAMW) {
                        tma_store_2d(&pd.map_W, base, x, y, kEvictFirst);
                        tma_store_2d(&pd.map_m, base + Cfg::W_CHUNK, x, y, kEvictFirst);
                        tma_store_2d(&pd.map_v, base + Cfg::W_CHUNK + Cfg::M_CHUNK, x, y, kEvictFirst);
                    } else {
                        tma_store_2d(&pd.map_m, base + Cfg::W_CHUNK, x, y, kEvictFirst);
                    }
                    tma_store_commit();
                    if (held >= 0) {
                        tma_store_wait_read<1>();             // the previous group's source has been read
                        mbar_arrive(bar_st_empty + 8 * held);
                    }
                    held = static_cast<int>(s);
                }
            }
            tma_store_wait_all<0>();
            if (held >= 0) mbar_arrive(bar_st_empty + 8 * held);
        }
    } else {
        // ================= epilogue warpgroups (Alg. 1 lines 7-10 on the TMEM tile) ==============
        const int ew = warp - kCtrlWarps;
        const int wg = ew >> 2;                       // warpgroup 0/1
        const uint32_t quad = warp & 3;               // TMEM lane quadrant this warp may read
        const uint32_t row = quad * 32 + lane;        // row of the tile == TMEM lane
        const AdamWScalars hp = P.hp;
        uint32_t titer = 0;
        for (int tile = first_tile; tile < P.total_tiles; tile += tile_step, ++titer) {
            const uint32_t as = titer & 1u, aph = (titer >> 1) & 1u;
            if (!(P.debug & DBG_NO_MAINLOOP)) mbar_wait(bar_tm_full + 8 * as, aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((quad * 32u) << 16) + as * BLOCK_N;
            if constexpr (MDT != MDT_INT8) {
                for (int c = wg; c < CHUNKS; c += 2) {
                    const uint32_t ci = titer * CHUNKS + c;
                    const uint32_t s = ci % kStateStages, ph = (ci / kStateStages) & 1u;
                    uint32_t g[32];
                    tmem_ld_32x32b_x32(taddr + c * CHUNK_N, g);
                    const uint32_t base = sST + s * Cfg::ST_STAGE;
                    if constexpr (MODE == MODE_ADAMW) {
                        if (!(P.debug & DBG_NO_STATE)) mbar_wait(bar_st_full + 8 * s, ph);
                        else mbar_wait(bar_st_empty + 8 * s, ph ^ 1u);
                        tmem_ld_wait();
                        if (!(P.debug & DBG_NO_EPILOGUE))
                            epi_chunk_fp<MDT>(hp, g, base, base + Cfg::W_CHUNK,
                                              base + Cfg::W_CHUNK + Cfg::M_CHUNK, row);
                    } else {
                        mbar_wait(bar_st_empty + 8 * s, ph ^ 1u);
                        tmem_ld_wait();
                        epi_chunk_store_g(g, base + Cfg::W_CHUNK, row);
                    }
                    fence_proxy_async_smem();
                    mbar_arrive(bar_st_done + 8 * s);
                }
            } else {
                epi_tile_int8<Cfg, kStateStages, CG>(P, hp, tile, rank, titer, taddr, sST, bar_st_full,
                                                 bar_st_done, row, wg, s_xchg);
            }
            // this warp has drained the accumulator: tell the (leader's) MMA issuer
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if constexpr (CG == 2) mbar_arrive_cluster(mapa_shared(bar_tm_empty + 8 * as, 0));
                else mbar_arrive(bar_tm_empty + 8 * as);
            }
        }
    }

    __syncwarp();                                // lanes 1-31 of the single-thread roles rejoin lane 0
    tc_fence_before();
    if constexpr (CG == 2) cluster_sync_all();   // the peer may still read this CTA's smem / signal its barriers
    else __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        if constexpr (CG == 2) tmem_dealloc_cg2(tmem_base, kTmemCols);
        else tmem_dealloc(tmem_base, kTmemCols);
    }
}

}  // namespace forge
