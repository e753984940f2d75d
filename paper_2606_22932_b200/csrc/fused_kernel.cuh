// fused_kernel.cuh -- the persistent, warp-specialised sm_100a kernel of forge-b200.
//
// Per weight tile (128 rows of `out` x 256 columns of `in`), Algorithm 1:
//   lines 2-5  G_ij = sum_k dY_k,i^T X_k,j      tcgen05.mma, bf16 x bf16 -> fp32 in tensor memory
//   line  6    load W_ij, m_ij, v_ij            TMA, CM x CN chunks (64 x 128 with fp32 moments) into a smem ring
//   lines 7-10 AdamW in fp32 registers          adamw_math.cuh
//   line  11   store W_ij, m_ij, v_ij           in place in the smem chunk, then TMA store
// G never leaves the SM.  One CTA owns a tile for the whole token loop, so a
// partial-K update can never be applied.
//
// Warp roles (384 threads, one CTA per SM, CTA pairs share a 256 x 256 tile, persistent over a static tile list):
//   warp 0      operand producer: TMA loads of dY / X token chunks into the mainloop ring
//   warp 1      MMA issuer: one thread issues tcgen05.mma; accumulators double-buffered in TMEM
//   warp 2      TMEM allocator + state loader: TMA loads of W/m/v chunks (independent of G, so
//               they run ahead of the mainloop and across tile boundaries)
//   warp 3      state storer: TMA stores of finished chunks, recycles ring slots
//   warps 4-11  two epilogue warpgroups; warp w reads TMEM lanes 32*(w%4).., one W row per thread,
//               32 columns at a time: a chunk is cut into 32 x 32 sub-blocks, the warp whose TMEM
//               lane quadrant holds the rows takes them, warpgroup g the sub-block columns g, g+2, ..
//
// Both GEMM operands are MN-major: A = dY^T has `out` contiguous, B = X has `in` contiguous, and
// the token axis (K) is the slow axis of both.  A token chunk is staged as 64-element (128 B)
// swizzled rows: smem[mn_block][k][64], which is the canonical MN-major SWIZZLE_128B UMMA layout
// with LBO = kBlockK*128 B between 64-wide MN blocks and SBO = 1024 B between 8-token groups.
#pragma once
#include <cstdint>
#include <cstdio>
#include <cuda.h>
#include <cuda_runtime.h>

#include "adamw_math.cuh"
#include "family_math.cuh"
#include "ptx.cuh"

namespace forge {

constexpr int kMaxProblems = 8;
constexpr int BLOCK_M = 128;   // tile rows  (out)  = TMEM lanes
constexpr int BLOCK_N = 256;   // tile cols  (in)   = TMEM columns = one int8 block per row
constexpr int SUB = 32;        // epilogue sub-block: 32 rows (one warp's TMEM lanes) x 32 columns
constexpr int kCtrlWarps = 4;
// nwg = epilogue warpgroups (2, or 4: the floating-point paths then need four 32-column sub-blocks per chunk; with
// int8 moments nwg is the number of warps of one TMEM quadrant that share a row -- 3 measured slower: 485 vs 461 us/layer)
__host__ __device__ constexpr int epi_warps(int /*mdt*/, int nwg = 2) { return 4 * nwg; }
__host__ __device__ constexpr int block_threads(int mdt, int nwg = 2) { return (kCtrlWarps + epi_warps(mdt, nwg)) * 32; }
// L2 eviction priority of the state stream (W, m, v loads and the in-place stores).  Measured on the cfg-1 layer:
// evict_first for both 762 us, normal for both 729 us (fp32 moments; bf16 484 -> 459 us): the store that follows
// the load of the same lines a few microseconds later should still find them in L2.
constexpr uint64_t kStatePolicy = kEvictNormal;
constexpr int kTmemCols = 512;  // 2 accumulator buffers x 256 fp32 columns

enum : int { MDT_FP32 = 0, MDT_BF16 = 1, MDT_INT8 = 2, MDT_FP8 = 3 };
enum : int { MODE_ADAMW = 0, MODE_STORE_G = 1, MODE_FAMILY = 2,      // FAMILY: family_math.cuh, 0-2 state tensors
             MODE_ACCUM = 3,                                          // B <- mu*B + G, no weight
             MODE_ADAMW_SR = 4 };                                     // AdamW, stochastic-rounding store of W

struct alignas(64) ProblemDesc {
    CUtensorMap map_dY;  // [T, out] bf16, box {64, kBlockK}, SWIZZLE_128B
    CUtensorMap map_X;   // [T, in]  bf16, box {64, kBlockK}, SWIZZLE_128B
    CUtensorMap map_W;   // [out, in] bf16, box {min(CN, 64), CM}, swizzle = row bytes
    CUtensorMap map_m;   // [out, in] state dtype, box {min(CN, 128 B worth), CM}, swizzle = row bytes
    CUtensorMap map_v;   //   (MODE_STORE_G: map_m is the fp32 G output)
    CUtensorMap map_m1;  // INT8 only: the same m / v codes with box {128, 128}, SWIZZLE_128B, for the
    CUtensorMap map_v1;  //   absmax pass (read-only first-pass ring)
    float *m_scale;      // INT8: [out, in/256] block absmax; FP8: float[2] = {scale in use, amax out}
    float *v_scale;
    int32_t T, out, in;
    int32_t tiles_n;     // ceil(in / 256)
    int32_t tile_begin;  // first linear tile index of this problem
    uint32_t sr_inner;   // MODE_ADAMW_SR: fmix32(seed_hi ^ step ^ stream) of this problem
    char *pW, *pM, *pV;  // raw bases of W, m, v: the direct (ring-less) state path only
};

struct alignas(64) KernelParams {
    ProblemDesc prob[kMaxProblems];
    AdamWScalars hp;
    FamilyScalars fs;    // MODE_FAMILY only
    uint64_t pol_dy, pol_x;   // L2 eviction priority of the dY / X operand loads (host: by token count, see launch_fused)
    int32_t num_problems;
    int32_t total_tiles;
    uint32_t sr_seed_lo; // MODE_ADAMW_SR
    int32_t debug;       // -DFORGE_PROFILING builds only (libforge_b200_prof.so, used by the profiles/ commands): ablation
                         // switches, results are WRONG when set.  1 = no operand loads / MMA, 2 = no state loads / stores,
                         // 4 = no epilogue math, 8 = no state stores (direct path only).  The product build never reads it.
};
enum : int { DBG_NO_MAINLOOP = 1, DBG_NO_STATE = 2, DBG_NO_EPILOGUE = 4, DBG_NO_STORE = 8 /* direct path only */,
              DBG_NO_A = 16 /* CTA pairs: dY chunks loaded for the first ring pass only (operand traffic halved) */,
              DBG_TIMING = 64 /* print per-role wait / work clocks (results unchanged) */ };
#ifdef FORGE_PROFILING
#define FORGE_DBG(P, bit) (((P).debug & (bit)) != 0)
// FORGE_ABLATE bit 64: per-role clock accounting, printed by CTA 0 / 1 at exit (profiles/ only)
#define FORGE_TIMED_WAIT(acc, stmt) do { const long long t_ = clock64(); stmt; (acc) += clock64() - t_; } while (0)
#else
#define FORGE_DBG(P, bit) false
#define FORGE_TIMED_WAIT(acc, stmt) do { stmt; } while (0)
#endif

// CG = 1: one CTA per 128x256 tile.  CG = 2: a CTA pair (cluster of 2, tcgen05 cta_group::2) shares
// a 256x256 tile: each CTA stages its own 128 rows of A = dY^T and only HALF of B = X (128 of the
// 256 columns), the pair's leader issues one M=256 MMA that reads both CTAs' shared memory, and
// each CTA's TMEM receives its own 128 x 256 accumulator.  Operand bytes per CTA fall by a third
// (L2 -> SM traffic and smem per stage), the state path stays CTA-local.
// State chunk geometry.  The state stream (W, m, v once in, once out) is the roofline of the
// HBM-bound shapes, and what it achieves depends on the chunk shape more than on the depth of the
// ring: with fp32 moments 128 x 32 chunks x 4 slots give 0.83 of the copy peak, 64 x 64 x 4 slots 0.86
// and 64 x 128 x 2 slots 0.90 (profiles/r01_summary.md) -- longer contiguous runs per DRAM page and
// fewer pages open at once matter more than bytes in flight.
template <int MDT, int kBlockK, int kStages, int kStateStages, int CG = 1, int CM_ = 64, int CN_ = 64, int P1C_ = 128, int P1S_ = 2,
          int NST_ = 2, int HASW_ = 1, int NWG_ = 2>
struct KernelCfg {
    static constexpr int NWG = NWG_;                        // epilogue warpgroups (fp paths)
    static constexpr int HASW = HASW_;                      // the chunk image carries W (not in MODE_ACCUM)
    static constexpr int NST = NST_;                        // state tensors besides W in a chunk (AdamW: m, v)
    static constexpr int kMomBytes = (MDT == MDT_FP32) ? 4 : (MDT == MDT_BF16 ? 2 : 1);   // int8 and fp8: 1
    static constexpr int A_STAGE = kBlockK * 128 * (BLOCK_M / 64);
    static constexpr int B_STAGE = kBlockK * 128 * (BLOCK_N / 64) / CG;
    static constexpr int ML_STAGE = A_STAGE + B_STAGE;
    // chunk = CM rows x CN columns of the tile; RB x CB chunks per tile, row block fastest
    static constexpr int CM = CM_, CN = CN_;
    static constexpr int RB = BLOCK_M / CM, CB = BLOCK_N / CN, CHUNKS = RB * CB;
    static constexpr int SUBS = CN / SUB;                   // 32-column sub-blocks per chunk row
    static constexpr int WGS = SUBS >= NWG ? NWG : (SUBS >= 2 ? 2 : 1);   // warpgroups that share one chunk
    static_assert(NWG == 2 || (NWG == 4 && (SUBS >= 4 || MDT == MDT_INT8)), "four epilogue warpgroups need four sub-blocks per chunk row");
    // chunks ci and ci + PERIOD are consumed by the same warps
    static constexpr int PERIOD = RB * (SUBS >= 2 ? 1 : 2);
    static constexpr int DONE_COUNT = (CM / SUB) * (MDT == MDT_INT8 ? NWG : WGS);   // one arrival per warp that works on a chunk
    // TMA boxes: at most 128 B per row (one swizzle span), CM rows
    static constexpr int W_BOX_COLS = CN < 64 ? CN : 64;
    static constexpr int W_ROW = W_BOX_COLS * 2;
    static constexpr int W_BOXES = CN / W_BOX_COLS;
    static constexpr int W_BOX = CM * W_ROW;
    static constexpr int W_CHUNK = HASW ? W_BOXES * W_BOX : 0;
    static constexpr int M_BOX_COLS = CN < 128 / kMomBytes ? CN : 128 / kMomBytes;
    static constexpr int M_ROW = M_BOX_COLS * kMomBytes;
    static constexpr int M_BOXES = CN / M_BOX_COLS;
    static constexpr int M_BOX = CM * M_ROW;
    static constexpr int M_CHUNK = M_BOXES * M_BOX;
    static constexpr int ST_STAGE = W_CHUNK + NST * M_CHUNK;
    static constexpr int ST_TX_BYTES = ST_STAGE;
    // INT8: a second, read-only ring feeds the absmax pass: chunks of 128 rows x 128 columns of m and
    // of v codes (one 128 x 128 B box each), two slots = one tile
    static constexpr int P1_COLS = P1C_;                       // 128 or 64 columns per chunk (row bytes = swizzle span)
    static constexpr int P1_CHUNKS = BLOCK_N / P1_COLS;
    static constexpr int P1_STAGES = (MDT == MDT_INT8) ? P1S_ : 0;
    static constexpr int P1_BOX = 128 * P1_COLS;
    static constexpr int P1_STAGE = 2 * P1_BOX;
    static constexpr int kNumBars = 2 * kStages + 4 + 3 * kStateStages + 2 * P1_STAGES;
    // partial row maxima of the warps sharing a row.  Two buffers (alternating by tile) with the code ring; ONE with the
    // resident tile: a warp can only write the next tile's maxima after the next tile's first chunk has been loaded, which
    // needs every warp's arrival on that slot in pass 2 of this tile, i.e. after every warp has read this tile's maxima.
    static constexpr int XCHG_BUFS = (MDT == MDT_INT8 && P1S_ == 0) ? 1 : 2;
    static constexpr int XCHG_BYTES = (MDT == MDT_INT8) ? XCHG_BUFS * NWG * 1024 : 0;
    // the dynamic shared memory is declared __align__(1024) (checked at kernel entry): no alignment slack is reserved
    static constexpr int SMEM_BYTES = kStages * ML_STAGE + kStateStages * ST_STAGE +
                                      P1_STAGES * P1_STAGE + kNumBars * 8 + 16 + XCHG_BYTES;
    static_assert(SMEM_BYTES <= 232448, "shared memory budget exceeded");
    static_assert(kBlockK % 16 == 0 && kBlockK >= 16, "kBlockK must be a multiple of UMMA_K");
    static_assert(CG == 1 || CG == 2, "CTA group is 1 or 2");
    static_assert(BLOCK_M % CM == 0 && BLOCK_N % CN == 0 && CM % SUB == 0 && CN % SUB == 0, "chunk must tile the tile");
    static_assert(W_BOX % 1024 == 0 && M_BOX % 1024 == 0, "boxes must keep the swizzle pattern aligned");
    static_assert(MDT != MDT_INT8 || (CM == 128 && CN == 64), "the int8 path is written for 128 x 64 chunks (one 32-column half per warpgroup)");
    // Chunk ci lives in ring slot ci % kStateStages.  With the ring a multiple of PERIOD every slot is
    // always consumed by the same warps, so a warp observes every phase of the slot barriers it
    // waits on; otherwise it would skip phases and an mbarrier parity wait could alias to a phase
    // two steps back.
    static_assert(kStateStages % PERIOD == 0 && CHUNKS % PERIOD == 0, "ring must be a multiple of the consumer period");
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

// byte offset of 16-byte piece j of row r in a TMA-swizzled box whose rows are ROW bytes long
template <int ROW>
__device__ __forceinline__ uint32_t swz(uint32_t r, uint32_t j) {
    if constexpr (ROW == 128) return r * 128u + ((j ^ (r & 7u)) << 4);
    else if constexpr (ROW == 64) return r * 64u + ((j ^ ((r >> 1) & 3u)) << 4);
    else return r * 32u + ((j ^ ((r >> 2) & 1u)) << 4);
}

// Where the 32 columns [col, col + 32) of chunk row r live in the chunk's shared-memory image.
template <class Cfg>
struct SubAddr {
    uint32_t w, m, v;      // box base addresses (shared window)
    uint32_t pw, pm;       // first 16-byte piece of the sub-block inside the box row
    __device__ __forceinline__ SubAddr(uint32_t chunk_base, int col) {
        const int wb = col / Cfg::W_BOX_COLS, mb = col / Cfg::M_BOX_COLS;
        w = chunk_base + wb * Cfg::W_BOX;
        m = chunk_base + Cfg::W_CHUNK + mb * Cfg::M_BOX;
        v = m + Cfg::M_CHUNK;
        pw = (col % Cfg::W_BOX_COLS) * 2 / 16;
        pm = (col % Cfg::M_BOX_COLS) * Cfg::kMomBytes / 16;
    }
};

// ---------------------------------------------------------------------------------------------
// epilogue bodies: one thread = one W row of the chunk, one 32-column sub-block at a time
// ---------------------------------------------------------------------------------------------
template <int MDT, class Cfg, bool SR = false>
__device__ __forceinline__ void epi_sub_fp(const AdamWScalars &hp, const uint32_t (&g)[32],
                                           const SubAddr<Cfg> &a, uint32_t row, uint32_t rowkey = 0, uint32_t col0 = 0) {
    // 4 groups of 8 columns: one 16 B piece of W (8 bf16) + matching moments, as 4 coordinate pairs
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t aw = a.w + swz<Cfg::W_ROW>(row, a.pw + j);
        const uint4 wq = lds128(aw);
        f32x2 w[4] = {bf16x2_to_f32x2(wq.x), bf16x2_to_f32x2(wq.y), bf16x2_to_f32x2(wq.z), bf16x2_to_f32x2(wq.w)};
        f32x2 m[4], v[4];
        if constexpr (MDT == MDT_FP32) {
            const uint32_t o0 = swz<Cfg::M_ROW>(row, a.pm + 2 * j), o1 = swz<Cfg::M_ROW>(row, a.pm + 2 * j + 1);
            const uint32_t am0 = a.m + o0, am1 = a.m + o1, av0 = a.v + o0, av1 = a.v + o1;
            const uint4 x = lds128(am0), b = lds128(am1), c = lds128(av0), d = lds128(av1);
            m[0] = pk2u(x.x, x.y); m[1] = pk2u(x.z, x.w); m[2] = pk2u(b.x, b.y); m[3] = pk2u(b.z, b.w);
            v[0] = pk2u(c.x, c.y); v[1] = pk2u(c.z, c.w); v[2] = pk2u(d.x, d.y); v[3] = pk2u(d.z, d.w);
#pragma unroll
            for (int e = 0; e < 4; ++e) adamw_update2(hp, pk2u(g[8 * j + 2 * e], g[8 * j + 2 * e + 1]), w[e], m[e], v[e]);
            sts128(am0, make_uint4(lo2u(m[0]), hi2u(m[0]), lo2u(m[1]), hi2u(m[1])));
            sts128(am1, make_uint4(lo2u(m[2]), hi2u(m[2]), lo2u(m[3]), hi2u(m[3])));
            sts128(av0, make_uint4(lo2u(v[0]), hi2u(v[0]), lo2u(v[1]), hi2u(v[1])));
            sts128(av1, make_uint4(lo2u(v[2]), hi2u(v[2]), lo2u(v[3]), hi2u(v[3])));
        } else {
            const uint32_t o = swz<Cfg::M_ROW>(row, a.pm + j);
            const uint32_t am = a.m + o, av = a.v + o;
            const uint4 x = lds128(am), c = lds128(av);
            m[0] = bf16x2_to_f32x2(x.x); m[1] = bf16x2_to_f32x2(x.y); m[2] = bf16x2_to_f32x2(x.z); m[3] = bf16x2_to_f32x2(x.w);
            v[0] = bf16x2_to_f32x2(c.x); v[1] = bf16x2_to_f32x2(c.y); v[2] = bf16x2_to_f32x2(c.z); v[3] = bf16x2_to_f32x2(c.w);
#pragma unroll
            for (int e = 0; e < 4; ++e) adamw_update2(hp, pk2u(g[8 * j + 2 * e], g[8 * j + 2 * e + 1]), w[e], m[e], v[e]);
            sts128(am, make_uint4(f32x2_to_bf16x2(m[0]), f32x2_to_bf16x2(m[1]), f32x2_to_bf16x2(m[2]), f32x2_to_bf16x2(m[3])));
            sts128(av, make_uint4(f32x2_to_bf16x2(v[0]), f32x2_to_bf16x2(v[1]), f32x2_to_bf16x2(v[2]), f32x2_to_bf16x2(v[3])));
        }
        if constexpr (SR) {
            const uint32_t c = col0 + 8 * j;
            sts128(aw, make_uint4(f32x2_to_bf16x2_sr(w[0], rowkey, c), f32x2_to_bf16x2_sr(w[1], rowkey, c + 2),
                                  f32x2_to_bf16x2_sr(w[2], rowkey, c + 4), f32x2_to_bf16x2_sr(w[3], rowkey, c + 6)));
        } else {
            sts128(aw, make_uint4(f32x2_to_bf16x2(w[0]), f32x2_to_bf16x2(w[1]), f32x2_to_bf16x2(w[2]), f32x2_to_bf16x2(w[3])));
        }
    }
}

// fp8 (e4m3) moments with per-tensor delayed scaling: ONE pass -- the scale in use comes from
// the previous step, this step only reports its amax -- so the mode streams like bf16 at int8's byte count
struct Fp8Row {
    float bm, bv, inv_m, inv_v;    // beta * scale (dequantisation folded into the moment update), 1 / scale
};
// Direct state path (kStateStages == 0, tensor-bound shapes).  At large T the mainloop's operand traffic alone
// takes most of the shared-memory bandwidth (per MMA of 128 clocks each SM reads 8 KB of operands and TMA writes
// 8 KB), and the state ring adds four more passes over 20 B/element (TMA in, ld.shared, st.shared, TMA out):
// measured at T = 8192 the ring costs 114 us on a 650 us mainloop.  Here each thread owns one row of the tile and
// moves its 16 columns per step with 32-byte global accesses, registers only; step s + 1 is loaded before step s
// is computed.  Same arithmetic and rounding as epi_sub_fp.
template <int MDT>
struct DirectRegs {
    static constexpr int MV = (MDT == MDT_FP32) ? 2 : 1;   // 32-byte vectors of m (and of v) per 16 columns
    uint32_t w[8], m[MV][8], v[MV][8];
};
template <int MDT>
__device__ __forceinline__ void direct_load(DirectRegs<MDT> &r, const char *Wp, const char *Mp, const char *Vp) {
    ldg256(Wp, r.w);
#pragma unroll
    for (int i = 0; i < DirectRegs<MDT>::MV; ++i) {
        ldg256(Mp + 32 * i, r.m[i]);
        ldg256(Vp + 32 * i, r.v[i]);
    }
}
template <int MDT>
__device__ __forceinline__ void direct_step(const AdamWScalars &hp, const uint32_t (&g)[16], DirectRegs<MDT> &r,
                                            char *Wp, char *Mp, char *Vp, bool no_store = false) {
#pragma unroll
    for (int e = 0; e < 8; ++e) {               // coordinate pairs (2e, 2e + 1)
        f32x2 w = bf16x2_to_f32x2(r.w[e]), m, v;
        if constexpr (MDT == MDT_FP32) {
            m = pk2u(r.m[e / 4][(2 * e) % 8], r.m[e / 4][(2 * e) % 8 + 1]);
            v = pk2u(r.v[e / 4][(2 * e) % 8], r.v[e / 4][(2 * e) % 8 + 1]);
        } else {
            m = bf16x2_to_f32x2(r.m[0][e]);
            v = bf16x2_to_f32x2(r.v[0][e]);
        }
        adamw_update2(hp, pk2u(g[2 * e], g[2 * e + 1]), w, m, v);
        r.w[e] = f32x2_to_bf16x2(w);
        if constexpr (MDT == MDT_FP32) {
            r.m[e / 4][(2 * e) % 8] = lo2u(m); r.m[e / 4][(2 * e) % 8 + 1] = hi2u(m);
            r.v[e / 4][(2 * e) % 8] = lo2u(v); r.v[e / 4][(2 * e) % 8 + 1] = hi2u(v);
        } else {
            r.m[0][e] = f32x2_to_bf16x2(m);
            r.v[0][e] = f32x2_to_bf16x2(v);
        }
    }
    if (no_store) return;                       // profiling ablation only
    stg256(Wp, r.w);
#pragma unroll
    for (int i = 0; i < DirectRegs<MDT>::MV; ++i) {
        stg256(Mp + 32 * i, r.m[i]);
        stg256(Vp + 32 * i, r.v[i]);
    }
}

template <class Cfg>
__device__ __forceinline__ void epi_sub_fp8(const AdamWScalars &hp, const Fp8Row &R, const uint32_t (&g)[32],
                                            const SubAddr<Cfg> &a, uint32_t row, float &pm, float &pv) {
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const uint32_t o = swz<Cfg::M_ROW>(row, a.pm + j);
        const uint32_t am = a.m + o, av = a.v + o;
        const uint4 mq = lds128(am), vq = lds128(av);
        const uint32_t aw0 = a.w + swz<Cfg::W_ROW>(row, a.pw + 2 * j), aw1 = a.w + swz<Cfg::W_ROW>(row, a.pw + 2 * j + 1);
        const uint4 w0 = lds128(aw0), w1 = lds128(aw1);
        const uint32_t mw[4] = {mq.x, mq.y, mq.z, mq.w}, vw[4] = {vq.x, vq.y, vq.z, vq.w};
        const uint32_t ww[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
        uint32_t mo[4], vo[4], wo[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t mc = 0, vc = 0;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int gi = 16 * j + 4 * q + 2 * e;
                f32x2 m, v, w = bf16x2_to_f32x2(ww[2 * q + e]);
                adamw_moments2_q(hp, pk2u(g[gi], g[gi + 1]), e4m3x2_to_f32x2(mw[q] >> (16 * e)), e4m3x2_to_f32x2(vw[q] >> (16 * e)),
                                 R.bm, R.bv, m, v);
                adamw_weight2(hp, m, v, w);
                wo[2 * q + e] = f32x2_to_bf16x2(w);
                pm = fmaxf(pm, fmaxf(fabsf(lo2(m)), fabsf(hi2(m))));
                pv = fmaxf(pv, fmaxf(lo2(v), hi2(v)));
                mc |= f32x2_to_e4m3x2(mul2(m, bc2(R.inv_m))) << (16 * e);
                vc |= f32x2_to_e4m3x2(mul2(v, bc2(R.inv_v))) << (16 * e);
            }
            mo[q] = mc;
            vo[q] = vc;
        }
        sts128(am, make_uint4(mo[0], mo[1], mo[2], mo[3]));
        sts128(av, make_uint4(vo[0], vo[1], vo[2], vo[3]));
        sts128(aw0, make_uint4(wo[0], wo[1], wo[2], wo[3]));
        sts128(aw1, make_uint4(wo[4], wo[5], wo[6], wo[7]));
    }
}

// the other coordinate-wise families (family_math.cuh): 0, 1 or 2 state tensors in the chunk image
template <int MDT, class Cfg, bool HAS_M, int V_MODE, bool LION, bool DENOM>
__device__ __forceinline__ void epi_sub_family_t(const FamilyScalars &fs, const uint32_t (&g)[32],
                                                 const SubAddr<Cfg> &a, uint32_t row) {
    constexpr int NST = Cfg::NST;
    constexpr bool ONE_IS_V = (NST == 1) && !HAS_M;        // a single state tensor is the momentum when the
                                                           // family has one, else the second-moment state
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t aw = a.w + swz<Cfg::W_ROW>(row, a.pw + j);
        const uint4 wq = lds128(aw);
        f32x2 w[4] = {bf16x2_to_f32x2(wq.x), bf16x2_to_f32x2(wq.y), bf16x2_to_f32x2(wq.z), bf16x2_to_f32x2(wq.w)};
        f32x2 s[2][4];                                     // s[0]: state 0, s[1]: state 1
        uint32_t as[2][2];
#pragma unroll
        for (int t = 0; t < 2; ++t) {
#pragma unroll
            for (int e = 0; e < 4; ++e) s[t][e] = 0ull;
            if (t >= NST) continue;
            const uint32_t base = t == 0 ? a.m : a.v;
            if constexpr (MDT == MDT_FP32) {
                as[t][0] = base + swz<Cfg::M_ROW>(row, a.pm + 2 * j);
                as[t][1] = base + swz<Cfg::M_ROW>(row, a.pm + 2 * j + 1);
                const uint4 x = lds128(as[t][0]), y = lds128(as[t][1]);
                s[t][0] = pk2u(x.x, x.y); s[t][1] = pk2u(x.z, x.w); s[t][2] = pk2u(y.x, y.y); s[t][3] = pk2u(y.z, y.w);
            } else {
                as[t][0] = base + swz<Cfg::M_ROW>(row, a.pm + j);
                const uint4 x = lds128(as[t][0]);
                s[t][0] = bf16x2_to_f32x2(x.x); s[t][1] = bf16x2_to_f32x2(x.y);
                s[t][2] = bf16x2_to_f32x2(x.z); s[t][3] = bf16x2_to_f32x2(x.w);
            }
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const f32x2 gg = pk2u(g[8 * j + 2 * e], g[8 * j + 2 * e + 1]);
            if constexpr (ONE_IS_V) family_update2<HAS_M, V_MODE, LION, DENOM>(fs, gg, w[e], s[1][e], s[0][e]);
            else family_update2<HAS_M, V_MODE, LION, DENOM>(fs, gg, w[e], s[0][e], s[1][e]);
        }
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            if (t >= NST) continue;
            if constexpr (MDT == MDT_FP32) {
                sts128(as[t][0], make_uint4(lo2u(s[t][0]), hi2u(s[t][0]), lo2u(s[t][1]), hi2u(s[t][1])));
                sts128(as[t][1], make_uint4(lo2u(s[t][2]), hi2u(s[t][2]), lo2u(s[t][3]), hi2u(s[t][3])));
            } else {
                sts128(as[t][0], make_uint4(f32x2_to_bf16x2(s[t][0]), f32x2_to_bf16x2(s[t][1]),
                                            f32x2_to_bf16x2(s[t][2]), f32x2_to_bf16x2(s[t][3])));
            }
        }
        sts128(aw, make_uint4(f32x2_to_bf16x2(w[0]), f32x2_to_bf16x2(w[1]), f32x2_to_bf16x2(w[2]), f32x2_to_bf16x2(w[3])));
    }
}

// one uniform switch per sub-block on the family's structure; only the kinds its state count allows
template <int MDT, class Cfg>
__device__ __forceinline__ void epi_sub_family(const FamilyScalars &fs, const uint32_t (&g)[32],
                                               const SubAddr<Cfg> &a, uint32_t row) {
    if constexpr (Cfg::NST == 0) {
        epi_sub_family_t<MDT, Cfg, false, V_NONE, false, false>(fs, g, a, row);
    } else if constexpr (Cfg::NST == 1) {
        if (fs.kind == FK_M) epi_sub_family_t<MDT, Cfg, true, V_NONE, false, false>(fs, g, a, row);
        else if (fs.kind == FK_LION) epi_sub_family_t<MDT, Cfg, true, V_NONE, true, false>(fs, g, a, row);
        else epi_sub_family_t<MDT, Cfg, false, V_EMA, false, true>(fs, g, a, row);
    } else {
        if (fs.kind == FK_MV) epi_sub_family_t<MDT, Cfg, true, V_EMA, false, true>(fs, g, a, row);
        else if (fs.kind == FK_MV_MAX) epi_sub_family_t<MDT, Cfg, true, V_MAX, false, true>(fs, g, a, row);
        else epi_sub_family_t<MDT, Cfg, true, V_EMA, false, false>(fs, g, a, row);
    }
}

// accumulate-into-state (regime 2): B <- mu*B + G "through the GEMM's own beta";
// the chunk image holds B only, no weight is read or written and no gradient exists
template <int MDT, class Cfg>
__device__ __forceinline__ void epi_sub_accum(float mu, const uint32_t (&g)[32], const SubAddr<Cfg> &a, uint32_t row) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        f32x2 b[4];
        if constexpr (MDT == MDT_FP32) {
            const uint32_t a0 = a.m + swz<Cfg::M_ROW>(row, a.pm + 2 * j), a1 = a.m + swz<Cfg::M_ROW>(row, a.pm + 2 * j + 1);
            const uint4 x = lds128(a0), y = lds128(a1);
            b[0] = pk2u(x.x, x.y); b[1] = pk2u(x.z, x.w); b[2] = pk2u(y.x, y.y); b[3] = pk2u(y.z, y.w);
#pragma unroll
            for (int e = 0; e < 4; ++e) b[e] = fma2(bc2(mu), b[e], pk2u(g[8 * j + 2 * e], g[8 * j + 2 * e + 1]));
            sts128(a0, make_uint4(lo2u(b[0]), hi2u(b[0]), lo2u(b[1]), hi2u(b[1])));
            sts128(a1, make_uint4(lo2u(b[2]), hi2u(b[2]), lo2u(b[3]), hi2u(b[3])));
        } else {
            const uint32_t a0 = a.m + swz<Cfg::M_ROW>(row, a.pm + j);
            const uint4 x = lds128(a0);
            b[0] = bf16x2_to_f32x2(x.x); b[1] = bf16x2_to_f32x2(x.y); b[2] = bf16x2_to_f32x2(x.z); b[3] = bf16x2_to_f32x2(x.w);
#pragma unroll
            for (int e = 0; e < 4; ++e) b[e] = fma2(bc2(mu), b[e], pk2u(g[8 * j + 2 * e], g[8 * j + 2 * e + 1]));
            sts128(a0, make_uint4(f32x2_to_bf16x2(b[0]), f32x2_to_bf16x2(b[1]), f32x2_to_bf16x2(b[2]), f32x2_to_bf16x2(b[3])));
        }
    }
}

// store-G twin: the fp32 sub-block goes to the chunk's m image unchanged
template <class Cfg>
__device__ __forceinline__ void epi_sub_store_g(const uint32_t (&g)[32], const SubAddr<Cfg> &a, uint32_t row) {
#pragma unroll
    for (int j = 0; j < 8; ++j)
        sts128(a.m + swz<Cfg::M_ROW>(row, a.pm + j), make_uint4(g[4 * j], g[4 * j + 1], g[4 * j + 2], g[4 * j + 3]));
}


// int8 blockwise moments (App. B; 256-element blocks along `in` == one block per tile
// row).  The new block absmax is only known once all 256 m', v' of the row exist, and a tile's state
// (128 KB) cannot be double-buffered in shared memory, so the tile is walked twice over the TMEM
// accumulator with the state STREAMED both times:
//   pass 1: the m / v codes of the tile come through a small read-only ring (128 rows x 128 columns
//       per chunk); m', v' are formed from the accumulator and only the row maxima are kept;
//   pass 2: W and the codes come through the in-place ring (the codes again: an L2 hit, they were
//       read microseconds ago); the identical m', v' are recomputed (same instructions, same
//       operands), W' formed, the state requantised with the new scales and stored in place.
// A row is owned by one thread of each warpgroup (each takes half of the columns); the two partial
// maxima are combined through shared memory.  DRAM traffic is unchanged (8.06 B / element);
// L2 -> SM traffic grows by the 2 B / element of the second code read.
struct Int8Smem {
    uint32_t p1, bar_p1_full, bar_p1_empty, xchg;
};
struct Int8Row {           // per-thread view of its row's 256-block in one tile
    size_t sidx;
    float a_m, a_v;        // old block absmax as stored (loaded a tile ahead; no arithmetic on them until used)
    float bm, bv;          // beta * (old absmax / levels): dequantisation folded into the moment update
    bool valid;
    __device__ __forceinline__ void finish(const AdamWScalars &hp) {
        bm = __fmul_rn(hp.q_b1, dequant_step(a_m, 127.0f));      // scaled moments m'' = m'/(1-beta1), v'' = v'/(1-beta2)
        bv = __fmul_rn(hp.q_b2, dequant_step(a_v, 255.0f));
    }
};

// pass 1: row maxima of m', v' ("absmax") over this warp's half of the columns
template <class Cfg>
__device__ __forceinline__ void int8_pass1(const AdamWScalars &hp, const Int8Row &R, uint32_t titer, uint32_t taddr,
                                           const Int8Smem &S, uint32_t row_t, int wg, float &pm, float &pv,
                                           bool skip_math, bool no_state, long long &t_wait) {
    pm = 0.0f;
    pv = 0.0f;
    constexpr int kSubs = Cfg::P1_COLS / SUB;              // 32-column sub-blocks per chunk; sub-block t of the
                                                           // row goes to warp t % NWG of the quadrant
#pragma unroll 1
    for (int c1 = 0; c1 < Cfg::P1_CHUNKS; ++c1) {
        const uint32_t i1 = titer * Cfg::P1_CHUNKS + c1, s = i1 % Cfg::P1_STAGES, ph = (i1 / Cfg::P1_STAGES) & 1u;
        const uint32_t am = S.p1 + s * Cfg::P1_STAGE, av = am + Cfg::P1_BOX;
        if (!no_state) FORGE_TIMED_WAIT(t_wait, mbar_wait(S.bar_p1_full + 8 * s, ph));
#pragma unroll 1
        for (int j32 = 0; j32 < (skip_math ? 0 : kSubs); ++j32) {
            if ((c1 * kSubs + j32) % Cfg::NWG != wg) continue;
            uint32_t g[32];
            tmem_ld_32x32b_x32(taddr + c1 * Cfg::P1_COLS + j32 * SUB, g);
            const uint32_t o0 = swz<Cfg::P1_COLS>(row_t, 2 * j32), o1 = swz<Cfg::P1_COLS>(row_t, 2 * j32 + 1);
            const uint4 mq[2] = {lds128(am + o0), lds128(am + o1)}, vq[2] = {lds128(av + o0), lds128(av + o1)};
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const uint32_t mw[4] = {mq[j].x, mq[j].y, mq[j].z, mq[j].w}, vw[4] = {vq[j].x, vq[j].y, vq[j].z, vq[j].w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    f32x2 cm[2], cv[2];
                    codes4_to_f32(mw[q], true, cm[0], cm[1]);
                    codes4_to_f32(vw[q], false, cv[0], cv[1]);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int gi = 16 * j + 4 * q + 2 * e;
                        f32x2 m, v;
                        adamw_moments2_qs(pk2u(g[gi], g[gi + 1]), cm[e], cv[e], R.bm, R.bv, m, v);
                        pm = fmaxf(pm, fmaxf(fabsf(lo2(m)), fabsf(hi2(m))));
                        pv = fmaxf(pv, fmaxf(lo2(v), hi2(v)));           // v' >= 0
                    }
                }
            }
        }
        __syncwarp();
        if ((row_t & 31u) == 0) mbar_arrive(S.bar_p1_empty + 8 * s);   // this warp has read the codes: one arrival per warp
    }
}

// pass 1, resident-tile variant (P1_STAGES == 0): there is no separate code ring -- the state ring holds every chunk of
// the tile (W + codes, loaded ONCE) from its first use here until pass 2 has rewritten it in place, plus one or two
// spare slots in which the next tile's first chunks arrive meanwhile.  The codes cross L2 -> SM once instead of twice.
template <class Cfg, int kStateStages>
__device__ __forceinline__ void int8_pass1_ring(const Int8Row &R, uint32_t titer, uint32_t taddr, uint32_t sST,
                                                uint32_t bar_st_full, uint32_t row_t, int wg, float &pm, float &pv,
                                                bool skip_math, bool no_state, long long &t_wait) {
    pm = 0.0f;
    pv = 0.0f;
    const uint32_t rb = row_t / Cfg::CM, row = row_t % Cfg::CM;
#pragma unroll 1
    for (int cb = 0; cb < Cfg::CB; ++cb) {
        const uint32_t ci = titer * Cfg::CHUNKS + cb * Cfg::RB + rb;
        const uint32_t s = ci % kStateStages, ph = (ci / kStateStages) & 1u;
        if (!no_state) FORGE_TIMED_WAIT(t_wait, mbar_wait(bar_st_full + 8 * s, ph));
#pragma unroll 1
        for (int half = 0; half < Cfg::SUBS; ++half) {
            if (skip_math || (cb * Cfg::SUBS + half) % Cfg::NWG != wg) continue;
            uint32_t g[32];
            tmem_ld_32x32b_x32(taddr + cb * Cfg::CN + half * SUB, g);
            const SubAddr<Cfg> a(sST + s * Cfg::ST_STAGE, half * SUB);
            const uint32_t o0 = swz<Cfg::M_ROW>(row, a.pm), o1 = swz<Cfg::M_ROW>(row, a.pm + 1);
            const uint4 mq[2] = {lds128(a.m + o0), lds128(a.m + o1)}, vq[2] = {lds128(a.v + o0), lds128(a.v + o1)};
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const uint32_t mw[4] = {mq[j].x, mq[j].y, mq[j].z, mq[j].w}, vw[4] = {vq[j].x, vq[j].y, vq[j].z, vq[j].w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    f32x2 cm[2], cv[2];
                    codes4_to_f32(mw[q], true, cm[0], cm[1]);
                    codes4_to_f32(vw[q], false, cv[0], cv[1]);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int gi = 16 * j + 4 * q + 2 * e;
                        f32x2 m, v;
                        adamw_moments2_qs(pk2u(g[gi], g[gi + 1]), cm[e], cv[e], R.bm, R.bv, m, v);
                        pm = fmaxf(pm, fmaxf(fabsf(lo2(m)), fabsf(hi2(m))));
                        pv = fmaxf(pv, fmaxf(lo2(v), hi2(v)));           // v' >= 0
                    }
                }
            }
        }
    }
}

// pass 2: W' and the requantised state for this warp's 32-column half of every chunk
template <class Cfg, int kStateStages>
__device__ __forceinline__ void int8_pass2(const AdamWScalars &hp, const Int8Row &R, float a_m, float a_v,
                                           uint32_t titer, uint32_t taddr, uint32_t sST, uint32_t bar_st_full,
                                           uint32_t bar_st_done, uint32_t bar_st_empty, uint32_t row_t, int wg,
                                           bool skip_math, bool no_state, long long &t_wait) {
    const uint32_t rb = row_t / Cfg::CM, row = row_t % Cfg::CM;
    const float bm = R.bm, bv = R.bv;
    const float inv_m = quant_inv_scale(a_m, 127.0f), inv_v = quant_inv_scale(a_v, 255.0f);
    const float v_floor = quant_v_floor(inv_v);
#pragma unroll 1
    for (int cb = 0; cb < Cfg::CB; ++cb) {
        const uint32_t ci = titer * Cfg::CHUNKS + cb * Cfg::RB + rb;
        const uint32_t s = ci % kStateStages, ph = (ci / kStateStages) & 1u;
        if (!no_state) FORGE_TIMED_WAIT(t_wait, mbar_wait(bar_st_full + 8 * s, ph));
        else mbar_wait(bar_st_empty + 8 * s, ph ^ 1u);
#pragma unroll 1
        for (int half = 0; half < Cfg::SUBS; ++half) {
        if (skip_math || (cb * Cfg::SUBS + half) % Cfg::NWG != wg) continue;
        uint32_t g[32];
        tmem_ld_32x32b_x32(taddr + cb * Cfg::CN + half * SUB, g);
        const SubAddr<Cfg> a(sST + s * Cfg::ST_STAGE, half * SUB);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const uint32_t o = swz<Cfg::M_ROW>(row, a.pm + j);
            const uint32_t am = a.m + o, av = a.v + o;
            const uint4 mq = lds128(am), vq = lds128(av);
            const uint32_t aw0 = a.w + swz<Cfg::W_ROW>(row, a.pw + 2 * j), aw1 = a.w + swz<Cfg::W_ROW>(row, a.pw + 2 * j + 1);
            const uint4 w0 = lds128(aw0), w1 = lds128(aw1);
            const uint32_t mw[4] = {mq.x, mq.y, mq.z, mq.w}, vw[4] = {vq.x, vq.y, vq.z, vq.w};
            const uint32_t ww[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
            uint32_t mo[4], vo[4], wo[8];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                f32x2 cm[2], cv[2], qm[2], qv[2];
                codes4_to_f32(mw[q], true, cm[0], cm[1]);
                codes4_to_f32(vw[q], false, cv[0], cv[1]);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int gi = 16 * j + 4 * q + 2 * e;
                    f32x2 m, v, w = bf16x2_to_f32x2(ww[2 * q + e]);
                    adamw_moments2_qs(pk2u(g[gi], g[gi + 1]), cm[e], cv[e], bm, bv, m, v);
                    adamw_weight2_s(hp, m, v, w);
                    wo[2 * q + e] = f32x2_to_bf16x2(w);
                    qm[e] = quant_m2(m, inv_m);
                    qv[e] = quant_v2(v, inv_v, v_floor);
                }
                mo[q] = pack_codes4(qm[0], qm[1]);
                vo[q] = pack_codes4(qv[0], qv[1]);
            }
            sts128(am, make_uint4(mo[0], mo[1], mo[2], mo[3]));
            sts128(av, make_uint4(vo[0], vo[1], vo[2], vo[3]));
            sts128(aw0, make_uint4(wo[0], wo[1], wo[2], wo[3]));
            sts128(aw1, make_uint4(wo[4], wo[5], wo[6], wo[7]));
        }
        }
        // every thread orders its own writes before the async proxy, the warp synchronises, one lane signals the storer
        fence_proxy_async_smem();
        __syncwarp();
        if ((row_t & 31u) == 0) mbar_arrive(bar_st_done + 8 * s);
    }
}

template <int CG>
__device__ __forceinline__ Int8Row int8_row(const KernelParams &P, const AdamWScalars &hp, int tile, uint32_t rank,
                                            uint32_t row_t) {
    const TileCoord tc = decode_tile<CG>(P, tile, rank);
    const ProblemDesc &pd = P.prob[tc.p];
    const int row_g = tc.tm * BLOCK_M + static_cast<int>(row_t);
    Int8Row R;
    R.valid = row_g < pd.out;
    R.sidx = static_cast<size_t>(R.valid ? row_g : 0) * static_cast<size_t>(pd.in / BLOCK_N) + tc.tn;
    R.a_m = R.valid ? pd.m_scale[R.sidx] : 0.0f;
    R.a_v = R.valid ? pd.v_scale[R.sidx] : 0.0f;
    R.bm = R.bv = 0.0f;
    return R;
}

// int8 state loader: one thread feeds both rings, polling whichever has a free slot
template <class Cfg, int kStateStages, int CG>
__device__ __forceinline__ void int8_loader(const KernelParams &P, uint32_t rank, int first_tile, int tile_step,
                                            uint32_t sST, uint32_t bar_st_full, uint32_t bar_st_empty,
                                            const Int8Smem &S) {
    if (first_tile >= P.total_tiles) return;
    const uint32_t my_tiles = (P.total_tiles - first_tile + tile_step - 1) / tile_step;
    const uint32_t n1 = my_tiles * Cfg::P1_CHUNKS, n2 = my_tiles * Cfg::CHUNKS;
    uint32_t i1 = 0, i2 = 0;
    TileCoord tc1 = decode_tile<CG>(P, first_tile, rank), tc2 = tc1;
    while (i1 < n1 || i2 < n2) {
        if (i1 < n1) {
            const uint32_t s = i1 % Cfg::P1_STAGES, ph = (i1 / Cfg::P1_STAGES) & 1u;
            if (mbar_test_wait(S.bar_p1_empty + 8 * s, ph ^ 1u)) {
                if ((i1 % Cfg::P1_CHUNKS) == 0 && i1 > 0) tc1 = decode_tile<CG>(P, first_tile + (i1 / Cfg::P1_CHUNKS) * tile_step, rank);
                const ProblemDesc &pd = P.prob[tc1.p];
                const uint32_t full = S.bar_p1_full + 8 * s, base = S.p1 + s * Cfg::P1_STAGE;
                mbar_expect_tx(full, Cfg::P1_STAGE);
                const int x = tc1.tn * BLOCK_N + (i1 % Cfg::P1_CHUNKS) * Cfg::P1_COLS, y = tc1.tm * BLOCK_M;
                tma_load_2d(base, &pd.map_m1, full, x, y, kEvictNormal);
                tma_load_2d(base + Cfg::P1_BOX, &pd.map_v1, full, x, y, kEvictNormal);
                ++i1;
            }
        }
        if (i2 < n2) {
            const uint32_t s = i2 % kStateStages, ph = (i2 / kStateStages) & 1u;
            if (mbar_test_wait(bar_st_empty + 8 * s, ph ^ 1u)) {
                const uint32_t c = i2 % Cfg::CHUNKS;
                if (c == 0 && i2 > 0) tc2 = decode_tile<CG>(P, first_tile + (i2 / Cfg::CHUNKS) * tile_step, rank);
                const ProblemDesc &pd = P.prob[tc2.p];
                const uint32_t full = bar_st_full + 8 * s, base = sST + s * Cfg::ST_STAGE;
                mbar_expect_tx(full, Cfg::ST_TX_BYTES);
                const int x = tc2.tn * BLOCK_N + (c / Cfg::RB) * Cfg::CN, y = tc2.tm * BLOCK_M + (c % Cfg::RB) * Cfg::CM;
                tma_load_2d(base, &pd.map_W, full, x, y, kStatePolicy);
                tma_load_2d(base + Cfg::W_CHUNK, &pd.map_m, full, x, y, kStatePolicy);
                tma_load_2d(base + Cfg::W_CHUNK + Cfg::M_CHUNK, &pd.map_v, full, x, y, kStatePolicy);
                ++i2;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <int MDT, int MODE, int kBlockK, int kStages, int kStateStages, int CG, int CM, int CN, int P1C, int P1S, int NST, int NWG>
__global__ void __launch_bounds__(block_threads(MDT, NWG), 1)
forge_fused_kernel(const __grid_constant__ KernelParams P) {
    constexpr int HASW = (MODE == MODE_ACCUM) ? 0 : 1;
    using Cfg = KernelCfg<MDT, kBlockK, kStages, kStateStages, CG, CM, CN, P1C, P1S, NST, HASW, NWG>;
    static_assert(MODE != MODE_ADAMW_SR || (MDT != MDT_INT8 && MDT != MDT_FP8), "the SR store is implemented for fp32 / bf16 moments");
    static_assert(MDT != MDT_FP8 || MODE == MODE_ADAMW, "fp8 moments are implemented for AdamW");
    static_assert(MODE == MODE_FAMILY || MODE == MODE_ACCUM || NST == 2, "AdamW and the store-G twin use the two-state chunk image");
    static_assert(MODE != MODE_ACCUM || NST == 1, "accumulate-into-state has exactly one state tensor");
    static_assert((MODE != MODE_FAMILY && MODE != MODE_ACCUM) || MDT != MDT_INT8, "int8 state is implemented for AdamW only");
    constexpr int CHUNKS = Cfg::CHUNKS;
    constexpr bool DIRECT = (kStateStages == 0);      // no state ring: the epilogue moves W, m, v itself (direct_step)
    constexpr uint32_t SSN = DIRECT ? 1 : kStateStages;
    static_assert(!DIRECT || (MODE == MODE_ADAMW && (MDT == MDT_FP32 || MDT == MDT_BF16)), "the direct state path is AdamW, fp32 / bf16 moments");
    const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;   // rank 0 = the pair's leader
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem_base = smem_u32(smem_raw);
    if (smem_base & 1023u) __trap();   // the swizzled TMA / UMMA layouts need 1024-byte aligned stages
    const uint32_t sML = smem_base;                                   // mainloop ring
    const uint32_t sST = sML + kStages * Cfg::ML_STAGE;               // state ring
    const uint32_t sP1 = sST + kStateStages * Cfg::ST_STAGE;          // INT8: first-pass code ring
    const uint32_t sBAR = sP1 + Cfg::P1_STAGES * Cfg::P1_STAGE;       // mbarriers
    // barrier map
    const uint32_t bar_ml_full = sBAR;
    const uint32_t bar_ml_empty = bar_ml_full + 8 * kStages;
    const uint32_t bar_tm_full = bar_ml_empty + 8 * kStages;          // [2]
    const uint32_t bar_tm_empty = bar_tm_full + 16;                   // [2]
    const uint32_t bar_st_full = bar_tm_empty + 16;
    const uint32_t bar_st_done = bar_st_full + 8 * kStateStages;
    const uint32_t bar_st_empty = bar_st_done + 8 * kStateStages;
    const uint32_t bar_p1_full = bar_st_empty + 8 * kStateStages;     // INT8 only [P1_STAGES]
    const uint32_t bar_p1_empty = bar_p1_full + 8 * Cfg::P1_STAGES;
    const uint32_t s_tmem_ptr = bar_p1_empty + 8 * Cfg::P1_STAGES;
    const Int8Smem i8{sP1, bar_p1_full, bar_p1_empty, s_tmem_ptr + 16};

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        for (int i = 0; i < kStages; ++i) {
            mbar_init(bar_ml_full + 8 * i, 1);
            mbar_init(bar_ml_empty + 8 * i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar_tm_full + 8 * i, 1);
            mbar_init(bar_tm_empty + 8 * i, epi_warps(MDT, NWG) * CG);   // one arrival per epilogue warp of the pair
        }
        for (int i = 0; i < kStateStages; ++i) {
            mbar_init(bar_st_full + 8 * i, 1);
            mbar_init(bar_st_done + 8 * i, Cfg::DONE_COUNT);
            mbar_init(bar_st_empty + 8 * i, 1);
        }
        for (int i = 0; i < Cfg::P1_STAGES; ++i) {
            mbar_init(bar_p1_full + 8 * i, 1);
            mbar_init(bar_p1_empty + 8 * i, epi_warps(MDT, NWG));          // every epilogue warp reads its part of the chunk
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
        if (lane == 0 && !FORGE_DBG(P, DBG_NO_MAINLOOP)) {
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
                                        kb * kBlockK, P.pol_dy);
#pragma unroll
                        for (int i = 0; i < BLOCK_N / 64; ++i)
                            tma_load_2d(b + i * kBlockK * 128, &pd.map_X, full, tc.tn * BLOCK_N + i * 64,
                                        kb * kBlockK, P.pol_x);
                    } else {
                        // both CTAs' bytes are counted on the LEADER's full barrier
                        const bool no_a = FORGE_DBG(P, DBG_NO_A) && it >= kStages;
                        if (rank == 0) mbar_expect_tx(bar_ml_full + 8 * s, 2 * (Cfg::ML_STAGE - (no_a ? Cfg::A_STAGE : 0)));
                        const uint32_t full = mapa_shared(bar_ml_full + 8 * s, 0);
#pragma unroll
                        for (int i = 0; i < (no_a ? 0 : BLOCK_M / 64); ++i)
                            tma_load_2d_cg2(a + i * kBlockK * 128, &pd.map_dY, full, tc.tm * BLOCK_M + i * 64,
                                            kb * kBlockK, P.pol_dy);
#pragma unroll
                        for (int i = 0; i < BLOCK_N / 128; ++i)   // this CTA's half of the 256 columns
                            tma_load_2d_cg2(b + i * kBlockK * 128, &pd.map_X, full,
                                            tc.tn * BLOCK_N + static_cast<int>(rank) * (BLOCK_N / 2) + i * 64,
                                            kb * kBlockK, P.pol_x);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (Alg. 1 line 4: G_ij += dY_k,i^T X_k,j) =====================
        if (lane == 0 && rank == 0 && !FORGE_DBG(P, DBG_NO_MAINLOOP)) {
            constexpr uint32_t idesc = make_idesc_bf16_f32_mnmn(BLOCK_M * CG, BLOCK_N);
            uint32_t it = 0, titer = 0;
            [[maybe_unused]] long long t_acc = 0, t_ops = 0;
#ifdef FORGE_PROFILING
            const long long t_begin = clock64();
#endif
            for (int tile = first_tile; tile < P.total_tiles; tile += tile_step, ++titer) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const int num_kb = (P.prob[tc.p].T + kBlockK - 1) / kBlockK;
                const uint32_t as = titer & 1u, aph = (titer >> 1) & 1u;
                FORGE_TIMED_WAIT(t_acc, mbar_wait(bar_tm_empty + 8 * as, aph ^ 1u));   // epilogue has drained this buffer
                tc_fence_after();
                const uint32_t tmem_d = tmem_base + as * BLOCK_N;
                for (int kb = 0; kb < num_kb; ++kb, ++it) {
                    const uint32_t s = it % kStages, ph = (it / kStages) & 1u;
                    FORGE_TIMED_WAIT(t_ops, mbar_wait(bar_ml_full + 8 * s, ph));
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
#ifdef FORGE_PROFILING
            if (FORGE_DBG(P, DBG_TIMING) && blockIdx.x < 2)
                printf("cta %d MMA issuer tiles %u total %lld | wait accumulator free %lld | wait operands %lld\n", blockIdx.x, titer,
                       clock64() - t_begin, t_acc, t_ops);
#endif
        }
    } else if (warp == 2) {
        // ================= state loader (Alg. 1 line 6: load W_ij, m_ij, v_ij) ===================
        if constexpr (MDT == MDT_INT8 && Cfg::P1_STAGES > 0) {
            if (lane == 0 && !FORGE_DBG(P, DBG_NO_STATE))
                int8_loader<Cfg, kStateStages, CG>(P, rank, first_tile, tile_step, sST, bar_st_full, bar_st_empty, i8);
        } else if (!DIRECT && MODE != MODE_STORE_G && lane == 0 && !FORGE_DBG(P, DBG_NO_STATE)) {
            uint32_t ci = 0;  // running chunk counter
            for (int tile = first_tile; tile < P.total_tiles; tile += tile_step) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const ProblemDesc &pd = P.prob[tc.p];
                for (int c = 0; c < CHUNKS; ++c, ++ci) {
                    const uint32_t s = ci % SSN, ph = (ci / SSN) & 1u;
                    mbar_wait(bar_st_empty + 8 * s, ph ^ 1u);
                    const uint32_t full = bar_st_full + 8 * s;
                    mbar_expect_tx(full, Cfg::ST_TX_BYTES);
                    const uint32_t base = sST + s * Cfg::ST_STAGE;
                    const int x = tc.tn * BLOCK_N + (c / Cfg::RB) * CN, y = tc.tm * BLOCK_M + (c % Cfg::RB) * CM;
                    if constexpr (HASW) {
#pragma unroll
                        for (int i = 0; i < Cfg::W_BOXES; ++i)
                            tma_load_2d(base + i * Cfg::W_BOX, &pd.map_W, full, x + i * Cfg::W_BOX_COLS, y, kStatePolicy);
                    }
                    if constexpr (NST >= 1) {
#pragma unroll
                        for (int i = 0; i < Cfg::M_BOXES; ++i)
                            tma_load_2d(base + Cfg::W_CHUNK + i * Cfg::M_BOX, &pd.map_m, full, x + i * Cfg::M_BOX_COLS, y, kStatePolicy);
                    }
                    if constexpr (NST >= 2) {
#pragma unroll
                        for (int i = 0; i < Cfg::M_BOXES; ++i)
                            tma_load_2d(base + Cfg::W_CHUNK + Cfg::M_CHUNK + i * Cfg::M_BOX, &pd.map_v, full,
                                        x + i * Cfg::M_BOX_COLS, y, kStatePolicy);
                    }
                }
            }
        }
    } else if (warp == 3) {
        // ================= state storer (Alg. 1 line 11: store W_ij, m_ij, v_ij) ================
        if (!DIRECT && lane == 0) {
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
                    const uint32_t s = ci % SSN, ph = (ci / SSN) & 1u;
                    if (held >= 0 && !mbar_test_wait(bar_st_done + 8 * s, ph)) {
                        tma_store_wait_read<0>();
                        mbar_arrive(bar_st_empty + 8 * held);
                        held = -1;
                    }
                    mbar_wait(bar_st_done + 8 * s, ph);
                    const uint32_t base = sST + s * Cfg::ST_STAGE;
                    const int x = tc.tn * BLOCK_N + (c / Cfg::RB) * CN, y = tc.tm * BLOCK_M + (c % Cfg::RB) * CM;
                    if (FORGE_DBG(P, DBG_NO_STATE)) {
                    } else {
                        if constexpr (MODE != MODE_STORE_G && HASW) {
#pragma unroll
                            for (int i = 0; i < Cfg::W_BOXES; ++i)
                                tma_store_2d(&pd.map_W, base + i * Cfg::W_BOX, x + i * Cfg::W_BOX_COLS, y, kStatePolicy);
                        }
                        if constexpr (NST >= 1) {
#pragma unroll
                            for (int i = 0; i < Cfg::M_BOXES; ++i)      // MODE_STORE_G: the m image carries G
                                tma_store_2d(&pd.map_m, base + Cfg::W_CHUNK + i * Cfg::M_BOX, x + i * Cfg::M_BOX_COLS, y, kStatePolicy);
                        }
                        if constexpr (MODE != MODE_STORE_G && NST >= 2) {
#pragma unroll
                            for (int i = 0; i < Cfg::M_BOXES; ++i)
                                tma_store_2d(&pd.map_v, base + Cfg::W_CHUNK + Cfg::M_CHUNK + i * Cfg::M_BOX,
                                             x + i * Cfg::M_BOX_COLS, y, kStatePolicy);
                        }
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
        const int wg = ew >> 2;                       // warpgroup 0 .. NWG-1
        const uint32_t quad = warp & 3;               // TMEM lane quadrant this warp may read
        const uint32_t row_t = quad * 32 + lane;      // row of the tile == TMEM lane
        const uint32_t rb = row_t / CM, row = row_t % CM;   // this warp's row block, row inside the chunk
        const AdamWScalars hp = P.hp;
        Int8Row i8row{};
        uint32_t titer = 0;
        [[maybe_unused]] long long t_tm = 0, t_w1 = 0, t_w2 = 0, t_p1 = 0, t_x = 0, t_p2 = 0;   // DBG_TIMING: wait / work clocks of this warp
#ifdef FORGE_PROFILING
        const long long t_begin = clock64();
#endif
        for (int tile = first_tile; tile < P.total_tiles; tile += tile_step, ++titer) {
            const uint32_t as = titer & 1u, aph = (titer >> 1) & 1u;
            if (!FORGE_DBG(P, DBG_NO_MAINLOOP)) FORGE_TIMED_WAIT(t_tm, mbar_wait(bar_tm_full + 8 * as, aph));
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((quad * 32u) << 16) + as * BLOCK_N;
            uint32_t sr_rowkey = 0, sr_col0 = 0;
            if constexpr (MODE == MODE_ADAMW_SR) {
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                sr_rowkey = sr_row_key(static_cast<uint32_t>(tc.tm * BLOCK_M) + row_t, P.sr_seed_lo, P.prob[tc.p].sr_inner);
                sr_col0 = static_cast<uint32_t>(tc.tn * BLOCK_N);
            }
            Fp8Row f8{};
            float f8_pm = 0.0f, f8_pv = 0.0f;
            if constexpr (MDT == MDT_FP8) {
                const ProblemDesc &pd = P.prob[decode_tile<CG>(P, tile, rank).p];
                const float sm = __ldg(pd.m_scale), sv = __ldg(pd.v_scale);     // [0] = scale in use (previous step's amax / 448)
                f8.bm = __fmul_rn(hp.beta1, sm);
                f8.bv = __fmul_rn(hp.beta2, sv);
                f8.inv_m = fp8_inv_scale(sm);
                f8.inv_v = fp8_inv_scale(sv);
            }
            if constexpr (DIRECT) {
                // each warpgroup takes one 128-column half of the tile, each thread its row, 16 columns per step
                const TileCoord tc = decode_tile<CG>(P, tile, rank);
                const ProblemDesc &pd = P.prob[tc.p];
                constexpr int MB = Cfg::kMomBytes;
                const int grow = tc.tm * BLOCK_M + static_cast<int>(row_t);
                const int col0 = tc.tn * BLOCK_N + wg * (BLOCK_N / 2);
                const bool row_ok = grow < pd.out && !FORGE_DBG(P, DBG_NO_STATE);
                const size_t e0 = static_cast<size_t>(row_ok ? grow : 0) * pd.in + col0;
                char *Wp = pd.pW + e0 * 2, *Mp = pd.pM + e0 * MB, *Vp = pd.pV + e0 * MB;
                constexpr int STEPS = BLOCK_N / 2 / 16;
                DirectRegs<MDT> R[2];
                if (row_ok && col0 < pd.in) direct_load<MDT>(R[0], Wp, Mp, Vp);
#pragma unroll
                for (int st = 0; st < STEPS; ++st) {
                    uint32_t g[16];
                    tmem_ld_32x32b_x16(taddr + wg * (BLOCK_N / 2) + st * 16, g);
                    const bool ok = row_ok && col0 + st * 16 < pd.in;
                    if (st + 1 < STEPS && row_ok && col0 + (st + 1) * 16 < pd.in)
                        direct_load<MDT>(R[(st + 1) & 1], Wp + (st + 1) * 32, Mp + (st + 1) * 16 * MB, Vp + (st + 1) * 16 * MB);
                    tmem_ld_wait();
                    if (ok && !FORGE_DBG(P, DBG_NO_EPILOGUE))
                        direct_step<MDT>(hp, g, R[st & 1], Wp + st * 32, Mp + st * 16 * MB, Vp + st * 16 * MB,
                                         FORGE_DBG(P, DBG_NO_STORE));
                }
            } else if constexpr (MDT != MDT_INT8) {
                for (int cb = 0; cb < Cfg::CB; ++cb) {
                    if (Cfg::SUBS < 2 && (cb & 1) != wg) continue;
                    const uint32_t ci = titer * CHUNKS + cb * Cfg::RB + rb;
                    const uint32_t s = ci % SSN, ph = (ci / SSN) & 1u;
                    const uint32_t base = sST + s * Cfg::ST_STAGE;
                    if (MODE != MODE_STORE_G && !FORGE_DBG(P, DBG_NO_STATE)) FORGE_TIMED_WAIT(t_w2, mbar_wait(bar_st_full + 8 * s, ph));
                    else mbar_wait(bar_st_empty + 8 * s, ph ^ 1u);
                    for (int j32 = (Cfg::SUBS >= 2 ? wg : 0); j32 < Cfg::SUBS; j32 += Cfg::WGS) {
                        uint32_t g[32];
                        tmem_ld_32x32b_x32(taddr + cb * CN + j32 * SUB, g);
                        const SubAddr<Cfg> a(base, j32 * SUB);
                        tmem_ld_wait();
                        if constexpr (MODE == MODE_ADAMW && MDT == MDT_FP8) {
                            if (!FORGE_DBG(P, DBG_NO_EPILOGUE)) epi_sub_fp8<Cfg>(hp, f8, g, a, row, f8_pm, f8_pv);
                        } else if constexpr (MODE == MODE_ADAMW) {
                            if (!FORGE_DBG(P, DBG_NO_EPILOGUE)) epi_sub_fp<MDT, Cfg>(hp, g, a, row);
                        } else if constexpr (MODE == MODE_ADAMW_SR) {
                            epi_sub_fp<MDT, Cfg, true>(hp, g, a, row, sr_rowkey, sr_col0 + cb * CN + j32 * SUB);
                        } else if constexpr (MODE == MODE_FAMILY) {
                            epi_sub_family<MDT, Cfg>(P.fs, g, a, row);
                        } else if constexpr (MODE == MODE_ACCUM) {
                            epi_sub_accum<MDT, Cfg>(P.fs.a1, g, a, row);
                        } else {
                            epi_sub_store_g<Cfg>(g, a, row);
                        }
                    }
                    fence_proxy_async_smem();             // each thread's writes -> async proxy; then one arrival per warp
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_st_done + 8 * s);
                }
                if constexpr (MDT == MDT_FP8) {          // this step's amax of m', v' for the NEXT step's scale
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        f8_pm = fmaxf(f8_pm, __shfl_xor_sync(0xffffffffu, f8_pm, o));
                        f8_pv = fmaxf(f8_pv, __shfl_xor_sync(0xffffffffu, f8_pv, o));
                    }
                    if (lane == 0) {                     // non-negative floats order like their bit patterns
                        const ProblemDesc &pd = P.prob[decode_tile<CG>(P, tile, rank).p];
                        atomicMax(reinterpret_cast<unsigned int *>(pd.m_scale + 1), __float_as_uint(f8_pm));
                        atomicMax(reinterpret_cast<unsigned int *>(pd.v_scale + 1), __float_as_uint(f8_pv));
                    }
                }
            } else {
                // old block scales of this row: loaded one tile ahead (global latency off the critical path)
                if (titer == 0) i8row = int8_row<CG>(P, hp, tile, rank, row_t);
                Int8Row R = i8row;
                if (tile + tile_step < P.total_tiles) i8row = int8_row<CG>(P, hp, tile + tile_step, rank, row_t);
                R.finish(hp);
                float pm, pv;
                if constexpr (Cfg::P1_STAGES > 0)
                    FORGE_TIMED_WAIT(t_p1, int8_pass1<Cfg>(hp, R, titer, taddr, i8, row_t, wg, pm, pv, FORGE_DBG(P, DBG_NO_EPILOGUE),
                                                           FORGE_DBG(P, DBG_NO_STATE), t_w1));
                else
                    FORGE_TIMED_WAIT(t_p1, (int8_pass1_ring<Cfg, kStateStages>(R, titer, taddr, sST, bar_st_full, row_t, wg, pm, pv,
                                                                               FORGE_DBG(P, DBG_NO_EPILOGUE), FORGE_DBG(P, DBG_NO_STATE),
                                                                               t_w1)));
#ifdef FORGE_PROFILING
                const long long t_x0 = clock64();
#endif
                // combine the two warpgroups' halves of the row (same TMEM quadrant: warps quad and 4 + quad)
                const uint32_t xb = i8.xchg + (Cfg::XCHG_BUFS == 2 ? (titer & 1u) * (NWG * 1024u) : 0u);
                asm volatile("st.shared.v2.f32 [%0], {%1, %2};\n" ::"r"(xb + (wg * 128u + row_t) * 8u), "f"(pm), "f"(pv) : "memory");
                asm volatile("bar.sync %0, %1;\n" ::"r"(1u + quad), "n"(NWG * 32) : "memory");
                float a_m = pm, a_v = pv;
#pragma unroll
                for (int o = 1; o < NWG; ++o) {
                    float om, ov;
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(om), "=f"(ov) : "r"(xb + (((wg + o) % NWG) * 128u + row_t) * 8u));
                    a_m = fmaxf(a_m, om);
                    a_v = fmaxf(a_v, ov);
                }
#ifdef FORGE_PROFILING
                t_x += clock64() - t_x0;
#endif
                FORGE_TIMED_WAIT(t_p2, (int8_pass2<Cfg, kStateStages>(hp, R, a_m, a_v, titer, taddr, sST, bar_st_full, bar_st_done,
                                                                      bar_st_empty, row_t, wg, FORGE_DBG(P, DBG_NO_EPILOGUE),
                                                                      FORGE_DBG(P, DBG_NO_STATE), t_w2)));
                if (wg == 0 && R.valid) {
                    const ProblemDesc &pd = P.prob[decode_tile<CG>(P, tile, rank).p];
                    pd.m_scale[R.sidx] = __fmul_rn(hp.one_minus_beta1, a_m);     // absmax of m', v' from the scaled maxima
                    pd.v_scale[R.sidx] = __fmul_rn(hp.one_minus_beta2, a_v);
                }
            }
            // this warp has drained the accumulator: tell the (leader's) MMA issuer
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if constexpr (CG == 2) mbar_arrive_cluster(mapa_shared(bar_tm_empty + 8 * as, 0));
                else mbar_arrive(bar_tm_empty + 8 * as);
            }
        }
#ifdef FORGE_PROFILING
        if (FORGE_DBG(P, DBG_TIMING) && blockIdx.x < 2 && lane == 0 && (warp == 4 || warp == 9))
            printf("cta %d warp %d tiles %u total %lld | wait G %lld | p1 %lld (wait codes %lld) | xchg %lld | p2/epi %lld (wait state %lld)\n",
                   blockIdx.x, warp, titer, clock64() - t_begin, t_tm, t_p1, t_w1, t_x, t_p2, t_w2);
#endif
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
