// forge_api.cu -- the C ABI of include/forge.h: argument validation, host-side scalars, tensor-map
// construction and kernel launches.  Allocates no device memory (except the scratch of the
// explicitly host-buffer entry point forge_wgrad_adamw_host, freed before it returns).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/forge.h"
#include "dgrad_kernel.cuh"
#include "elementwise_kernel.cuh"
#include "fused_kernel.cuh"

namespace {

using namespace forge;

std::atomic<uint64_t> g_launches{0};
std::atomic<int> g_last_cuda_error{0};
std::atomic<const char *> g_last_kernel{""};
std::atomic<int> g_tuning{FORGE_TUNE_BOOST_CLOCK};   // forge_set_tuning: explicit, process-wide, bit-identical either way     // signature of the instantiation the last launch used (forge_last_kernel)

forge_status_t cuda_fail(cudaError_t e) {
    g_last_cuda_error.store(static_cast<int>(e));
    return FORGE_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// driver entry point for tensor-map encoding (no link-time dependency on libcuda)
// ---------------------------------------------------------------------------------------------
using EncodeTiledFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                   const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                   CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                   CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    });
    return fn;
}

// 2D row-major tensor [rows, cols] of `esize`-byte elements; box {box_cols, box_rows}.
bool encode_2d(CUtensorMap *map, CUtensorMapDataType dt, int esize, const void *base, uint64_t rows,
               uint64_t cols, uint32_t box_cols, uint32_t box_rows, CUtensorMapSwizzle swz, uint64_t pitch_elems = 0) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {(pitch_elems ? pitch_elems : cols) * static_cast<uint64_t>(esize)};
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, dt, 2, const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

CUtensorMapSwizzle swizzle_for_row_bytes(int row_bytes) {
    return row_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                            : (row_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B);
}

// ---------------------------------------------------------------------------------------------
// validation and scalars
// ---------------------------------------------------------------------------------------------
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

forge_status_t validate_hp(int64_t step, float lr, float b1, float b2, float eps, float wd) {
    if (step < 1) return FORGE_ERR_BAD_HYPERPARAM;
    if (!std::isfinite(lr) || lr < 0.f) return FORGE_ERR_BAD_HYPERPARAM;
    if (!(b1 >= 0.f && b1 < 1.f) || !(b2 >= 0.f && b2 < 1.f)) return FORGE_ERR_BAD_HYPERPARAM;
    if (!std::isfinite(eps) || eps < 0.f) return FORGE_ERR_BAD_HYPERPARAM;
    if (!std::isfinite(wd) || wd < 0.f) return FORGE_ERR_BAD_HYPERPARAM;
    return FORGE_OK;
}

forge_status_t validate_state(const void *W, const void *m, const void *v, const float *ms, const float *vs,
                              int32_t out, int32_t in, int mdt) {
    if (mdt < 0 || mdt > 3) return FORGE_ERR_BAD_DTYPE;
    if (!W || !m || !v) return FORGE_ERR_NULL_PTR;
    if (mdt == FORGE_MOMENT_INT8 || mdt == FORGE_MOMENT_FP8) {
        if (!ms || !vs) return FORGE_ERR_NULL_PTR;
    } else if (ms || vs) {
        return FORGE_ERR_BAD_DTYPE;   // scales are meaningful for INT8 only
    }
    if (out < 8 || in < 8 || (out % 8) != 0 || (in % 8) != 0) return FORGE_ERR_BAD_SHAPE;
    if (mdt == FORGE_MOMENT_BF16 && (in % 8) != 0) return FORGE_ERR_BAD_SHAPE;
    if (mdt == FORGE_MOMENT_INT8 && (in % FORGE_QBLOCK) != 0) return FORGE_ERR_BAD_SHAPE;
    if (mdt == FORGE_MOMENT_FP8 && (in % 16) != 0) return FORGE_ERR_BAD_SHAPE;    // 16-byte rows of 1-byte codes
    if (!aligned16(W) || !aligned16(m) || !aligned16(v)) return FORGE_ERR_ALIGNMENT;
    if ((mdt == FORGE_MOMENT_INT8 || mdt == FORGE_MOMENT_FP8) &&
        ((reinterpret_cast<uintptr_t>(ms) & 3u) || (reinterpret_cast<uintptr_t>(vs) & 3u)))
        return FORGE_ERR_ALIGNMENT;
    return FORGE_OK;
}

// the two GEMM operands: pointers, token count, pitches, alignment (every entry point goes through this)
forge_status_t validate_operands(const forge_problem_t &p) {
    if (!p.X || !p.dY) return FORGE_ERR_NULL_PTR;
    if (p.T < 1 || p.out < 8 || p.in < 8 || (p.out % 8) != 0 || (p.in % 8) != 0) return FORGE_ERR_BAD_SHAPE;
    if (p.ldx != 0 && (p.ldx < p.in || p.ldx % 8 != 0)) return FORGE_ERR_BAD_SHAPE;
    if (p.lddy != 0 && (p.lddy < p.out || p.lddy % 8 != 0)) return FORGE_ERR_BAD_SHAPE;
    if (!aligned16(p.X) || !aligned16(p.dY)) return FORGE_ERR_ALIGNMENT;
    return FORGE_OK;
}
forge_status_t validate_problem(const forge_problem_t &p, int mdt) {
    if (!p.X || !p.dY) return FORGE_ERR_NULL_PTR;
    forge_status_t s = validate_state(p.W, p.m, p.v, p.m_scale, p.v_scale, p.out, p.in, mdt);
    if (s != FORGE_OK) return s;
    return validate_operands(p);
}
bool dense_operands(const forge_problem_t &p) {
    return (p.ldx == 0 || p.ldx == p.in) && (p.lddy == 0 || p.lddy == p.out);
}

// Aliasing (forge.h "Caller's obligations"): inside one call no updated tensor may overlap any other tensor the call
// touches -- overlapping state inside a group is a silent race between CTAs.  Read-only operands may be shared
// (q / k / v read one X).  Sort-and-sweep over the byte intervals, O(n log n) in the number of tensors.
struct Interval {
    uintptr_t lo, hi;
    bool written;
};
void add_interval(std::vector<Interval> &iv, const void *p, size_t bytes, bool written) {
    if (p && bytes) iv.push_back({reinterpret_cast<uintptr_t>(p), reinterpret_cast<uintptr_t>(p) + bytes, written});
}
size_t moment_bytes(int mdt) { return mdt == FORGE_MOMENT_FP32 ? 4 : (mdt == FORGE_MOMENT_BF16 ? 2 : 1); }
// every tensor of a problem: operands read-only, everything else written (absent tensors are NULL and skipped)
void add_problem_intervals(std::vector<Interval> &iv, const forge_problem_t &p, int mdt, size_t m_elem_bytes) {
    const size_t n = static_cast<size_t>(p.out) * p.in;
    const size_t ldx = p.ldx ? p.ldx : p.in, lddy = p.lddy ? p.lddy : p.out;
    add_interval(iv, p.X, ((static_cast<size_t>(p.T) - 1) * ldx + p.in) * 2, false);
    add_interval(iv, p.dY, ((static_cast<size_t>(p.T) - 1) * lddy + p.out) * 2, false);
    add_interval(iv, p.W, n * 2, true);
    add_interval(iv, p.m, n * m_elem_bytes, true);
    add_interval(iv, p.v, n * m_elem_bytes, true);
    const size_t sb = mdt == FORGE_MOMENT_INT8 ? n / FORGE_QBLOCK * 4 : (mdt == FORGE_MOMENT_FP8 ? 2 * sizeof(float) : 0);
    add_interval(iv, p.m_scale, sb, true);
    add_interval(iv, p.v_scale, sb, true);
}
forge_status_t check_disjoint(std::vector<Interval> &iv) {
    std::sort(iv.begin(), iv.end(), [](const Interval &a, const Interval &b) { return a.lo < b.lo; });
    uintptr_t end_any = 0, end_written = 0;
    for (const Interval &x : iv) {
        if (x.lo < end_written || (x.written && x.lo < end_any)) return FORGE_ERR_BAD_SHAPE;
        end_any = std::max(end_any, x.hi);
        if (x.written) end_written = std::max(end_written, x.hi);
    }
    return FORGE_OK;
}
forge_status_t validate_disjoint(const forge_problem_t *probs, int count, int mdt, size_t m_elem_bytes,
                                 void *const *extra_out = nullptr, const size_t *extra_bytes = nullptr) {
    std::vector<Interval> iv;
    iv.reserve(static_cast<size_t>(count) * 8);
    for (int i = 0; i < count; ++i) {
        add_problem_intervals(iv, probs[i], mdt, m_elem_bytes);
        if (extra_out) add_interval(iv, extra_out[i], extra_bytes[i], true);
    }
    return check_disjoint(iv);
}

// Alg. 1 line 9 bias terms and the folded constants, computed in double from the float
// hyper-parameters the ABI carries, rounded to float once.
AdamWScalars make_scalars(int64_t step, float lr, float b1, float b2, float eps, float wd) {
    AdamWScalars h;
    const double bc1 = 1.0 - std::pow(static_cast<double>(b1), static_cast<double>(step));
    const double bc2 = 1.0 - std::pow(static_cast<double>(b2), static_cast<double>(step));
    h.beta1 = b1;
    h.one_minus_beta1 = 1.0f - b1;
    h.beta2 = b2;
    h.one_minus_beta2 = 1.0f - b2;
    h.decay = static_cast<float>(1.0 - static_cast<double>(lr) * static_cast<double>(wd));
    const double d1 = 1.0 - static_cast<double>(b1), d2 = 1.0 - static_cast<double>(b2);
    h.q_b1 = static_cast<float>(static_cast<double>(b1) / d1);
    h.q_b2 = static_cast<float>(static_cast<double>(b2) / d2);
    // the step size lr / bc1 folded into the negated denominator (adamw_math.cuh); no step (lr = 0, or a quotient that
    // leaves the fp32 range): 0 * sqrt(v') - inf, whose reciprocal is -0
    const double step_size = static_cast<double>(lr) / bc1;
    const double c = 1.0 / std::sqrt(bc2);
    auto fold = [&](double coeff, double e, float &nc, float &ne) {
        nc = step_size > 0.0 ? static_cast<float>(-coeff / step_size) : 0.0f;
        ne = step_size > 0.0 ? static_cast<float>(-e / step_size) : -INFINITY;
        if (!std::isfinite(nc) || !std::isfinite(ne)) { nc = 0.0f; ne = -INFINITY; }
    };
    fold(c, static_cast<double>(eps), h.nd_c, h.nd_eps);
    fold(std::sqrt(d2) * c / d1, static_cast<double>(eps) / d1, h.nq_c, h.nq_eps);
    return h;
}

struct DeviceInfo {
    int device = -1, sm_count = 0, cc_major = 0;
    bool dry = false;   // encode every tensor map and set every function attribute, launch nothing (see for_each_launch)
};
forge_status_t device_info(DeviceInfo &d) {
    cudaError_t e = cudaGetDevice(&d.device);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, d.device);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, d.device);
    if (e != cudaSuccess) return cuda_fail(e);
    if (d.cc_major != 10) return FORGE_ERR_UNSUPPORTED_ARCH;
    return FORGE_OK;
}

// The tuning / ablation switches FORGE_CFG, FORGE_GRID, FORGE_ABLATE, FORGE_HOST_SLICE_MB exist only in the
// -DFORGE_PROFILING build (libforge_b200_prof.so, loaded by the profiles/ commands and two tests).  The product
// library reads no environment variable: nothing left over in a shell can change a launch or a result.
#ifdef FORGE_PROFILING
int env_int(const char *name, int dflt) {
    const char *s = std::getenv(name);
    return s ? std::atoi(s) : dflt;
}
#else
constexpr int env_int(const char *, int dflt) { return dflt; }
#endif

// A group of more than kMaxProblems problems takes several launches.  All of them are prepared (tensor maps encoded,
// function attributes set) in a dry pass BEFORE the first one is enqueued, so that the only failure left once state
// has been touched is a launch failure itself.  f(first, n, dev) prepares or launches problems [first, first + n).
template <class F>
forge_status_t for_each_launch(int count, DeviceInfo dev, F f) {
    for (int pass = (count > kMaxProblems ? 0 : 1); pass < 2; ++pass) {
        dev.dry = (pass == 0);
        for (int i = 0; i < count; i += kMaxProblems) {
            const forge_status_t s = f(i, std::min(count - i, kMaxProblems), dev);
            if (s != FORGE_OK) return s;
        }
    }
    return FORGE_OK;
}

// ---------------------------------------------------------------------------------------------
// launch of one fused-kernel instantiation over <= kMaxProblems problems
// ---------------------------------------------------------------------------------------------
template <int MDT, int MODE, int BK, int ST, int SS, int CG = 1, int CM = 64, int CN = 64, int P1C = 128, int P1S = 2,
          int NST = 2, int NWG = 2>
forge_status_t launch_fused(const forge_problem_t *probs, int count, const AdamWScalars &hp,
                            const DeviceInfo &dev, cudaStream_t stream, const FamilyScalars *fs = nullptr,
                            uint64_t sr_seed = 0, uint32_t sr_step = 0, uint32_t sr_stream0 = 0) {
    using Cfg = KernelCfg<MDT, BK, ST, SS, CG, CM, CN, P1C, P1S, NST, (MODE == MODE_ACCUM) ? 0 : 1, NWG>;
    auto kernel = forge_fused_kernel<MDT, MODE, BK, ST, SS, CG, CM, CN, P1C, P1S, NST, NWG>;
    // the opt-in shared-memory size is a per-device function attribute: set it once per device, not once per process
    static std::atomic<uint64_t> attr_done{0};
    const uint64_t dev_bit = 1ull << (dev.device & 63);
    if (!(attr_done.load(std::memory_order_acquire) & dev_bit)) {
        const cudaError_t ae = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
        if (ae != cudaSuccess) return cuda_fail(ae);
        attr_done.fetch_or(dev_bit, std::memory_order_release);
    }

    KernelParams P;
    std::memset(&P, 0, sizeof(P));
    P.hp = hp;
    if (fs) P.fs = *fs;
    P.num_problems = count;
    int tiles = 0;
    constexpr CUtensorMapDataType mom_dt = (MDT == MDT_FP32) ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                           : (MDT == MDT_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                                              : CU_TENSOR_MAP_DATA_TYPE_UINT8);   // int8 and fp8 codes
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = probs[i];
        ProblemDesc &d = P.prob[i];
        bool ok = true;
        ok &= encode_2d(&d.map_dY, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p.dY, p.T, p.out, 64, BK, CU_TENSOR_MAP_SWIZZLE_128B,
                        static_cast<uint64_t>(p.lddy));
        ok &= encode_2d(&d.map_X, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p.X, p.T, p.in, 64, BK, CU_TENSOR_MAP_SWIZZLE_128B,
                        static_cast<uint64_t>(p.ldx));
        if (MODE != MODE_STORE_G) {
            if (MODE != MODE_ACCUM)
                ok &= encode_2d(&d.map_W, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p.W, p.out, p.in, Cfg::W_BOX_COLS, CM,
                                swizzle_for_row_bytes(Cfg::W_ROW));
            if (NST >= 1)
                ok &= encode_2d(&d.map_m, mom_dt, Cfg::kMomBytes, p.m, p.out, p.in, Cfg::M_BOX_COLS, CM,
                                swizzle_for_row_bytes(Cfg::M_ROW));
            if (NST >= 2)
                ok &= encode_2d(&d.map_v, mom_dt, Cfg::kMomBytes, p.v, p.out, p.in, Cfg::M_BOX_COLS, CM,
                                swizzle_for_row_bytes(Cfg::M_ROW));
            if (MDT == MDT_INT8) {   // first-pass view of the same codes: 128 rows x 128 columns per box
                ok &= encode_2d(&d.map_m1, mom_dt, 1, p.m, p.out, p.in, P1C, 128, swizzle_for_row_bytes(P1C));
                ok &= encode_2d(&d.map_v1, mom_dt, 1, p.v, p.out, p.in, P1C, 128, swizzle_for_row_bytes(P1C));
            }
        } else {  // store-G twin: p.m carries the fp32 G output
            ok &= encode_2d(&d.map_m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, p.m, p.out, p.in, Cfg::M_BOX_COLS, CM,
                            swizzle_for_row_bytes(Cfg::M_ROW));
        }
        if (!ok) return cuda_fail(cudaErrorInvalidValue);
        d.m_scale = p.m_scale;
        d.v_scale = p.v_scale;
        d.pW = static_cast<char *>(p.W);
        d.pM = static_cast<char *>(p.m);
        d.pV = static_cast<char *>(p.v);
        d.T = p.T;
        d.out = p.out;
        d.in = p.in;
        d.tiles_n = (p.in + BLOCK_N - 1) / BLOCK_N;
        d.tile_begin = tiles;
        d.sr_inner = sr_inner_key_host(static_cast<uint32_t>(sr_seed >> 32), sr_step, sr_stream0 + static_cast<uint32_t>(i));
        tiles += ((p.out + BLOCK_M * CG - 1) / (BLOCK_M * CG)) * d.tiles_n;   // (128*CG) x 256 work units
    }
    P.total_tiles = tiles;
    // L2 eviction priority of the operand streams: evict_last for X; for dY evict_last, except evict_normal at
    // 2048 <= T < 8192.  Measured on gate_proj (profiles/r02_summary.md): dY evict_first is slower at every T (T = 8192:
    // 764 vs 750 us, DRAM reads 2.48 vs 1.80 GB -- the sixteen pairs of a tile row do not read a dY line at the same
    // instant); dY evict_normal is 2.2 % faster at T = 2048 (275.3 vs 281.4 us, three alternating runs each), 0.8 % at
    // T = 4096, equal at T = 512 and T = 8192.
    {
        const int pol = env_int("FORGE_POLICY", -1);   // FORGE_PROFILING build only: 0 both evict_last, 1 dY first, 2 dY normal, 3 X normal, 4 both normal
        int max_T = 0;
        for (int i = 0; i < count; ++i) max_T = std::max(max_T, static_cast<int>(probs[i].T));
        const bool dy_normal = pol < 0 ? (max_T >= 2048 && max_T < 8192) : (pol == 2 || pol == 4);
        P.pol_dy = pol == 1 ? kEvictFirst : (dy_normal ? kEvictNormal : kEvictLast);
        P.pol_x = (pol == 3 || pol == 4) ? kEvictNormal : kEvictLast;
    }
    P.sr_seed_lo = static_cast<uint32_t>(sr_seed);
    P.debug = env_int("FORGE_ABLATE", 0);          // FORGE_PROFILING build only (constant 0 otherwise)
    int grid = dev.sm_count / CG;                  // persistent: one CTA (or CTA pair) per SM (pair)
    const int forced = env_int("FORGE_GRID", 0);   // FORGE_PROFILING build only: determinism test across grid sizes
    if (forced > 0) grid = (forced + CG - 1) / CG;
    if (grid > tiles) grid = tiles;
    if (dev.dry) return FORGE_OK;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(grid * CG));
    cfg.blockDim = dim3(block_threads(MDT, NWG));
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, P);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1);
    static const std::string sig = [] {
        const int a[12] = {MDT, MODE, BK, ST, SS, CG, CM, CN, P1C, P1S, NST, NWG};
        std::string t = "forge_fused_kernel<";
        for (int i = 0; i < 12; ++i) t += std::to_string(a[i]) + (i < 11 ? ", " : ">");
        return t;
    }();
    g_last_kernel.store(sig.c_str());
    return FORGE_OK;
}

// Static per-shape configuration table (the paper searches this space with an autotuner,
// PAPER.md:706-710 App. H; here the choice is fixed per moment dtype and token count):
//   small T : HBM-bound -> short token chunks, state ring as deep as shared memory allows
//   large T : tensor-bound -> 64-token chunks, 4-stage operand ring, shallow state ring
//   T >= 8192 (fp32 / bf16 moments): the ring-less direct state path, all shared memory to the operand ring
//   (gate_proj: T = 8192 direct 741-770 us vs ring 770-784; T = 4096 direct 469 vs ring 446; T = 2048 320 vs 274)
// Template arguments: <moments, mode, token chunk, operand stages, state stages, CTA group, chunk rows, chunk cols>.
enum : int { V_SMALL_T = 0, V_LARGE_T = 5, V_DIRECT = 30 };
int pick_variant(int maxT) { return maxT >= 8192 ? V_DIRECT : (maxT > 1024 ? V_LARGE_T : V_SMALL_T); }

// The direct state path moves 16 columns per thread with 32-byte accesses: every row must be a
// whole number of such vectors and every base 32-byte aligned; anything else takes the TMA ring.
bool direct_ok(const forge_problem_t *probs, int count) {
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = probs[i];
        const uintptr_t bits = reinterpret_cast<uintptr_t>(p.W) | reinterpret_cast<uintptr_t>(p.m) | reinterpret_cast<uintptr_t>(p.v);
        if (p.in % 16 != 0 || bits % 32 != 0) return false;
    }
    return true;
}

int max_tokens(const forge_problem_t *probs, int count) {
    int maxT = 0;
    for (int i = 0; i < count; ++i) maxT = probs[i].T > maxT ? probs[i].T : maxT;
    return maxT;
}

forge_status_t dispatch_fused(const forge_problem_t *probs, int count, int mdt, const AdamWScalars &hp,
                              const DeviceInfo &dev, cudaStream_t stream) {
    int variant = pick_variant(max_tokens(probs, count));
    if (variant == V_DIRECT && (!direct_ok(probs, count) || mdt > FORGE_MOMENT_BF16)) variant = V_LARGE_T;
#ifdef FORGE_PROFILING
    if (env_int("FORGE_CFG", -1) >= 0) {
        variant = env_int("FORGE_CFG", -1);
        switch (mdt) {
#include "profiling_variants.inc"
        default: break;
        }
    }
#endif
    switch (mdt) {
    case FORGE_MOMENT_FP32:
        // T > 1024: 128 KB operand ring; the 80 KB left for the state go further as 4 x 20 KB (32 x 64) than as 2 x 40 KB
        if (variant == V_DIRECT) return launch_fused<MDT_FP32, MODE_ADAMW, 64, 6, 0, 2, 64, 128>(probs, count, hp, dev, stream);
        if (variant == V_LARGE_T) return launch_fused<MDT_FP32, MODE_ADAMW, 64, 4, 4, 2, 32, 64>(probs, count, hp, dev, stream);
        // 64 x 128 chunks: 729 us / layer at the boost clock, 790-820 under the power cap; 128 x 64 chunks with a 48 KB
        // operand ring: 755 / 745 (profiles/r02_summary.md).  No geometry tried wins both; the caller says which clock
        // it expects (forge_set_tuning), the library does not guess.  Bit-identical.
        if (g_tuning.load(std::memory_order_relaxed) == FORGE_TUNE_SUSTAINED_CLOCK)
            return launch_fused<MDT_FP32, MODE_ADAMW, 32, 3, 2, 2, 128, 64>(probs, count, hp, dev, stream);
        return launch_fused<MDT_FP32, MODE_ADAMW, 32, 4, 2, 2, 64, 128>(probs, count, hp, dev, stream);
    case FORGE_MOMENT_BF16:
        if (variant == V_DIRECT) return launch_fused<MDT_BF16, MODE_ADAMW, 64, 6, 0, 2, 64, 64>(probs, count, hp, dev, stream);
        if (variant == V_LARGE_T) return launch_fused<MDT_BF16, MODE_ADAMW, 64, 4, 2, 2, 64, 64>(probs, count, hp, dev, stream);
        if (g_tuning.load(std::memory_order_relaxed) == FORGE_TUNE_SUSTAINED_CLOCK)      // 478 / 483 us against 457 / 498
            return launch_fused<MDT_BF16, MODE_ADAMW, 64, 4, 4, 2, 64, 64>(probs, count, hp, dev, stream);
        return launch_fused<MDT_BF16, MODE_ADAMW, 32, 4, 4, 2, 64, 64>(probs, count, hp, dev, stream);
    case FORGE_MOMENT_INT8:
        // resident-tile epilogue (P1S = 0: the four 128 x 64 chunks of a tile stay in the state ring through both passes, no
        // second read of the codes): 4 slots + 80 KB operand ring 428 us / layer against 440 for the streamed two-ring
        // variant <32, 5, 3, .., 64, 2> on the same box; 5 slots + 48 KB operand ring 451 (mainloop starved); sixteen
        // epilogue warps 487 (profiles/r02_summary.md).  The epilogue warps wait for G 5-14 % of the time (the T = 512
        // mainloop is bound by operand bytes in flight), so the ring takes every byte the SM has left: six 16 KB stages
        // next to the 128 KB tile (413 us against 422 with five; 3 x 32 KB: 417)
        if (variant == V_LARGE_T) return launch_fused<MDT_INT8, MODE_ADAMW, 64, 2, 2, 2, 128, 64>(probs, count, hp, dev, stream);
        return launch_fused<MDT_INT8, MODE_ADAMW, 32, 6, 4, 2, 128, 64, 64, 0>(probs, count, hp, dev, stream);
    case FORGE_MOMENT_FP8:
        // 8 B/element of state: the T = 512 mainloop needs operand bytes in flight more than the state ring needs slots
        // (the epilogue warps wait for G 10-12 % of the time): 4 x 32 KB of operands + 3 slots of 128 x 64 345 us against
        // 353 for 3 x 32 KB + 4 slots of 64 x 128; 5 x 32 KB + 2 slots 385; 16 KB stages 361-385 (profiles/r02_summary.md)
        return launch_fused<MDT_FP8, MODE_ADAMW, 64, 4, 3, 2, 128, 64>(probs, count, hp, dev, stream);
    default:
        return FORGE_ERR_BAD_DTYPE;
    }
}

// ---------------------------------------------------------------------------------------------
// the other coordinate-wise families (family_math.cuh): scalars in double from the ABI's floats
// ---------------------------------------------------------------------------------------------
int family_states(int family) {
    switch (family) {
    case FORGE_OPT_SGD: return 0;
    case FORGE_OPT_MOMENTUM: case FORGE_OPT_LION: case FORGE_OPT_RMSPROP: case FORGE_OPT_ADAGRAD: return 1;
    default: return 2;
    }
}

double nadam_mu(double beta1, int64_t t) { return beta1 * (1.0 - 0.5 * std::pow(0.96, static_cast<double>(t) * 4e-3)); }

FamilyScalars make_family(const forge_opt_desc_t &o) {
    FamilyScalars f;
    std::memset(&f, 0, sizeof(f));
    const double lr = o.lr, b1 = o.beta1, b2 = o.beta2, eps = o.eps, wd = o.wd, mu = o.momentum, t = static_cast<double>(o.step);
    f.decay = 1.0f;
    f.c2 = 1.0f;
    f.e1 = 1.0f;
    f.step = o.lr;
    switch (o.family) {
    case FORGE_OPT_SGD:
        f.cwd = o.wd;
        break;
    case FORGE_OPT_MOMENTUM:                       // buf = mu*buf + g' (buf = g' at step 1); d = buf or g' + mu*buf
        f.cwd = o.wd; f.has_m = 1; f.a1 = o.step == 1 ? 0.0f : o.momentum; f.a2 = 1.0f;
        f.c1 = o.nesterov ? o.momentum : 1.0f; f.c2 = o.nesterov ? 1.0f : 0.0f;
        break;
    case FORGE_OPT_LION:                           // n = sign(b1 m + (1-b1) g); m' = b2 m + (1-b2) g; decoupled decay
        f.has_m = 1; f.lion = 1; f.l1 = o.beta1; f.l2 = 1.0f - o.beta1; f.a1 = o.beta2; f.a2 = 1.0f - o.beta2;
        f.decay = static_cast<float>(1.0 - lr * wd);
        break;
    case FORGE_OPT_RMSPROP:                        // alpha is passed as beta2
        f.cwd = o.wd; f.v_mode = V_EMA; f.b1 = o.beta2; f.b2 = 1.0f - o.beta2; f.has_denom = 1; f.e2 = o.eps;
        break;
    case FORGE_OPT_ADAGRAD:
        f.cwd = o.wd; f.v_mode = V_EMA; f.b1 = 1.0f; f.b2 = 1.0f; f.has_denom = 1; f.e2 = o.eps;
        break;
    case FORGE_OPT_ADAMAX:                         // u = max(b2 u, |g'| + eps); w -= lr/(1-b1^t) m/u
        f.cwd = o.wd; f.has_m = 1; f.a1 = o.beta1; f.a2 = 1.0f - o.beta1; f.c1 = 1.0f; f.c2 = 0.0f;
        f.v_mode = V_MAX; f.b1 = o.beta2; f.e2 = o.eps; f.has_denom = 1;
        f.step = static_cast<float>(lr / (1.0 - std::pow(b1, t)));
        break;
    case FORGE_OPT_NADAM: {                        // torch.optim.NAdam: momentum_decay 4e-3, coupled decay
        double prod = 1.0;
        for (int64_t i = 1; i <= o.step; ++i) prod *= nadam_mu(b1, i);
        const double mu_t = nadam_mu(b1, o.step), mu_n = nadam_mu(b1, o.step + 1);
        f.cwd = o.wd; f.has_m = 1; f.a1 = o.beta1; f.a2 = 1.0f - o.beta1;
        f.v_mode = V_EMA; f.b1 = o.beta2; f.b2 = 1.0f - o.beta2; f.has_denom = 1;
        f.e1 = static_cast<float>(1.0 / std::sqrt(1.0 - std::pow(b2, t))); f.e2 = o.eps;
        f.c1 = static_cast<float>(lr * mu_n / (1.0 - prod * mu_n));
        f.c2 = static_cast<float>(lr * (1.0 - mu_t) / (1.0 - prod));
        f.step = 1.0f;
        break; }
    case FORGE_OPT_RADAM: {                        // torch.optim.RAdam, coupled decay
        const double bc1 = 1.0 - std::pow(b1, t), bc2 = 1.0 - std::pow(b2, t);
        const double rho_inf = 2.0 / (1.0 - b2) - 1.0, rho_t = rho_inf - 2.0 * t * std::pow(b2, t) / bc2;
        f.cwd = o.wd; f.has_m = 1; f.a1 = o.beta1; f.a2 = 1.0f - o.beta1; f.c1 = 1.0f; f.c2 = 0.0f;
        f.v_mode = V_EMA; f.b1 = o.beta2; f.b2 = 1.0f - o.beta2; f.e2 = o.eps;
        if (rho_t > 5.0) {
            const double rect = std::sqrt((rho_t - 4.0) * (rho_t - 2.0) * rho_inf / ((rho_inf - 4.0) * (rho_inf - 2.0) * rho_t));
            f.has_denom = 1;
            f.step = static_cast<float>(lr * std::sqrt(bc2) * rect / bc1);
        } else {
            f.step = static_cast<float>(lr / bc1);
        }
        break; }
    default: break;
    }
    (void)eps; (void)mu;
    f.kind = !f.has_m ? (f.v_mode == V_NONE ? FK_PLAIN : FK_V)
                      : (f.lion ? FK_LION
                                : (f.v_mode == V_NONE ? FK_M
                                                      : (f.v_mode == V_MAX ? FK_MV_MAX : (f.has_denom ? FK_MV : FK_MV_NODENOM))));
    return f;
}

// chunk geometry per state count: the ring is sized so that ~160 KB of state are resident
template <int MDT>
forge_status_t dispatch_family(const forge_problem_t *probs, int count, int nst, const FamilyScalars &fs,
                               const DeviceInfo &dev, cudaStream_t stream) {
    AdamWScalars hp;
    std::memset(&hp, 0, sizeof(hp));
    const bool big = max_tokens(probs, count) > 1024;
    if (nst == 0) {
        if (big) return launch_fused<MDT, MODE_FAMILY, 64, 4, 4, 2, 64, 128, 128, 2, 0>(probs, count, hp, dev, stream, &fs);
        // measured: 128 KB operand ring 229 us / layer, 64 KB 298 us (4 B/element of state: the mainloop is the long pole)
        return launch_fused<MDT, MODE_FAMILY, 64, 4, 6, 2, 64, 128, 128, 2, 0>(probs, count, hp, dev, stream, &fs);
    }
    if (nst == 1) {
        if (big) return launch_fused<MDT, MODE_FAMILY, 64, 4, 2, 2, 64, 128, 128, 2, 1>(probs, count, hp, dev, stream, &fs);
        // measured (momentum, fp32 / bf16 state): 32 x 128 x 4 slots 465 / 376 us, 64 x 64 x 4 483 / 396, 64 x 128 x 2 514 / 417;
        // 128 KB operand ring + 32 x 128 x 4 slots: momentum 439 us (fp32 state), 355 us (bf16); with a 64 KB operand ring 448 / 370
        return launch_fused<MDT, MODE_FAMILY, 64, 4, 4, 2, 32, 128, 128, 2, 1>(probs, count, hp, dev, stream, &fs);
    }
    if (big) return launch_fused<MDT, MODE_FAMILY, 64, 4, 2, 2, 64, 64, 128, 2, 2>(probs, count, hp, dev, stream, &fs);
    if (MDT == MDT_FP32) {      // two fp32 states: AdamW's byte count and AdamW's two instantiations
        if (g_tuning.load(std::memory_order_relaxed) == FORGE_TUNE_SUSTAINED_CLOCK)
            return launch_fused<MDT, MODE_FAMILY, 32, 3, 2, 2, 128, 64, 128, 2, 2>(probs, count, hp, dev, stream, &fs);
        return launch_fused<MDT, MODE_FAMILY, 32, 4, 2, 2, 64, 128, 128, 2, 2>(probs, count, hp, dev, stream, &fs);
    }
    return launch_fused<MDT, MODE_FAMILY, 32, 4, 4, 2, 64, 64, 128, 2, 2>(probs, count, hp, dev, stream, &fs);
}

// ---------------------------------------------------------------------------------------------
// dgrad launch (dgrad_kernel.cuh): dX_i = dY_i . W_i for <= kDgMaxProblems problems
// ---------------------------------------------------------------------------------------------
forge_status_t launch_dgrad(const forge_problem_t *probs, void *const *dX, int count, const DeviceInfo &dev,
                            cudaStream_t stream) {
    constexpr int kStages = 5;
    using Cfg = DgradCfg<kStages>;
    auto kernel = forge_dgrad_kernel<kStages>;
    static std::atomic<uint64_t> attr_done{0};
    const uint64_t dev_bit = 1ull << (dev.device & 63);
    if (!(attr_done.load(std::memory_order_acquire) & dev_bit)) {
        const cudaError_t ae = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
        if (ae != cudaSuccess) return cuda_fail(ae);
        attr_done.fetch_or(dev_bit, std::memory_order_release);
    }
    static_assert(sizeof(DgradParams) <= 32 * 1024 - 64, "kernel parameter space");
    DgradParams P;
    std::memset(&P, 0, sizeof(P));
    P.num_problems = count;
    int tiles = 0;
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = probs[i];
        DgradProblem &d = P.prob[i];
        bool ok = true;
        ok &= encode_2d(&d.map_dY, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p.dY, p.T, p.out, 64, DG_BM, CU_TENSOR_MAP_SWIZZLE_128B,
                        static_cast<uint64_t>(p.lddy));
        ok &= encode_2d(&d.map_W, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p.W, p.out, p.in, 64, DG_BK, CU_TENSOR_MAP_SWIZZLE_128B);
        ok &= encode_2d(&d.map_dX, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dX[i], p.T, p.in, 64, 32, CU_TENSOR_MAP_SWIZZLE_128B);
        if (!ok) return cuda_fail(cudaErrorInvalidValue);
        d.T = p.T; d.out = p.out; d.in = p.in;
        d.tiles_n = (p.in + DG_BN - 1) / DG_BN;
        d.tile_begin = tiles;
        tiles += ((p.T + 2 * DG_BM - 1) / (2 * DG_BM)) * d.tiles_n;
    }
    P.total_tiles = tiles;
    int pairs = std::min(dev.sm_count / 2, kDgMaxPairs);
    if (pairs > tiles) pairs = tiles;
    // longest-processing-time-first assignment of tiles (cost = depth `out`) to CTA pairs
    P.use_list = tiles <= kDgMaxTiles ? 1 : 0;
    if (P.use_list) {
        std::vector<std::pair<int, int>> by_depth;            // (depth, tile)
        by_depth.reserve(tiles);
        for (int i = 0; i < count; ++i) {
            const int n = (i + 1 < count ? P.prob[i + 1].tile_begin : tiles) - P.prob[i].tile_begin;
            for (int t = 0; t < n; ++t) by_depth.push_back({probs[i].out, P.prob[i].tile_begin + t});
        }
        std::stable_sort(by_depth.begin(), by_depth.end(), [](const std::pair<int, int> &a, const std::pair<int, int> &b) { return a.first > b.first; });
        std::vector<long long> load(pairs, 0);
        std::vector<std::vector<uint16_t>> mine(pairs);
        for (const auto &dt : by_depth) {
            int best = 0;
            for (int g = 1; g < pairs; ++g) if (load[g] < load[best]) best = g;
            load[best] += dt.first + 256;                        // + per-tile overhead (epilogue hand-over) in depth units
            mine[best].push_back(static_cast<uint16_t>(dt.second));
        }
        int o = 0;
        for (int g = 0; g < pairs; ++g) {
            P.pair_begin[g] = static_cast<uint16_t>(o);
            for (uint16_t t : mine[g]) P.order[o++] = t;
        }
        P.pair_begin[pairs] = static_cast<uint16_t>(o);
    }
    if (dev.dry) return FORGE_OK;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(pairs * 2));
    cfg.blockDim = dim3(kDgThreads);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, P);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1);
    g_last_kernel.store("forge_dgrad_kernel<5>");
    return FORGE_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// static device staging of forge_wgrad_adamw_host_noalloc (include/forge.h).  In host code the name below is only a
// host-side handle of the symbol, NOT a device address: the address is resolved per device with cudaGetSymbolAddress
// (that device current) the first time the entry point runs there, and only that pointer is handed to copies / kernels.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) uint8_t forge_noalloc_scratch[FORGE_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
uint8_t *g_noalloc_ptr[kNoallocMaxDevices] = {};

forge_status_t noalloc_scratch(uint8_t **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (dev < 0 || dev >= kNoallocMaxDevices) return FORGE_ERR_UNSUPPORTED_ARCH;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, forge_noalloc_scratch);
        if (e != cudaSuccess) return cuda_fail(e);
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return FORGE_ERR_ALIGNMENT;
        g_noalloc_ptr[dev] = static_cast<uint8_t *>(p);
    }
    *out = g_noalloc_ptr[dev];
    return FORGE_OK;
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

forge_status_t forge_wgrad_adamw_grouped(const forge_problem_t *problems, int32_t count, int64_t step, float lr,
                                         float beta1, float beta2, float eps, float wd,
                                         forge_moment_dtype_t moment_dtype, forge_stream_t stream) {
    if (!problems) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt < 0 || mdt > 3) return FORGE_ERR_BAD_DTYPE;
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    for (int i = 0; i < count; ++i) {
        s = validate_problem(problems[i], mdt);
        if (s != FORGE_OK) return s;
    }
    s = validate_disjoint(problems, count, mdt, moment_bytes(mdt));
    if (s != FORGE_OK) return s;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    const AdamWScalars hp = make_scalars(step, lr, beta1, beta2, eps, wd);
    return for_each_launch(count, dev, [&](int i, int n, const DeviceInfo &d) {
        return dispatch_fused(problems + i, n, mdt, hp, d, reinterpret_cast<cudaStream_t>(stream));
    });
}

forge_status_t forge_wgrad_adamw(const void *X, const void *dY, void *W, void *m, void *v, float *m_scale,
                                 float *v_scale, int32_t T, int32_t out, int32_t in, int64_t step, float lr,
                                 float beta1, float beta2, float eps, float wd,
                                 forge_moment_dtype_t moment_dtype, forge_stream_t stream) {
    forge_problem_t p;
    std::memset(&p, 0, sizeof(p));
    p.X = X; p.dY = dY; p.W = W; p.m = m; p.v = v; p.m_scale = m_scale; p.v_scale = v_scale;
    p.T = T; p.out = out; p.in = in;
    return forge_wgrad_adamw_grouped(&p, 1, step, lr, beta1, beta2, eps, wd, moment_dtype, stream);
}

forge_status_t forge_wgrad_step_grouped(const forge_problem_t *problems, int32_t count, const forge_opt_desc_t *opt,
                                        forge_moment_dtype_t state_dtype, forge_stream_t stream) {
    if (!problems || !opt) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    const int fam = static_cast<int>(opt->family);
    if (fam < FORGE_OPT_ADAMW || fam > FORGE_OPT_RADAM) return FORGE_ERR_BAD_HYPERPARAM;
    if (fam == FORGE_OPT_ADAMW)
        return forge_wgrad_adamw_grouped(problems, count, opt->step, opt->lr, opt->beta1, opt->beta2, opt->eps, opt->wd,
                                         state_dtype, stream);
    const int mdt = static_cast<int>(state_dtype);
    if (mdt != FORGE_MOMENT_FP32 && mdt != FORGE_MOMENT_BF16) return FORGE_ERR_BAD_DTYPE;   // int8 state: AdamW only
    forge_status_t s = validate_hp(opt->step, opt->lr, opt->beta1, opt->beta2, opt->eps, opt->wd);
    if (s != FORGE_OK) return s;
    if (!(opt->momentum >= 0.f && opt->momentum < 1.f)) return FORGE_ERR_BAD_HYPERPARAM;
    const int nst = family_states(fam);
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = problems[i];
        if (!p.X || !p.dY || !p.W) return FORGE_ERR_NULL_PTR;
        if ((nst >= 1) != (p.m != nullptr) || (nst >= 2) != (p.v != nullptr)) return FORGE_ERR_NULL_PTR;   // exactly the family's states
        if (p.m_scale || p.v_scale) return FORGE_ERR_BAD_DTYPE;
        s = validate_operands(p);
        if (s != FORGE_OK) return s;
        if (!aligned16(p.W) || !aligned16(p.m) || !aligned16(p.v)) return FORGE_ERR_ALIGNMENT;
    }
    s = validate_disjoint(problems, count, mdt, moment_bytes(mdt));
    if (s != FORGE_OK) return s;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    const FamilyScalars fs = make_family(*opt);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    return for_each_launch(count, dev, [&](int i, int n, const DeviceInfo &d) {
        return mdt == FORGE_MOMENT_FP32 ? dispatch_family<MDT_FP32>(problems + i, n, nst, fs, d, st)
                                        : dispatch_family<MDT_BF16>(problems + i, n, nst, fs, d, st);
    });
}

forge_status_t forge_wgrad_accumulate_grouped(const forge_problem_t *problems, int32_t count, float mu,
                                              forge_moment_dtype_t state_dtype, forge_stream_t stream) {
    if (!problems) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    const int mdt = static_cast<int>(state_dtype);
    if (mdt != FORGE_MOMENT_FP32 && mdt != FORGE_MOMENT_BF16) return FORGE_ERR_BAD_DTYPE;
    if (!std::isfinite(mu) || mu < 0.f) return FORGE_ERR_BAD_HYPERPARAM;
    int maxT = 0;
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = problems[i];
        if (!p.X || !p.dY || !p.m) return FORGE_ERR_NULL_PTR;
        if (p.W || p.v || p.m_scale || p.v_scale) return FORGE_ERR_BAD_DTYPE;      // B only: no weight is touched
        const forge_status_t so = validate_operands(p);
        if (so != FORGE_OK) return so;
        if (!aligned16(p.m)) return FORGE_ERR_ALIGNMENT;
        maxT = p.T > maxT ? p.T : maxT;
    }
    forge_status_t s = validate_disjoint(problems, count, mdt, moment_bytes(mdt));
    if (s != FORGE_OK) return s;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    AdamWScalars hp;
    std::memset(&hp, 0, sizeof(hp));
    FamilyScalars fs;
    std::memset(&fs, 0, sizeof(fs));
    fs.a1 = mu;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    return for_each_launch(count, dev, [&](int i, int n, const DeviceInfo &d) {
        const forge_problem_t *pp = problems + i;
        if (mdt == FORGE_MOMENT_FP32)
            return maxT > 1024 ? launch_fused<MDT_FP32, MODE_ACCUM, 64, 4, 2, 2, 64, 128, 128, 2, 1>(pp, n, hp, d, st, &fs)
                               : launch_fused<MDT_FP32, MODE_ACCUM, 64, 4, 4, 2, 32, 128, 128, 2, 1>(pp, n, hp, d, st, &fs);
        return maxT > 1024 ? launch_fused<MDT_BF16, MODE_ACCUM, 64, 4, 2, 2, 64, 128, 128, 2, 1>(pp, n, hp, d, st, &fs)
                           : launch_fused<MDT_BF16, MODE_ACCUM, 64, 4, 4, 2, 32, 128, 128, 2, 1>(pp, n, hp, d, st, &fs);
    });
}

forge_status_t forge_wgrad_adamw_sr_grouped(const forge_problem_t *problems, int32_t count, int64_t step, float lr,
                                           float beta1, float beta2, float eps, float wd,
                                           forge_moment_dtype_t moment_dtype, uint64_t seed, forge_stream_t stream) {
    if (!problems) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt != FORGE_MOMENT_FP32 && mdt != FORGE_MOMENT_BF16) return FORGE_ERR_BAD_DTYPE;
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    int maxT = 0;
    for (int i = 0; i < count; ++i) {
        s = validate_problem(problems[i], mdt);
        if (s != FORGE_OK) return s;
        maxT = problems[i].T > maxT ? problems[i].T : maxT;
    }
    s = validate_disjoint(problems, count, mdt, moment_bytes(mdt));
    if (s != FORGE_OK) return s;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    const AdamWScalars hp = make_scalars(step, lr, beta1, beta2, eps, wd);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const uint32_t st32 = static_cast<uint32_t>(step);
    return for_each_launch(count, dev, [&](int i, int n, const DeviceInfo &d) {    // the random stream of a problem is its index in the call
        const forge_problem_t *pp = problems + i;
        const uint32_t s0 = static_cast<uint32_t>(i);
        if (mdt == FORGE_MOMENT_FP32)
            return maxT > 1024 ? launch_fused<MDT_FP32, MODE_ADAMW_SR, 64, 4, 2, 2, 64, 64>(pp, n, hp, d, st, nullptr, seed, st32, s0)
                               : launch_fused<MDT_FP32, MODE_ADAMW_SR, 32, 4, 2, 2, 64, 128>(pp, n, hp, d, st, nullptr, seed, st32, s0);
        return maxT > 1024 ? launch_fused<MDT_BF16, MODE_ADAMW_SR, 64, 4, 2, 2, 64, 64>(pp, n, hp, d, st, nullptr, seed, st32, s0)
                           : launch_fused<MDT_BF16, MODE_ADAMW_SR, 32, 4, 4, 2, 64, 64>(pp, n, hp, d, st, nullptr, seed, st32, s0);
    });
}

forge_status_t forge_layer_backward_grouped(const forge_problem_t *problems, void *const *dX, int32_t count,
                                            int64_t step, float lr, float beta1, float beta2, float eps, float wd,
                                            forge_moment_dtype_t moment_dtype, forge_stream_t stream) {
    if (!problems || !dX) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt < 0 || mdt > 3) return FORGE_ERR_BAD_DTYPE;
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    for (int i = 0; i < count; ++i) {          // everything is validated before anything is enqueued
        s = validate_problem(problems[i], mdt);
        if (s != FORGE_OK) return s;
        if (!dX[i]) return FORGE_ERR_NULL_PTR;
        if (!aligned16(dX[i])) return FORGE_ERR_ALIGNMENT;
    }
    // dX may not overlap anything the call reads or writes
    std::vector<size_t> dx_bytes(count);
    for (int i = 0; i < count; ++i) dx_bytes[i] = static_cast<size_t>(problems[i].T) * problems[i].in * 2;
    s = validate_disjoint(problems, count, mdt, moment_bytes(mdt), dX, dx_bytes.data());
    if (s != FORGE_OK) return s;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const AdamWScalars hp = make_scalars(step, lr, beta1, beta2, eps, wd);
    // Everything is prepared before anything is enqueued: a dry pass over the dgrad launches and the fused launches
    // encodes every tensor map and sets every function attribute.
    DeviceInfo dry = dev;
    dry.dry = true;
    for (int i = 0; i < count; i += kDgMaxProblems) {
        s = launch_dgrad(problems + i, dX + i, std::min(count - i, kDgMaxProblems), dry, st);
        if (s != FORGE_OK) return s;
    }
    for (int i = 0; i < count; i += kMaxProblems) {
        s = dispatch_fused(problems + i, std::min(count - i, kMaxProblems), mdt, hp, dry, st);
        if (s != FORGE_OK) return s;
    }
    // 1. dX = dY . W from the PRE-update W (Alg. 1 line 1; 296 Remark 2): the hand-written tcgen05 dgrad
    for (int i = 0; i < count; i += kDgMaxProblems) {
        s = launch_dgrad(problems + i, dX + i, std::min(count - i, kDgMaxProblems), dev, st);
        if (s != FORGE_OK) return s;
    }
    // 2. the fused weight-gradient + AdamW step, stream-ordered after every dgrad launch that reads W
    for (int i = 0; i < count; i += kMaxProblems) {
        s = dispatch_fused(problems + i, std::min(count - i, kMaxProblems), mdt, hp, dev, st);
        if (s != FORGE_OK) return s;
    }
    return FORGE_OK;
}

forge_status_t forge_wgrad_store_g_grouped(const forge_problem_t *problems, int32_t count, forge_stream_t stream) {
    if (!problems) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    int maxT = 0;
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = problems[i];
        if (!p.X || !p.dY || !p.m) return FORGE_ERR_NULL_PTR;
        if (p.W || p.v || p.m_scale || p.v_scale) return FORGE_ERR_BAD_DTYPE;   // a gradient has no state besides G
        const forge_status_t so = validate_operands(p);
        if (so != FORGE_OK) return so;
        if (!aligned16(p.m)) return FORGE_ERR_ALIGNMENT;
        maxT = p.T > maxT ? p.T : maxT;
    }
    forge_status_t s = validate_disjoint(problems, count, FORGE_MOMENT_FP32, 4);
    if (s != FORGE_OK) return s;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    AdamWScalars hp;
    std::memset(&hp, 0, sizeof(hp));
    // The accumulator sums the tokens in ascending order 16 at a time whatever the token-chunk length and the CTA
    // grouping, so store-G + forge_adamw_from_g is bit-identical to the fused call of any instantiation
    const int variant = pick_variant(maxT);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    return for_each_launch(count, dev, [&](int i, int n, const DeviceInfo &d) {
        if (variant != V_SMALL_T) return launch_fused<MDT_FP32, MODE_STORE_G, 64, 4, 2, 2, 64, 64>(problems + i, n, hp, d, st);
        return launch_fused<MDT_FP32, MODE_STORE_G, 32, 4, 2, 2, 64, 128>(problems + i, n, hp, d, st);
    });
}

forge_status_t forge_wgrad_store_g(const void *X, const void *dY, float *G, int32_t T, int32_t out, int32_t in,
                                   forge_stream_t stream) {
    forge_problem_t p;
    std::memset(&p, 0, sizeof(p));
    p.X = X; p.dY = dY; p.m = G; p.T = T; p.out = out; p.in = in;
    return forge_wgrad_store_g_grouped(&p, 1, stream);
}

forge_status_t forge_adamw_from_g(const float *G, void *W, void *m, void *v, float *m_scale, float *v_scale,
                                  int32_t out, int32_t in, int64_t step, float lr, float beta1, float beta2,
                                  float eps, float wd, forge_moment_dtype_t moment_dtype, forge_stream_t stream) {
    if (!G) return FORGE_ERR_NULL_PTR;
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt == FORGE_MOMENT_FP8) return FORGE_ERR_BAD_DTYPE;   // the unfused twin covers fp32 / bf16 / int8
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    s = validate_state(W, m, v, m_scale, v_scale, out, in, mdt);
    if (s != FORGE_OK) return s;
    if (!aligned16(G)) return FORGE_ERR_ALIGNMENT;
    DeviceInfo dev;
    s = device_info(dev);
    if (s != FORGE_OK) return s;
    const AdamWScalars hp = make_scalars(step, lr, beta1, beta2, eps, wd);
    const size_t n = static_cast<size_t>(out) * static_cast<size_t>(in);
    const size_t groups = n / 8;
    const unsigned blocks = static_cast<unsigned>((groups + 255) / 256);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    uint16_t *Wp = static_cast<uint16_t *>(W);
    if (mdt == FORGE_MOMENT_FP32)
        forge_adamw_from_g_kernel<MDT_FP32><<<blocks, 256, 0, st>>>(G, Wp, m, v, m_scale, v_scale, n, hp);
    else if (mdt == FORGE_MOMENT_BF16)
        forge_adamw_from_g_kernel<MDT_BF16><<<blocks, 256, 0, st>>>(G, Wp, m, v, m_scale, v_scale, n, hp);
    else
        forge_adamw_from_g_kernel<MDT_INT8><<<blocks, 256, 0, st>>>(G, Wp, m, v, m_scale, v_scale, n, hp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(1);
    return FORGE_OK;
}

forge_status_t forge_wgrad_adamw_host(const void *X, const void *dY, void *W, void *m, void *v, float *m_scale,
                                      float *v_scale, int32_t T, int32_t out, int32_t in, int64_t step, float lr,
                                      float beta1, float beta2, float eps, float wd,
                                      forge_moment_dtype_t moment_dtype) {
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt < 0 || mdt > 2) return FORGE_ERR_BAD_DTYPE;
    forge_problem_t hp_;
    std::memset(&hp_, 0, sizeof(hp_));
    hp_.X = X; hp_.dY = dY; hp_.W = W; hp_.m = m; hp_.v = v; hp_.m_scale = m_scale; hp_.v_scale = v_scale;
    hp_.T = T; hp_.out = out; hp_.in = in;
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    s = validate_problem(hp_, mdt);
    if (s != FORGE_OK) return s;
    const size_t n = static_cast<size_t>(out) * in;
    const size_t mom = mdt == FORGE_MOMENT_FP32 ? 4 : (mdt == FORGE_MOMENT_BF16 ? 2 : 1);
    const size_t bX = static_cast<size_t>(T) * in * 2, bY = static_cast<size_t>(T) * out * 2, bW = n * 2,
                 bM = n * mom, bS = mdt == FORGE_MOMENT_INT8 ? n / FORGE_QBLOCK * 4 : 0;
    auto up = [](size_t b) { return (b + 255) / 256 * 256; };
    const size_t total = up(bX) + up(bY) + up(bW) + 2 * up(bM) + 2 * up(bS);
    uint8_t *d = nullptr;
    cudaError_t e = cudaMalloc(&d, total);
    if (e != cudaSuccess) return cuda_fail(e);
    uint8_t *dX = d, *dYp = dX + up(bX), *dW = dYp + up(bY), *dM = dW + up(bW), *dV = dM + up(bM),
            *dMs = dV + up(bM), *dVs = dMs + up(bS);
    cudaStream_t st = nullptr;
    auto fail = [&](cudaError_t err) { cudaFree(d); return cuda_fail(err); };
    if ((e = cudaMemcpyAsync(dX, X, bX, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpyAsync(dYp, dY, bY, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpyAsync(dW, W, bW, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpyAsync(dM, m, bM, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpyAsync(dV, v, bM, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
    if (bS) {
        if ((e = cudaMemcpyAsync(dMs, m_scale, bS, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
        if ((e = cudaMemcpyAsync(dVs, v_scale, bS, cudaMemcpyHostToDevice, st)) != cudaSuccess) return fail(e);
    }
    s = forge_wgrad_adamw(dX, dYp, dW, dM, dV, bS ? reinterpret_cast<float *>(dMs) : nullptr,
                          bS ? reinterpret_cast<float *>(dVs) : nullptr, T, out, in, step, lr, beta1, beta2, eps, wd,
                          moment_dtype, nullptr);
    if (s != FORGE_OK) { cudaFree(d); return s; }
    if ((e = cudaMemcpyAsync(W, dW, bW, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpyAsync(m, dM, bM, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpyAsync(v, dV, bM, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return fail(e);
    if (bS) {
        if ((e = cudaMemcpyAsync(m_scale, dMs, bS, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return fail(e);
        if ((e = cudaMemcpyAsync(v_scale, dVs, bS, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return fail(e);
    }
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return fail(e);
    cudaFree(d);
    return FORGE_OK;
}

forge_status_t forge_wgrad_adamw_host_noalloc(const void *X, const void *dY, void *W, void *m, void *v, float *m_scale,
                                              float *v_scale, int32_t T, int32_t out, int32_t in, int64_t step,
                                              float lr, float beta1, float beta2, float eps, float wd,
                                              forge_moment_dtype_t moment_dtype) {
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt < 0 || mdt > 2) return FORGE_ERR_BAD_DTYPE;
    forge_problem_t hp_;
    std::memset(&hp_, 0, sizeof(hp_));
    hp_.X = X; hp_.dY = dY; hp_.W = W; hp_.m = m; hp_.v = v; hp_.m_scale = m_scale; hp_.v_scale = v_scale;
    hp_.T = T; hp_.out = out; hp_.in = in;
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    s = validate_problem(hp_, mdt);
    if (s != FORGE_OK) return s;
    const size_t n = static_cast<size_t>(out) * in;
    const size_t mom = mdt == FORGE_MOMENT_FP32 ? 4 : (mdt == FORGE_MOMENT_BF16 ? 2 : 1);
    const size_t bX = static_cast<size_t>(T) * in * 2, bY = static_cast<size_t>(T) * out * 2, bW = n * 2,
                 bM = n * mom, bS = mdt == FORGE_MOMENT_INT8 ? n / FORGE_QBLOCK * 4 : 0;
    auto up = [](size_t b) { return (b + 255) / 256 * 256; };
    const size_t total = up(bX) + up(bY) + up(bW) + 2 * up(bM) + 2 * up(bS);
    if (total > static_cast<size_t>(FORGE_NOALLOC_SCRATCH_BYTES)) return FORGE_ERR_TOO_LARGE;   // before any CUDA call
    uint8_t *d = nullptr;
    s = noalloc_scratch(&d);
    if (s != FORGE_OK) return s;
    uint8_t *dX = d, *dYp = dX + up(bX), *dW = dYp + up(bY), *dM = dW + up(bW), *dV = dM + up(bM),
            *dMs = dV + up(bM), *dVs = dMs + up(bS);
    cudaStream_t st = nullptr;
    cudaError_t e;
    // every region the kernel reads is written here first: the previous call's bytes in the array never matter
    if ((e = cudaMemcpyAsync(dX, X, bX, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(dYp, dY, bY, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(dW, W, bW, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(dM, m, bM, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(dV, v, bM, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if (bS) {
        if ((e = cudaMemcpyAsync(dMs, m_scale, bS, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
        if ((e = cudaMemcpyAsync(dVs, v_scale, bS, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    }
    s = forge_wgrad_adamw(dX, dYp, dW, dM, dV, bS ? reinterpret_cast<float *>(dMs) : nullptr,
                          bS ? reinterpret_cast<float *>(dVs) : nullptr, T, out, in, step, lr, beta1, beta2, eps, wd,
                          moment_dtype, nullptr);
    if (s != FORGE_OK) return s;
    if ((e = cudaMemcpyAsync(W, dW, bW, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(m, dM, bM, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(v, dV, bM, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if (bS) {
        if ((e = cudaMemcpyAsync(m_scale, dMs, bS, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
        if ((e = cudaMemcpyAsync(v_scale, dVs, bS, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    }
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    return FORGE_OK;
}

forge_status_t forge_wgrad_adamw_grouped_host(const forge_problem_t *problems, int32_t count, int64_t step, float lr,
                                             float beta1, float beta2, float eps, float wd,
                                             forge_moment_dtype_t moment_dtype) {
    if (!problems) return FORGE_ERR_NULL_PTR;
    if (count < 1) return FORGE_ERR_BAD_SHAPE;
    const int mdt = static_cast<int>(moment_dtype);
    if (mdt < 0 || mdt > 3) return FORGE_ERR_BAD_DTYPE;
    forge_status_t s = validate_hp(step, lr, beta1, beta2, eps, wd);
    if (s != FORGE_OK) return s;
    for (int i = 0; i < count; ++i) {
        s = validate_problem(problems[i], mdt);
        if (s != FORGE_OK) return s;
        if (!dense_operands(problems[i])) return FORGE_ERR_BAD_SHAPE;   // host buffers are copied as dense blocks
    }
    const size_t mom = mdt == FORGE_MOMENT_FP32 ? 4 : (mdt == FORGE_MOMENT_BF16 ? 2 : 1);
    auto up = [](size_t b) { return (b + 255) / 256 * 256; };
    struct Sizes { size_t bX, bY, bW, bM, bS, off; };
    Sizes *sz = static_cast<Sizes *>(std::malloc(sizeof(Sizes) * count));
    forge_problem_t *dp = static_cast<forge_problem_t *>(std::malloc(sizeof(forge_problem_t) * count));
    if (!sz || !dp) { std::free(sz); std::free(dp); return cuda_fail(cudaErrorMemoryAllocation); }
    size_t total = 0;
    for (int i = 0; i < count; ++i) {
        const forge_problem_t &p = problems[i];
        const size_t n = static_cast<size_t>(p.out) * p.in;
        sz[i] = {static_cast<size_t>(p.T) * p.in * 2, static_cast<size_t>(p.T) * p.out * 2, n * 2, n * mom,
                 mdt == FORGE_MOMENT_INT8 ? n / FORGE_QBLOCK * 4 : (mdt == FORGE_MOMENT_FP8 ? 2 * sizeof(float) : 0), total};
        total += up(sz[i].bX) + up(sz[i].bY) + up(sz[i].bW) + 2 * up(sz[i].bM) + 2 * up(sz[i].bS);
    }
    // Row chunks: a problem's state goes up, is stepped and comes down in slices of about 64 MB (whole 256-row tile
    // rows, so the tiles -- and the bits -- are those of the unchunked call), each slice a sub-problem that reads a
    // column slice of the resident dY through lddy.  The download of slice c overlaps the upload of slice c + 1
    // (PCIe is full duplex); without the slicing the first upload and the last download (0.6 GB each for gate_proj)
    // overlap nothing.
    const bool i8 = mdt == FORGE_MOMENT_INT8, f8 = mdt == FORGE_MOMENT_FP8;
    const int slice_mb = env_int("FORGE_HOST_SLICE_MB", 64);   // FORGE_PROFILING build only; 0 = one slice per problem
    auto chunk_rows = [&](const forge_problem_t &p) {
        if (slice_mb <= 0) return static_cast<int>(p.out);
        const size_t row_bytes = static_cast<size_t>(p.in) * (2 + 2 * mom);
        size_t rows = ((static_cast<size_t>(slice_mb) << 20) / row_bytes + 255) / 256 * 256;
        if (rows < 256) rows = 256;
        return static_cast<int>(rows < static_cast<size_t>(p.out) ? rows : static_cast<size_t>(p.out));
    };
    int nev = 0;
    for (int i = 0; i < count; ++i) nev += 2 * ((problems[i].out + chunk_rows(problems[i]) - 1) / chunk_rows(problems[i]));
    uint8_t *d = nullptr;
    cudaStream_t s_in = nullptr, s_c = nullptr, s_out = nullptr;
    cudaEvent_t *ev = static_cast<cudaEvent_t *>(std::calloc(nev, sizeof(cudaEvent_t)));
    cudaError_t e = cudaMalloc(&d, total);
    auto cleanup = [&]() {
        if (ev) for (int i = 0; i < nev; ++i) if (ev[i]) cudaEventDestroy(ev[i]);
        if (s_in) cudaStreamDestroy(s_in);
        if (s_c) cudaStreamDestroy(s_c);
        if (s_out) cudaStreamDestroy(s_out);
        if (d) cudaFree(d);
        std::free(ev); std::free(sz); std::free(dp);
    };
    forge_status_t rc = FORGE_OK;
    if (!ev) e = cudaErrorMemoryAllocation;
#define FORGE_TRY(x) do { if (e == cudaSuccess) e = (x); } while (0)
    FORGE_TRY(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
    FORGE_TRY(cudaStreamCreateWithFlags(&s_c, cudaStreamNonBlocking));
    FORGE_TRY(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
    for (int i = 0; i < nev && ev; ++i) FORGE_TRY(cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming));
    // three-stage pipeline over the slices: copy-in (H2D), fused step, copy-out (D2H) on three streams;
    // largest problem first: the download that cannot overlap anything (the last one) is then the smallest
    int *order = static_cast<int *>(std::malloc(sizeof(int) * count));
    for (int i = 0; i < count && order; ++i) order[i] = i;
    for (int i = 0; i < count && order; ++i)
        for (int j = i + 1; j < count; ++j)
            if (sz[order[j]].bW > sz[order[i]].bW) { const int t = order[i]; order[i] = order[j]; order[j] = t; }
    int evi = 0;
    for (int k = 0; k < count && order && e == cudaSuccess && rc == FORGE_OK; ++k) {
        const int i = order[k];
        const forge_problem_t &p = problems[i];
        uint8_t *q = d + sz[i].off;
        forge_problem_t &g = dp[i];
        g = p;
        g.X = q; q += up(sz[i].bX);
        g.dY = q; q += up(sz[i].bY);
        g.W = q; q += up(sz[i].bW);
        g.m = q; q += up(sz[i].bM);
        g.v = q; q += up(sz[i].bM);
        g.m_scale = sz[i].bS ? reinterpret_cast<float *>(q) : nullptr; q += up(sz[i].bS);
        g.v_scale = sz[i].bS ? reinterpret_cast<float *>(q) : nullptr;
        // an operand shared with an earlier problem of the call (q / k / v read one X) is uploaded once
        const void *shared_x = nullptr, *shared_dy = nullptr;
        for (int kk = 0; kk < k; ++kk) {
            const forge_problem_t &q0 = problems[order[kk]];
            if (q0.X == p.X && q0.T == p.T && q0.in == p.in) shared_x = dp[order[kk]].X;
            if (q0.dY == p.dY && q0.T == p.T && q0.out == p.out) shared_dy = dp[order[kk]].dY;
        }
        if (shared_x) g.X = shared_x;
        else FORGE_TRY(cudaMemcpyAsync(const_cast<void *>(g.X), p.X, sz[i].bX, cudaMemcpyHostToDevice, s_in));
        if (shared_dy) g.dY = shared_dy;
        else FORGE_TRY(cudaMemcpyAsync(const_cast<void *>(g.dY), p.dY, sz[i].bY, cudaMemcpyHostToDevice, s_in));
        if (f8) {                                   // one {scale, amax} pair per tensor, shared by the slices
            FORGE_TRY(cudaMemcpyAsync(g.m_scale, p.m_scale, sz[i].bS, cudaMemcpyHostToDevice, s_in));
            FORGE_TRY(cudaMemcpyAsync(g.v_scale, p.v_scale, sz[i].bS, cudaMemcpyHostToDevice, s_in));
        }
        const int crow = chunk_rows(p);
        const size_t sblk = static_cast<size_t>(p.in) / FORGE_QBLOCK;     // int8: scales per row
        for (int r0 = 0; r0 < p.out && e == cudaSuccess && rc == FORGE_OK; r0 += crow, evi += 2) {
            const int rows = (p.out - r0) < crow ? (p.out - r0) : crow;
            const size_t e0 = static_cast<size_t>(r0) * p.in, n = static_cast<size_t>(rows) * p.in;
            forge_problem_t c = g;
            c.out = rows;
            c.ldx = 0;
            c.lddy = p.out;
            c.dY = static_cast<const uint8_t *>(g.dY) + static_cast<size_t>(r0) * 2;
            c.W = static_cast<uint8_t *>(g.W) + e0 * 2;
            c.m = static_cast<uint8_t *>(g.m) + e0 * mom;
            c.v = static_cast<uint8_t *>(g.v) + e0 * mom;
            if (i8) { c.m_scale = g.m_scale + r0 * sblk; c.v_scale = g.v_scale + r0 * sblk; }
            uint8_t *hW = static_cast<uint8_t *>(p.W) + e0 * 2, *hM = static_cast<uint8_t *>(p.m) + e0 * mom,
                    *hV = static_cast<uint8_t *>(p.v) + e0 * mom;
            FORGE_TRY(cudaMemcpyAsync(c.W, hW, n * 2, cudaMemcpyHostToDevice, s_in));
            FORGE_TRY(cudaMemcpyAsync(c.m, hM, n * mom, cudaMemcpyHostToDevice, s_in));
            FORGE_TRY(cudaMemcpyAsync(c.v, hV, n * mom, cudaMemcpyHostToDevice, s_in));
            if (i8) {
                FORGE_TRY(cudaMemcpyAsync(c.m_scale, p.m_scale + r0 * sblk, rows * sblk * 4, cudaMemcpyHostToDevice, s_in));
                FORGE_TRY(cudaMemcpyAsync(c.v_scale, p.v_scale + r0 * sblk, rows * sblk * 4, cudaMemcpyHostToDevice, s_in));
            }
            FORGE_TRY(cudaEventRecord(ev[evi], s_in));
            FORGE_TRY(cudaStreamWaitEvent(s_c, ev[evi], 0));
            if (e == cudaSuccess)
                rc = forge_wgrad_adamw_grouped(&c, 1, step, lr, beta1, beta2, eps, wd, moment_dtype, reinterpret_cast<forge_stream_t>(s_c));
            FORGE_TRY(cudaEventRecord(ev[evi + 1], s_c));
            FORGE_TRY(cudaStreamWaitEvent(s_out, ev[evi + 1], 0));
            FORGE_TRY(cudaMemcpyAsync(hW, c.W, n * 2, cudaMemcpyDeviceToHost, s_out));
            FORGE_TRY(cudaMemcpyAsync(hM, c.m, n * mom, cudaMemcpyDeviceToHost, s_out));
            FORGE_TRY(cudaMemcpyAsync(hV, c.v, n * mom, cudaMemcpyDeviceToHost, s_out));
            if (i8) {
                FORGE_TRY(cudaMemcpyAsync(p.m_scale + r0 * sblk, c.m_scale, rows * sblk * 4, cudaMemcpyDeviceToHost, s_out));
                FORGE_TRY(cudaMemcpyAsync(p.v_scale + r0 * sblk, c.v_scale, rows * sblk * 4, cudaMemcpyDeviceToHost, s_out));
            }
        }
        if (f8) {                                   // after the last slice's kernel: s_out already waits for it
            FORGE_TRY(cudaMemcpyAsync(p.m_scale, g.m_scale, sz[i].bS, cudaMemcpyDeviceToHost, s_out));
            FORGE_TRY(cudaMemcpyAsync(p.v_scale, g.v_scale, sz[i].bS, cudaMemcpyDeviceToHost, s_out));
        }
    }
    std::free(order);
    if (s_in) cudaStreamSynchronize(s_in);
    if (s_c) cudaStreamSynchronize(s_c);
    if (s_out) FORGE_TRY(cudaStreamSynchronize(s_out));
#undef FORGE_TRY
    cleanup();
    if (rc != FORGE_OK) return rc;
    return e == cudaSuccess ? FORGE_OK : cuda_fail(e);
}

forge_status_t forge_set_tuning(forge_tuning_t tuning) {
    if (tuning != FORGE_TUNE_BOOST_CLOCK && tuning != FORGE_TUNE_SUSTAINED_CLOCK) return FORGE_ERR_BAD_HYPERPARAM;
    g_tuning.store(static_cast<int>(tuning), std::memory_order_relaxed);
    return FORGE_OK;
}
forge_tuning_t forge_get_tuning(void) { return static_cast<forge_tuning_t>(g_tuning.load(std::memory_order_relaxed)); }

size_t forge_workspace_bytes(void) { return 0; }
uint64_t forge_launch_count(void) { return g_launches.load(); }
int forge_last_cuda_error(void) { return g_last_cuda_error.load(); }
const char *forge_last_kernel(void) { return g_last_kernel.load(); }
int forge_version(void) { return FORGE_VERSION; }

const char *forge_status_string(forge_status_t status) {
    switch (status) {
    case FORGE_OK: return "FORGE_OK";
    case FORGE_ERR_NULL_PTR: return "FORGE_ERR_NULL_PTR";
    case FORGE_ERR_BAD_SHAPE: return "FORGE_ERR_BAD_SHAPE";
    case FORGE_ERR_ALIGNMENT: return "FORGE_ERR_ALIGNMENT";
    case FORGE_ERR_BAD_HYPERPARAM: return "FORGE_ERR_BAD_HYPERPARAM";
    case FORGE_ERR_BAD_DTYPE: return "FORGE_ERR_BAD_DTYPE";
    case FORGE_ERR_UNSUPPORTED_ARCH: return "FORGE_ERR_UNSUPPORTED_ARCH";
    case FORGE_ERR_CUDA: return "FORGE_ERR_CUDA";
    case FORGE_ERR_TOO_LARGE: return "FORGE_ERR_TOO_LARGE";
    }
    return "FORGE_ERR_UNKNOWN";
}

}  // extern "C"
