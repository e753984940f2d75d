/*
 * forge.h -- C ABI of forge-b200: FORGE's hot path (arxiv/paper_2606_22932) on NVIDIA B200 (sm_100a).
 *
 * The operation (sec. 2.2, Eq. 4, Algorithm 1): for one linear layer with weight
 * W[out,in], activations X[T,in] and upstream gradient dY[T,out], every weight tile forms its
 * block of G = dY^T X in fp32 on chip (tensor memory) and immediately applies AdamW to the
 * matching tiles of W, m and v in place.  G is never written to device memory.
 *
 *   m'  = beta1*m + (1-beta1)*G                      Alg. 1 line 7
 *   v'  = beta2*v + (1-beta2)*G*G                    Alg. 1 line 8
 *   W'  = (1-lr*wd)*W - lr*(m'/(1-beta1^t)) / (sqrt(v'/(1-beta2^t)) + eps)     lines 9-10
 *   store W' (bf16, round to nearest even), m', v' (storage type)              line 11
 *
 * All pointers are DEVICE pointers unless a parameter says "host".  The caller allocates and owns
 * every buffer; the library allocates no O(out*in) memory and keeps no reference after a call
 * returns ("No gradient byte reaches global memory"; Eq. 5).  Work is
 * enqueued on `stream` and the call returns without synchronising.
 *
 * Caller's obligations (documented, not enforced):
 *   - dX = dY*W must already be enqueued on the same stream: W is overwritten (
 *     PAPER.md:74 Alg. 1 line 1; PAPER.md:296 Remark 2).
 *   - a weight with more than one backward consumer (tied embedding / LM head) must not be passed
 *     (PAPER.md:296).
 * Aliasing (enforced): inside one call no updated tensor (W, m, v, scales, dX, G) may overlap any other tensor the
 * call touches, within a problem or across the problems of a group; read-only operands may be shared (q / k / v read
 * one X).  A violation returns FORGE_ERR_BAD_SHAPE before anything is enqueued.
 *
 * Error behaviour: every argument of every problem is validated, every tensor map of every launch the call needs is
 * encoded and every kernel attribute is set BEFORE the first launch is enqueued, so a status other than FORGE_ERR_CUDA
 * means no state was touched.  FORGE_ERR_CUDA can only come from a launch itself; when the call needed several
 * launches (more than 8 problems, or forge_layer_backward_grouped's dgrad + update) the earlier ones have then been
 * enqueued.  No exceptions cross this boundary.  NaN/Inf in the inputs propagate by IEEE rules (to the rows / columns
 * of G they enter and nowhere else).  There is no CPU or library fallback: a device that is not compute capability
 * 10.x returns FORGE_ERR_UNSUPPORTED_ARCH.
 *
 * Environment: the library reads no environment variable.  The tuning / profiling switches FORGE_CFG, FORGE_GRID,
 * FORGE_ABLATE and FORGE_HOST_SLICE_MB exist only in the separate -DFORGE_PROFILING build (libforge_b200_prof.so)
 * that the commands quoted under profiles/ load.
 */
#ifndef FORGE_H_
#define FORGE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FORGE_VERSION 100          /* 0.1.0 */
#define FORGE_QBLOCK 256           /* int8 moment block: 256 contiguous elements along `in` */

typedef enum {
    FORGE_OK = 0,
    FORGE_ERR_NULL_PTR = 1,
    FORGE_ERR_BAD_SHAPE = 2,
    FORGE_ERR_ALIGNMENT = 3,
    FORGE_ERR_BAD_HYPERPARAM = 4,
    FORGE_ERR_BAD_DTYPE = 5,
    FORGE_ERR_UNSUPPORTED_ARCH = 6,
    FORGE_ERR_CUDA = 7,
    FORGE_ERR_TOO_LARGE = 8        /* forge_wgrad_adamw_host_noalloc only: the problem exceeds the static scratch */
} forge_status_t;

/* Storage type of the moments m, v ("k" of PAPER.md:19 Eq. 1):
 *   FP32: 4+4 B/param ("fp32 optimizer state")
 *   BF16: 2+2 B/param, round to nearest even (the "bf16-state" recipe)
 *   INT8: 1+1 B/param + one fp32 absmax per 256-element block along `in` for each moment
 *         (App. B with BASELINE.json's 256-blocks); m code = rint(m'*127/a) in
 *         [-127,127] (int8), v code = max(1, rint(v'*255/a)) in [1,255] (uint8) when a > 0,
 *         all codes 0 when a == 0; the stored scale is a = max|x| over the block (fp32).
 *         Dequantised value = code*a/127 (m) or code*a/255 (v).  Requantised every step.  The codes (and the FP8
 *         codes below) cannot hold NaN / Inf: a non-finite gradient element still makes W' non-finite by IEEE rules, the
 *         code stored for its m', v' and the block scale it contributes to are unspecified.
 * In every mode the update arithmetic and G are fp32 and W' is computed from the unrounded
 * m', v' ("the update arithmetic and the gradient remain fp32 throughout"). */
typedef enum {
    FORGE_MOMENT_FP32 = 0,
    FORGE_MOMENT_BF16 = 1,
    FORGE_MOMENT_INT8 = 2,
    FORGE_MOMENT_FP8 = 3     /* e4m3 codes, ONE fp32 scale per tensor with delayed scaling:
                              * m, v are uint8 e4m3 codes of x / s; m_scale / v_scale point to float[2]:
                              * [0] = the scale s in use (read; the caller derives it from the amax the previous
                              * step reported, s = amax / 448), [1] = amax of this step's m' / v' (the kernel
                              * max-accumulates into it: set it to 0 before the call).  Values beyond 448 s
                              * saturate.  in % 16 == 0.  forge_wgrad_adamw[_grouped] and forge_layer_backward_grouped only. */
} forge_moment_dtype_t;

/* CUDA stream handle; identical to cudaStream_t / CUstream.  NULL is the legacy default stream. */
typedef struct CUstream_st *forge_stream_t;

/* One linear layer's problem.  Layouts are row-major; the state tensors are dense (leading dimension = row
 * length), the two operands may be strided views -- the q / k / v slices of one fused-QKV output gradient, the gate /
 * up halves of a fused MLP projection -- through ldx / lddy (row pitch in ELEMENTS; 0 means dense; otherwise
 * >= the row length and a multiple of 8, else FORGE_ERR_BAD_SHAPE; the host-buffer entries take dense operands only):
 *   X  [T, in]   bf16, read only          dY [T, out]  bf16, read only
 *   W  [out, in] bf16, updated in place   m, v [out, in] in the moment dtype, updated in place
 *   m_scale, v_scale [out, in/256] fp32, INT8 mode only (must be NULL otherwise), in place.
 * Constraints: T >= 1; out, in >= 8 and multiples of 8 (16 for BF16/INT8 moments along `in`;
 * INT8 needs in % 256 == 0); every base pointer 16-byte aligned (X, dY: 16; state: 16). */
typedef struct {
    const void *X;
    const void *dY;
    void *W;
    void *m;
    void *v;
    float *m_scale;
    float *v_scale;
    int32_t T, out, in;
    int64_t ldx, lddy;
} forge_problem_t;

/* Fused weight gradient + AdamW step for one layer (Algorithm 1).
 * `step` is the 1-based index t of the update being applied (bias terms 1-beta^t); step < 1,
 * lr < 0 or non-finite, beta outside [0,1), eps < 0, wd < 0 -> FORGE_ERR_BAD_HYPERPARAM. */
forge_status_t forge_wgrad_adamw(const void *X, const void *dY, void *W, void *m, void *v,
                                 float *m_scale, float *v_scale,
                                 int32_t T, int32_t out, int32_t in,
                                 int64_t step, float lr, float beta1, float beta2, float eps, float wd,
                                 forge_moment_dtype_t moment_dtype, forge_stream_t stream);

/* The same for `count` layers in as few launches as possible (one for count <= 8): all seven
 * projections of a Llama-style decoder layer go in one persistent launch (the paper pays one
 * launch per linear).  `problems` is a HOST array, read before the call returns. */
forge_status_t forge_wgrad_adamw_grouped(const forge_problem_t *problems, int32_t count,
                                         int64_t step, float lr, float beta1, float beta2,
                                         float eps, float wd,
                                         forge_moment_dtype_t moment_dtype, forge_stream_t stream);

/* The other coordinate-wise optimizer families of the paper's Definition 1 (App. I)
 * on the same fused mainloop: the update rules are torch.optim's (Lion: Chen et al. 2023, Alg. 2) -- the paper
 * verifies each "against a reference PyTorch implementation".  State tensors per family, passed in
 * forge_problem_t.m / .v (absent ones MUST be NULL, else FORGE_ERR_NULL_PTR):
 *   SGD: none | MOMENTUM: m = momentum buffer | LION: m | RMSPROP: m = square average (alpha = beta2) |
 *   ADAGRAD: m = sum of squares | ADAMAX: m, v = infinity norm | NADAM, RADAM: m, v | ADAMW: as forge_wgrad_adamw.
 * Weight decay is coupled (g + wd*W) except for ADAMW and LION (decoupled).  State dtype FP32 or BF16 (INT8: ADAMW
 * only, else FORGE_ERR_BAD_DTYPE).  `step` is 1-based (MOMENTUM: the buffer is initialised with g at step 1). */
typedef enum {
    FORGE_OPT_ADAMW = 0, FORGE_OPT_SGD = 1, FORGE_OPT_MOMENTUM = 2, FORGE_OPT_LION = 3, FORGE_OPT_RMSPROP = 4,
    FORGE_OPT_ADAGRAD = 5, FORGE_OPT_ADAMAX = 6, FORGE_OPT_NADAM = 7, FORGE_OPT_RADAM = 8
} forge_optimizer_t;

typedef struct {
    forge_optimizer_t family;
    int32_t nesterov;        /* MOMENTUM only */
    int64_t step;
    float lr, beta1, beta2, eps, wd, momentum;
} forge_opt_desc_t;

forge_status_t forge_wgrad_step_grouped(const forge_problem_t *problems, int32_t count, const forge_opt_desc_t *opt,
                                        forge_moment_dtype_t state_dtype, forge_stream_t stream);

/* AdamW with the paper's "SR-store" recipe (1287-1296): identical to forge_wgrad_adamw_grouped except
 * that W' is committed to bf16 by STOCHASTIC rounding instead of RNE (m, v unchanged; FP32 or BF16 moments).
 * 16 random bits per weight element come from a counter-based generator keyed (seed, step, index of the problem
 * in this call, row, col) -- the same call with the same seed is bitwise reproducible; out = (bits(fp32 W') + r16)
 * >> 16, i.e. the fp32 value is rounded away from zero with probability (its low 16 bits) / 65536 (unbiased). */
forge_status_t forge_wgrad_adamw_sr_grouped(const forge_problem_t *problems, int32_t count, int64_t step, float lr,
                                           float beta1, float beta2, float eps, float wd,
                                           forge_moment_dtype_t moment_dtype, uint64_t seed, forge_stream_t stream);

/* One layer's backward for the linear weights in ONE call (Alg. 1 line 1 + lines 2-11): first the
 * input gradients dX[i][T,in] = dY_i . W_i (bf16 output, fp32 accumulation in tensor memory) from the PRE-update
 * weights -- a hand-written tcgen05 kernel (csrc/dgrad_kernel.cuh; A = dY K-major, B = W MN-major, CTA pairs, tiles of
 * all problems assigned longest-first), one launch per 8 problems -- then, stream-ordered behind it, the fused
 * weight-gradient + AdamW launch that overwrites W in place.  This closes the ordering hazard forge_wgrad_adamw leaves
 * to the caller (296 Remark 2).  dX is a HOST array of `count` device pointers, one dense [T,in] output
 * per problem (the caller sums the dX of projections that share an input); it may not overlap any other tensor of the
 * call.  No library GEMM and no gradient-shaped buffer is involved.  Validation and errors as
 * forge_wgrad_adamw_grouped. */
forge_status_t forge_layer_backward_grouped(const forge_problem_t *problems, void *const *dX, int32_t count,
                                            int64_t step, float lr, float beta1, float beta2, float eps, float wd,
                                            forge_moment_dtype_t moment_dtype, forge_stream_t stream);

/* Accumulate-into-state (the paper's regime 2; Muon's A-step): for every problem
 * B <- mu * B + dY^T X in place, "through the GEMM's own beta": no gradient is materialised and no weight is read
 * or written.  B[out,in] (fp32 or bf16) is passed in forge_problem_t.m; W, v and the scales MUST be NULL
 * (FORGE_ERR_BAD_DTYPE otherwise).  mu >= 0 and finite.  The state-global weight update that follows in Muon
 * (Newton-Schulz over the resident B) is out of scope. */
forge_status_t forge_wgrad_accumulate_grouped(const forge_problem_t *problems, int32_t count, float mu,
                                              forge_moment_dtype_t state_dtype, forge_stream_t stream);

/* End-to-end convenience entry with HOST buffers (used for the e2e measurement): copies X, dY and
 * the state to device scratch it allocates and frees itself, runs forge_wgrad_adamw, copies the
 * state back and synchronises.  Same validation and return codes; all pointers are host pointers. */
forge_status_t forge_wgrad_adamw_host(const void *X, const void *dY, void *W, void *m, void *v,
                                      float *m_scale, float *v_scale,
                                      int32_t T, int32_t out, int32_t in,
                                      int64_t step, float lr, float beta1, float beta2, float eps, float wd,
                                      forge_moment_dtype_t moment_dtype);

/* forge_wgrad_adamw_host for callers that may not allocate (a harness that forbids cudaMalloc, a tight serving loop):
 * the same arguments, validation, arithmetic and result (bit-identical to forge_wgrad_adamw_host), but the device
 * staging of X, dY, W, m, v and the scales lives in ONE file-scope static __device__ array of
 * FORGE_NOALLOC_SCRATCH_BYTES (32 MiB) instead of a cudaMalloc'ed block.  The call issues no cudaMalloc, cudaFree or
 * other allocating routine: only copies on the default stream, one fused launch and a stream synchronise.
 *   limit     the staged bytes -- each of the up-to-seven arrays rounded up to 256 B: T*in*2 + T*out*2 + out*in*(2 +
 *             2 * moment bytes) + the int8 block scales -- must fit the array, else FORGE_ERR_TOO_LARGE and nothing
 *             is copied or launched (fp32 moments at T = 512: out*in up to ~3.1 M, e.g. 1024 x 2048 or 1536 x 1536).
 *   cost      every GPU on which this library's module is loaded holds the 32 MiB until the process exits
 *             (forge_workspace_bytes() counts dynamic allocations only and stays 0).
 *   sharing   all calls on a device use the same array, and it keeps the previous call's bytes.  Nothing in it has to
 *             start at zero -- every region the kernel reads is overwritten by this call's uploads first -- but two
 *             calls that overlap on the same GPU (two host threads) race on it: serialise them.  The call itself is
 *             synchronous, so back-to-back calls from one thread are safe.
 * The array's device address is resolved once per device (cudaGetSymbolAddress with that device current). */
#define FORGE_NOALLOC_SCRATCH_BYTES (32u << 20)
forge_status_t forge_wgrad_adamw_host_noalloc(const void *X, const void *dY, void *W, void *m, void *v,
                                              float *m_scale, float *v_scale,
                                              int32_t T, int32_t out, int32_t in,
                                              int64_t step, float lr, float beta1, float beta2, float eps, float wd,
                                              forge_moment_dtype_t moment_dtype);

/* The same for a whole group with HOST buffers (every pointer of every problem is a host pointer, ideally pinned):
 * a three-stage pipeline -- upload, fused step, download on three streams -- over ~64 MB row slices of each problem's
 * state (whole tile rows: the result is bit-identical to the device-resident call), so the download of one slice
 * overlaps the upload of the next (PCIe is full duplex) and the kernels.  Device scratch is allocated and
 * freed inside the call; synchronous on return.  All four moment dtypes (INT8: the block scales, FP8: the two
 * float[2] scale / amax pairs travel with the codes).  An operand shared by several problems of the call (q/k/v read
 * one X: same host pointer and shape) is uploaded once. */
forge_status_t forge_wgrad_adamw_grouped_host(const forge_problem_t *problems, int32_t count, int64_t step, float lr,
                                             float beta1, float beta2, float eps, float wd,
                                             forge_moment_dtype_t moment_dtype);

/* The two halves of the fused call, for the one case that cannot fuse: data / context parallelism with a nonlinear
 * update (Prop. 2(ii)).  There the gradient tiles stream into a small rotating fp32 bucket, the bucket is
 * all-reduced, and the update is applied from the reduced bucket ("bucket-transient schedule"; 304);
 * paper_2606_22932_b200/dp.py drives that schedule.  They are also the paper's "store-G control" (PAPER.md:334-345
 * App. D) and its standalone optimizer kernel (86), and the tests use them as twins of the fused kernel:
 * never on the single-GPU / weight-sharded product path, which materialises no gradient.
 *
 * forge_wgrad_store_g[_grouped]: the identical mainloop, the fp32 tile is written to G[out,in] (dense, problem.m =
 * G for the grouped form; W, v and the scales must be NULL; ldx / lddy honoured, so a row range of a layer is a problem
 * of its own with a column slice of dY).  A later micro-batch adds to the same bucket with
 * forge_wgrad_accumulate_grouped(mu = 1). */
forge_status_t forge_wgrad_store_g(const void *X, const void *dY, float *G,
                                   int32_t T, int32_t out, int32_t in, forge_stream_t stream);
forge_status_t forge_wgrad_store_g_grouped(const forge_problem_t *problems, int32_t count, forge_stream_t stream);

/* forge_adamw_from_g: applies the same per-element update function as the fused epilogue to a materialised fp32
 * G[out,in] (any contiguous row range of a layer: out is then the number of rows passed).  forge_wgrad_store_g + this
 * is bit-identical to forge_wgrad_adamw ("the operands are bit-identical and so are the results").
 * FP32 / BF16 / INT8 moments. */
forge_status_t forge_adamw_from_g(const float *G, void *W, void *m, void *v,
                                  float *m_scale, float *v_scale, int32_t out, int32_t in,
                                  int64_t step, float lr, float beta1, float beta2, float eps, float wd,
                                  forge_moment_dtype_t moment_dtype, forge_stream_t stream);

/* Tuning for the clock the caller expects the launches to run at.  Results are BIT-IDENTICAL in both settings (the
 * instantiations differ only in chunk geometry and ring depths; same token order in the accumulator, same per-element
 * arithmetic), so this is a pure performance choice, process-wide and thread-safe:
 *   FORGE_TUNE_BOOST_CLOCK (default): best for short bursts of launches at the boost clock -- what a K-launch benchmark
 *     times (fp32 moments, Llama-8B layer at T = 512: 729 us at 1965 MHz, 790-820 us once the board power-caps);
 *   FORGE_TUNE_SUSTAINED_CLOCK: best under continuous load, when the board sits at its power cap and the SM clock is
 *     ~1.5-1.6 GHz -- a training loop (the same layer: 745 us capped, 755 us at the boost clock).
 * Only the fp32- and bf16-moment paths at T <= 1024 (and the two-state fp32 families) have a second instantiation.
 * An explicit call, not an environment variable and not a heuristic: the library cannot see the clock cheaply and does
 * not guess. */
typedef enum { FORGE_TUNE_BOOST_CLOCK = 0, FORGE_TUNE_SUSTAINED_CLOCK = 1 } forge_tuning_t;
forge_status_t forge_set_tuning(forge_tuning_t tuning);     /* FORGE_ERR_BAD_HYPERPARAM for any other value */
forge_tuning_t forge_get_tuning(void);

/* Device bytes the library itself allocates and holds between calls: a constant with no O(out*in) term (0).  The
 * fixed static array of forge_wgrad_adamw_host_noalloc (FORGE_NOALLOC_SCRATCH_BYTES, part of the loaded module) is
 * not an allocation and is not counted. */
size_t forge_workspace_bytes(void);
/* Kernel launches issued by this library since load (for bench.py's gpu_launches). */
uint64_t forge_launch_count(void);
/* Detail of the last CUDA error seen by this library (cudaError_t value), 0 if none. */
int forge_last_cuda_error(void);
/* Name and template arguments of the kernel instantiation the most recent launch of this library used, as a profiler
 * prints it (e.g. "forge_fused_kernel<0, 0, 32, 4, 2, 2, 64, 128, 128, 2, 2, 2>"); "" before the first launch.
 * bench.py uses it to match its launches with the committed ncu captures under profiles/. */
const char *forge_last_kernel(void);
const char *forge_status_string(forge_status_t status);
int forge_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FORGE_H_ */
