/* vla_ternary.h -- C ABI of libvlaternary.so (sm_100a only).
 *
 * The ternary-weight linear layer of arxiv/paper_2606_08094 ("vla.cpp"), Section III-D, Eq. 4
 * (PAPER.md lines 71-82):
 *
 *     alpha_m = max(||x_m||_inf, 1e-5) / 127
 *     a_mj    = clip( round( x_mj / alpha_m ) )            int8, round-half-to-even
 *     y_mn    = alpha_m * beta_g(n) * sum_j a_mj q_nj      q in {-1,0,+1}, int32 accumulation
 *
 * with the weights "packed four two-bit codes per byte" and the result written
 * as fp32 or as bf16 with round-to-nearest-even.
 *
 * Conventions (all entry points):
 *  - Every pointer is a DEVICE pointer owned by the caller unless the argument says "host".
 *    The library allocates nothing persistent and creates no streams.
 *  - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = default stream)
 *    and capturable in a CUDA graph, except vla_ternary_pack, which synchronises the stream.
 *  - Layouts: W logical [N,K] (row n = output channel, K contiguous); X [M,K] row-major;
 *    Y [M,N] row-major.
 *  - Shapes: M >= 1; K % 128 == 0; N % 128 == 0; K <= 65536 (else VLA_ERR_SHAPE; the decode scales the weights by 64,
 *    and 64 * 127 * K < 2^31 holds up to K = 264 000).
 *  - One device per call: every call works on the CURRENT device (cudaSetDevice); nothing is cached across devices.
 *  - Every pointer must be 16-byte aligned (VLA_ERR_ALIGN).
 *  - Inputs must be finite; NaN/Inf are not checked (result unspecified, memory-safe).
 *  - Arguments are validated on the host before any launch.  A non-zero status leaves the
 *    outputs unspecified but in bounds.  No exceptions cross the ABI.  There is no CPU fallback:
 *    on a device that is not compute capability 10.x the compute calls return VLA_ERR_ARCH.
 */
#ifndef VLA_TERNARY_H
#define VLA_TERNARY_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    VLA_OK = 0,
    VLA_ERR_NULL = 1,       /* a required pointer is NULL */
    VLA_ERR_SHAPE = 2,      /* M/N/K outside the supported set, or not supported by the forced path */
    VLA_ERR_ALIGN = 3,      /* a pointer is not 16-byte aligned */
    VLA_ERR_VALUE = 4,      /* vla_ternary_pack: an element outside {-1,0,+1} */
    VLA_ERR_DTYPE = 5,      /* unknown vla_dtype / vla_path value */
    VLA_ERR_WORKSPACE = 6,  /* workspace NULL or smaller than vla_ternary_workspace_bytes */
    VLA_ERR_ARCH = 7,       /* current device is not sm_100 */
    VLA_ERR_CUDA = 8        /* a CUDA runtime/driver call failed (launch error, etc.) */
} vla_status;

typedef enum {
    VLA_F32 = 0,            /* y fp32 */
    VLA_BF16 = 1,           /* y bf16, round-to-nearest-even of the fp32 value */
    VLA_I32 = 2             /* raw int32 accumulators sum_j a_mj q_nj, no scaling (parity/debug) */
} vla_dtype;

typedef enum {
    VLA_PATH_AUTO = 0,      /* library chooses by M, and by (N,K) for 16 < M <= 32 (table in DESIGN.md 6d, measured) */
    VLA_PATH_SMALL_ALU = 1, /* in-register decode + dp4a on the integer ALUs; M <= 16 (M = 17: VLA_ERR_SHAPE) */
    VLA_PATH_SMALL_TC = 2,  /* in-register decode + warp-level int8 MMA; M <= 32 (M = 33: VLA_ERR_SHAPE) */
    VLA_PATH_LARGE = 3      /* TMA -> decode warps -> tcgen05.mma kind::i8 -> TMEM; any M */
} vla_path;

/* Bytes of the packed form of an [N,K] ternary tensor: exactly N*K/4 (four 2-bit codes per byte,
 * PAPER.md line 73; no padding at supported shapes).  0 if the shape is not supported. */
size_t vla_ternary_packed_bytes(int N, int K);

/* Bytes of scratch vla_ternary_gemm / vla_ternary_linear need for (M,N,K,path); a multiple of 256.
 * vla_ternary_linear uses it for the quantised activations when xq_opt / x_scale_opt are NULL. */
size_t vla_ternary_workspace_bytes(int M, int N, int K, vla_path path);

/* Weight packer (offline, once per tensor).
 *   w            [N,K] int8, every element in {-1,0,+1}
 *   packed       packed_bytes >= vla_ternary_packed_bytes(N,K); layout is private to the library
 *                (tile-permuted 2-bit two's-complement codes), defined only by pack/unpack
 * SYNCHRONISES `stream`.  Returns VLA_ERR_VALUE if any element is outside {-1,0,+1}
 * (packed is then unspecified), VLA_ERR_WORKSPACE if packed_bytes is too small. */
vla_status vla_ternary_pack(const int8_t* w, int N, int K, void* packed, size_t packed_bytes, void* stream);

/* Inverse of vla_ternary_pack: w[N,K] int8.  unpack(pack(W)) == W. */
vla_status vla_ternary_unpack(const void* packed, int N, int K, int8_t* w, void* stream);

/* Activation quantiser, Eq. 4 lines 1-2, per row m:
 *   alpha_m = fmaxf(absmax_m, 1e-5f) / 127.0f          (fp32 division, round-to-nearest)
 *   a_mj    = clamp(rint(x_mj / alpha_m), -127, 127)    (fp32 division, round-half-to-even)
 *   x_bf16  [M,K] bf16          xq [M,K] int8          x_scale [M] fp32 (= alpha_m) */
vla_status vla_act_quant(const void* x_bf16, int M, int K, int8_t* xq, float* x_scale, void* stream);

/* Ternary GEMM + dequant epilogue, Eq. 4 line 3:
 *   acc_mn = sum_j xq_mj * q_nj  (int32, exact);  y_mn = (float)acc_mn * (x_scale_m * w_scale)
 *   packed     from vla_ternary_pack for the same (N,K)
 *   w_scale    device pointer to ONE fp32 (beta, the per-tensor checkpoint scale); unused for VLA_I32
 *   xq         [M,K] int8, x_scale [M] fp32 (from vla_act_quant; x_scale unused for VLA_I32)
 *   out        [M,N] of out_dtype
 *   workspace  >= vla_ternary_workspace_bytes(M,N,K,path) bytes (may be NULL if that is 0) */
vla_status vla_ternary_gemm(const void* packed, const float* w_scale, const int8_t* xq, const float* x_scale,
                            int M, int N, int K, void* out, vla_dtype out_dtype, vla_path path,
                            void* workspace, size_t workspace_bytes, void* stream);

/* Eq. 4 end to end with the activation quant fused into the call: x_bf16 [M,K] -> out [M,N].
 *   xq_opt / x_scale_opt   optional outputs ([M,K] int8, [M] fp32): also return the quantised
 *                          activations; when NULL they live in `workspace`. */
vla_status vla_ternary_linear(const void* packed, const float* w_scale, const void* x_bf16,
                              int M, int N, int K, void* out, vla_dtype out_dtype, vla_path path,
                              int8_t* xq_opt, float* x_scale_opt,
                              void* workspace, size_t workspace_bytes, void* stream);

/* Host-buffer form of vla_ternary_linear (the end-to-end call a serving process makes; the weights stay
 * resident in HBM: "holds weights resident"):
 *   x_bf16_host  HOST [M,K] bf16 (pinned memory for an asynchronous copy)
 *   out_host     HOST [M,N] of out_dtype
 *   workspace    DEVICE, >= vla_ternary_host_workspace_bytes(M,N,K,out_dtype,path): staging for x and out
 *                plus the quantised activations
 * Copies x host->device, runs Eq. 4 in the kernels, copies out device->host, all on `stream`, and
 * SYNCHRONISES `stream` before returning. */
size_t vla_ternary_host_workspace_bytes(int M, int N, int K, vla_dtype out_dtype, vla_path path);
vla_status vla_ternary_linear_host(const void* packed, const float* w_scale, const void* x_bf16_host,
                                   int M, int N, int K, void* out_host, vla_dtype out_dtype, vla_path path,
                                   void* workspace, size_t workspace_bytes, void* stream);

/* vla_ternary_linear for callers that CANNOT ALLOCATE device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the scratch of the call -- the quantised activations [M,K] int8 and their
 * scales [M] fp32 -- lives in a fixed array inside the library (csrc/no_alloc.cu; every GPU that loads the library holds
 * its VLA_STATIC_MAX_MK + 4 * VLA_STATIC_MAX_M bytes until the process exits), so there is no workspace argument and the
 * call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine).  Same arithmetic, same kernels and
 * the same result, bit for bit, as vla_ternary_linear.
 *   limit   M * K <= VLA_STATIC_MAX_MK and M <= VLA_STATIC_MAX_M, else VLA_ERR_WORKSPACE (use vla_ternary_linear with
 *           a workspace of your own for larger problems); other errors as vla_ternary_linear
 *   sharing every call on a device uses the SAME array, which keeps the last call's contents (nothing in it has to be
 *           cleared: each call overwrites what it reads).  Calls that overlap on the GPU -- different streams, graphs
 *           replayed concurrently -- race on it: issue them on one stream, or order them with events.
 * Asynchronous on `stream`, capturable. */
#define VLA_STATIC_MAX_MK 8388608   /* 8 MiB of int8 activations, e.g. M = 1024 at K = 8192, M = 1213 at K = 6912 */
#define VLA_STATIC_MAX_M 16384
vla_status vla_ternary_linear_static(const void* packed, const float* w_scale, const void* x_bf16,
                                     int M, int N, int K, void* out, vla_dtype out_dtype, vla_path path, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * Programs: a whole list of ternary linears -- all small-M (decode) or all large-M (prefill) -- in ONE persistent launch.
 *
 * "graphs and buffers persist across same-shape requests ... GPU graph capture" removes
 * dispatch overhead.  On B200 one launch costs more than ten times the HBM time of a BitNet-2B weight
 * tensor, so the library goes one step further: a program is compiled once and then executed by a single
 * persistent kernel (csrc/gemm_program.cu) that streams the packed weights of every stage back to back
 * and synchronises only where a stage reads what an earlier stage wrote.
 *
 * A STAGE is one activation matrix x [M,K] bf16 (small programs: 1 <= M <= 16; K % 128 == 0, K <= 8192) and n_linears
 * (1..16) ternary linears that all consume it, each with its own packed W [N,K], scale beta and output:
 * the per-output-group scales beta_g(n) of Eq. 4, e.g. q|k|v or gate|up.
 * Every stage runs Eq. 4 end to end inside the one kernel: absmax int8 quant of x (fused: small stages are quantised by
 * every CTA of the stage straight into shared memory, larger ones once per row and shared through the program buffer),
 * int32 contraction, dequant to out_dtype.
 *   depends = 0   x does not depend on the stages since the last depends = 1 stage: the stage joins the
 *                 current PHASE, whose stages run concurrently on disjoint groups of SMs
 *   depends = 1   x is (part of) the output of EARLIER stages of this program: the stage opens a new
 *                 phase, which starts only after every earlier phase has completed on the whole grid
 *
 * LARGE programs (csrc/gemm_lprog.cu): if the stages have M > 16 tokens (17 <= M <= 32768, K <= 8192, 1..8 linears per
 * stage; ALL stages of a program are of one kind, else VLA_ERR_SHAPE) the program runs on the tcgen05 / TMEM kernel
 * instead: every CTA quantises a share of the rows of x into int8 scratch inside the program buffer (or into xq_opt /
 * x_scale_opt), the CTAs meet on a grid-wide counter, and the stage's 128-channel x token tiles are walked as in
 * VLA_PATH_LARGE; the launch does not end between stages.  Stages run in list order; depends = 1 makes a stage's
 * quantisation wait until EVERY earlier stage has stored its outputs, depends = 0 lets it run ahead (its x must not be
 * written by this program).  Large programs also accept depends = d in 2..s: stage s then waits only for the stages up to
 * s - d (its x is written by those), so that d independent chains -- e.g. a layer stack run on d row blocks of the
 * batch, the stages of the blocks interleaved -- overlap each other's hand-offs instead of running in lockstep.
 * Results are bit-identical to vla_ternary_linear.
 * All pointers inside the descriptors are DEVICE pointers, 16-byte aligned, and must stay valid for as
 * long as the program is run.  The descriptor arrays themselves are HOST memory.
 */
typedef struct {
    const void* packed;     /* from vla_ternary_pack for (N, K of the stage) */
    const float* w_scale;   /* device pointer to one fp32 (beta) */
    void* out;              /* [M,N] of out_dtype */
    int N;                  /* N % 128 == 0 */
    int out_dtype;          /* vla_dtype */
} vla_prog_linear;

typedef struct {
    const void* x_bf16;     /* [M,K] bf16 */
    int M, K;
    int depends;            /* 0 or 1 (large programs: 0..stage index), see above */
    int n_linears;
    const vla_prog_linear* linears;   /* HOST array of n_linears entries */
    int8_t* xq_opt;         /* optional: also return the quantised activations [M,K] int8 (NULL: kept inside the program) */
    float* x_scale_opt;     /* optional: alpha [M] fp32 */
} vla_prog_stage;

/* Eq. 4 for up to 8 linears that share ONE pre-quantised activation matrix (per-output-group scales beta_g(n),
 * q|k|v, gate|up) in as few launches as the path allows: one tcgen05 launch where the path is
 * VLA_PATH_LARGE (VLA_PATH_AUTO: M > 32, and 16 < M <= 32 by the group's total N and K), one launch per linear otherwise.  `lins` is a HOST array; its pointers are device pointers (see vla_prog_linear).
 * Every linear has the same K.  Asynchronous on `stream`, capturable. */
vla_status vla_ternary_gemm_grouped(const vla_prog_linear* lins /*host*/, int n_linears, const int8_t* xq,
                                    const float* x_scale, int M, int K, vla_path path, void* stream);

/* Device bytes a compiled program needs (descriptor tables, barrier counters, quantised activations: for a large
 * program eight int8 [M,K] + alpha [M] scratch sets of its largest stage); a multiple of 256.  0 if any stage is invalid
 * or small and large stages are mixed. */
size_t vla_program_bytes(const vla_prog_stage* stages /*host*/, int n_stages);

/* Compiles `stages` into prog_dev (device memory, >= vla_program_bytes, 256-byte aligned).
 * SYNCHRONISES `stream`.  VLA_ERR_SHAPE / _NULL / _ALIGN / _DTYPE as for the single calls. */
vla_status vla_program_build(const vla_prog_stage* stages /*host*/, int n_stages, void* prog_dev, size_t prog_bytes,
                             void* stream);

/* Runs a compiled program: ONE kernel launch, asynchronous on `stream`, capturable in a CUDA graph.
 * Returns VLA_ERR_VALUE if prog_dev was not produced by vla_program_build in this process.
 * Runs of the same program must not overlap in time (they share its counters and activation scratch).
 * The kernel is persistent (one CTA per SM) and, for programs with more than one phase or with cooperatively quantised
 * stages, its CTAs wait for each other: vla_program_build sizes the grid so that all of them are resident on an
 * otherwise idle device.  Do not run another persistent or SM-filling kernel concurrently with such a program (another
 * stream, MPS, a green context with fewer SMs): a CTA that never becomes resident makes the others wait until the
 * kernel's watchdog (~2 s of spinning) traps, which surfaces as VLA_ERR_CUDA on the next call, not as a hang. */
vla_status vla_program_run(const void* prog_dev, void* stream);

/* Host-buffer form of vla_program_run (the end-to-end call of a serving process): copies every `in` entry
 * host->device, runs the program, copies every `out` entry device->host, all on `stream`, then SYNCHRONISES
 * `stream`.  `host` pointers are HOST memory (pinned for asynchronous copies), `dev` pointers the device
 * buffers the program's stages read / write.  The arrays themselves are HOST memory. */
typedef struct {
    void* host;
    void* dev;
    size_t bytes;
} vla_copy;
vla_status vla_program_run_host(const void* prog_dev, const vla_copy* in /*host*/, int n_in,
                                const vla_copy* out /*host*/, int n_out, void* stream);
/* The same WITHOUT the final synchronisation: the three parts are only enqueued on `stream`.  A serving loop alternates two
 * programs (each with its own device and pinned host buffers) on two streams, so that the host->device copy of step t+1
 * and the device->host copy of step t-1 overlap the kernel of step t; the caller synchronises `stream` (or an event
 * recorded on it) before it reads an `out` host buffer or rewrites an `in` host buffer. */
vla_status vla_program_run_host_async(const void* prog_dev, const vla_copy* in /*host*/, int n_in,
                                      const vla_copy* out /*host*/, int n_out, void* stream);

/* Forgets a compiled program (the caller then frees prog_dev). */
vla_status vla_program_release(const void* prog_dev);

/* ---------------------------------------------------------------------------------------------------
 * Cached-conditioning cross-attention, Eq. 2 of the paper (section III-B), per head:
 *
 *     Attn(Q, K_C, V_C; M) = softmax(Q K_C^T / sqrt(d_k) + M) V_C          softmax over keys
 *
 * K_C = Z W_K and V_C = Z W_V are the cached projections of the conditioning sequence ("a cross-attention head caches
 * K_C and V_C"): the caller computes them ONCE per observation (e.g. with vla_ternary_linear on the
 * k / v weights) and passes the same buffers to every solver step; only q changes between steps.
 *   q_bf16       [Mq, n_q_heads * d_k] bf16, row-major (the q linear's output: head h is columns [h*d_k, (h+1)*d_k))
 *   kc_bf16      [Mc, n_kv_heads * d_k] bf16 (the k linear's output), vc_bf16 the same shape (the v linear's output)
 *   visible_opt  NULL (every key visible) or [Mq, Mc] bytes: 1 = visible (M = 0), 0 = masked (M = -inf)
 *   out          [Mq, n_q_heads * d_k] of out_dtype (VLA_F32 or VLA_BF16 with round-to-nearest-even)
 *   workspace    >= vla_cached_attention_workspace_bytes(...) bytes (partial results of the key splits)
 * Grouped-query heads: query head h reads KV head h / (n_q_heads / n_kv_heads).  A query row whose keys are all masked
 * gives 0.  Shapes: d_k == 128, n_q_heads % n_kv_heads == 0 with at most 8 query heads per KV head, 1 <= Mq <= 4096,
 * 1 <= Mc <= 65536 (else VLA_ERR_SHAPE).  Arithmetic: bf16 x bf16 products and all sums in fp32, probabilities kept to
 * 2^-17 relative; the result is within 2e-5 * max|V_C| of the float64 value of Eq. 2.  Asynchronous on
 * `stream`, capturable in a CUDA graph. */
size_t vla_cached_attention_workspace_bytes(int Mq, int Mc, int n_q_heads, int n_kv_heads, int d_k);
vla_status vla_cached_attention(const void* q_bf16, const void* kc_bf16, const void* vc_bf16, const uint8_t* visible_opt,
                                int Mq, int Mc, int n_q_heads, int n_kv_heads, int d_k, void* out, vla_dtype out_dtype,
                                void* workspace, size_t workspace_bytes, void* stream);

/* The path VLA_PATH_AUTO resolves to for (M,N,K). */
vla_path vla_ternary_auto_path(int M, int N, int K);

const char* vla_status_string(vla_status s);

/* ---------------------------------------------------------------------------------------------------
 * Instrumentation (benchmarks only; nothing below is on the hot path or needed to use the library).
 * --------------------------------------------------------------------------------------------------- */

/* Issue `mmas_per_cta` back-to-back
 * tcgen05.mma.cta_group::1.kind::i8 (M=128, N=256, K=32) per CTA on `ctas` CTAs with no loads,
 * and return the elapsed milliseconds through the HOST pointer ms_out.  Gives the box's INT8
 * tensor-pipe ceiling: ops = 2*128*256*32 * mmas_per_cta * ctas.  Synchronises the device. */
vla_status vla_i8_mma_issue_probe(int ctas, int mmas_per_cta, float* ms_out /*host*/);

/* Number of kernels this library has launched so far in this process. */
unsigned long long vla_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* VLA_TERNARY_H */
