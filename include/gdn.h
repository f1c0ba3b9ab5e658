/*
 * gdn.h -- C ABI of the B200-native Gated DeltaNet (GDN) chunk forward.
 *
 * One operator, the token-mixing forward of SANA-Streaming's GDN blocks (arxiv/paper_2605_30409,
 * cited below as PAPER.md:L<line>), with the fp32 recurrent state carried from streaming chunk to
 * streaming chunk.  Per (batch b, head h), with the T tokens of the call split into T/G consecutive
 * groups of G tokens (G = tokens per latent frame in the paper; G = 1 is the token-wise gated delta
 * rule S_t = a_t S_{t-1}(I - b_t k_t k_t^T) + b_t v_t k_t^T, o_t = S_t q_t):
 *
 *     S~    = alpha_g * S_{g-1}                                  PAPER.md Eq. 17  (L591)
 *     u_n   = beta_n * (v_n - k_n S~)      for every n in g      PAPER.md Eq. 18  (L595)
 *     S_g   = S~ + sum_n k_n^T u_n                               PAPER.md Eq. 18/19 (L595-L599)
 *     o_n   = scale * q_n S_g              for every n in g      PAPER.md Eq. 22  (L622), numerator
 *
 * and, with GDN_FLAG_NORMALIZER, the normaliser state z (Eq. 20-21, un-rotated keys) and
 * the normalised readout o_n / (q_raw_n . z_g + eps) (Eq. 22).  Row-token orientation of Alg. 1 /
 * Eq. 5 (L118, L369): q,k in R^{T x d_k}; v,o in R^{T x d_v}; S in R^{d_k x d_v}; z in R^{d_k}.
 * The state cache of App. G.6 (L630-L636) is `state_out` of call i fed as `state_in` of call i+1.
 *
 * Conventions for every entry point
 *   - All tensor pointers are DEVICE pointers unless the name says host; the caller owns them.
 *   - Layouts: q,k [B,T,H,d_k]; v,out [B,T,H,d_v] (element type io_dtype, feature dim contiguous,
 *     token stride configurable so a packed qkv [B,T,3,H,d] tensor works);
 *     alpha [B,H,T/G] fp32; beta [B,H,T] fp32; state [B,H,d_k,d_v] fp32 row-major; z [B,H,d_k] fp32.
 *   - Calls enqueue work on `stream` and return without synchronising; errors are return codes and
 *     nothing throws across the ABI.  A plan is bound to the device current at gdn_plan() time and
 *     must not be used from two host threads at once.  Two calls on the same plan must be issued to
 *     the same stream or be externally ordered (they share the plan's workspace).
 *   - Frame-wise tensor-core calls (three to five launches) issued on a NON-default stream are captured
 *     once per tuple of argument pointers into a CUDA graph and replayed on later calls with the same pointers (one
 *     graph launch per call; the plan keeps up to 32 graphs).  Results are bit-identical to direct launches.  Calls on
 *     the legacy default stream, calls made while the caller is capturing `stream`, and calls with per-kernel profiling
 *     enabled are issued directly.
 *   - There is no CPU fallback: on a device that is not sm_100 every compute call returns GDN_ERR_ARCH.
 */
#ifndef GDN_B200_H_
#define GDN_B200_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gdn_plan gdn_plan_t;          /* opaque; owned by the library, freed by gdn_destroy */
typedef void* gdn_stream_t;                  /* a cudaStream_t (0 = the legacy default stream)     */

typedef enum {
    GDN_OK = 0,
    GDN_ERR_INVALID_ARG = 1,   /* NULL where a pointer is required, non-positive sizes, T % G != 0, ...  */
    GDN_ERR_UNSUPPORTED = 2,   /* well-formed but not implemented (head dim, flag, dtype combination)   */
    GDN_ERR_ALIGNMENT = 3,     /* pointer not 16-byte aligned / token stride not a multiple of 8 elems  */
    GDN_ERR_NOMEM = 4,         /* workspace allocation failed                                           */
    GDN_ERR_ARCH = 5,          /* device is not sm_100 (B200); there is no fallback path                */
    GDN_ERR_CUDA = 6           /* a CUDA runtime/driver call failed; see gdn_last_error()               */
} gdn_status_t;

typedef enum { GDN_BF16 = 0, GDN_FP32 = 1 } gdn_dtype_t;     /* element type of q, k, v, out */

enum {
    GDN_FLAG_NORMALIZER = 1u,  /* also run the z path and divide (gdn_forward_chunk_norm only)          */
    GDN_FLAG_BIDIR      = 2u,  /* bidirectional in-chunk scan (Alg. 1 l.8-22): forward scan from the cache + reverse scan over the
                                  frames of this call, readout on S> + S<; state_out stays the forward terminal state.
                                  Frame-wise bf16 tensor-core plans only, else UNSUPPORTED */
    GDN_FLAG_LOG_ALPHA  = 4u,  /* `alpha` holds log(alpha) (<= 0) instead of alpha in (0,1]             */
    GDN_FLAG_FORCE_SIMT = 8u,  /* use the fp32 CUDA-core kernel even where a tensor-core path exists    */
    GDN_FLAG_UNFUSED    = 16u  /* token-wise tensor-core path as three kernels (prepass / chain / output)
                                  instead of the single persistent kernel (C = 128 only; for A/B tests)  */
};

typedef struct {
    uint32_t struct_size;      /* = sizeof(gdn_config_t); ABI versioning                                 */
    int32_t  B, H, T;          /* T = tokens per call (one streaming chunk); B,H,T >= 0                  */
    int32_t  d_k, d_v;               /* each in {32,64,128}; or both 112 (the paper's head dim): bf16 tensor-core plans
                                        compute it as 128 with the padding done by the tensor maps (Alg. 1 l.1)        */
    int32_t  group;            /* G: 1 = token-wise; tokens-per-frame = frame-wise (paper). T % G == 0   */
    int32_t  chunk;            /* token-wise compute tile C in {64, 128}; 0 = auto. Ignored when G > 1.
                                  Results do not depend on C beyond rounding.                           */
    int32_t  io_dtype;         /* gdn_dtype_t                                                            */
    float    scale;            /* multiplies the numerator q S; the paper has no query scale: use 1.0f   */
    float    eps;              /* 1e-6f; only used with GDN_FLAG_NORMALIZER              */
    uint32_t flags;
    int64_t  q_token_stride, k_token_stride, v_token_stride, o_token_stride;
                               /* elements between consecutive tokens; 0 => H*d (dense). The batch
                                  stride is T*token_stride, the head stride is d.                        */
} gdn_config_t;

/* Which kernels a plan resolved to (for logs, tests and the bench JSON). */
typedef enum { GDN_PATH_SIMT_FP32 = 0, GDN_PATH_TC_TOKEN = 1, GDN_PATH_TC_FRAME = 2 } gdn_path_t;

typedef struct {
    int32_t  path;             /* gdn_path_t                                                             */
    int32_t  chunk;            /* resolved compute tile C (token-wise tensor-core path), else 0          */
    int32_t  launches_per_call;/* number of kernel launches one gdn_forward_chunk enqueues               */
    int32_t  sm_count;         /* SMs of the plan's device (0 if no device was visible at plan time)     */
    uint64_t workspace_bytes;  /* device workspace owned by the plan                                     */
} gdn_plan_info_t;

/*
 * gdn_plan: validate `cfg`, choose the kernels, allocate the plan's device workspace.
 *   Returns GDN_OK and a plan in *plan_out, or an error and *plan_out = NULL.
 *   Shapes, dtype, G and flags are fixed per plan (the paper's first chunk has 5 frames, later chunks
 *   3 -- PAPER.md L460 -- so a stream holds one plan per distinct T).  With B, H or T equal to 0 the
 *   plan is valid and every forward call is a no-op (state_out = state_in).
 *   Plans can be created without a visible GPU (validation only); compute calls then return ARCH/CUDA.
 */
gdn_status_t gdn_plan(const gdn_config_t* cfg, gdn_plan_t** plan_out);

/*
 * gdn_forward_chunk: out, state_out = GDN(q, k, v, alpha, beta, state_in)  -- equations at the top.
 *   q,k        [B,T,H,d_k] io_dtype, device            alpha  [B,H,T/G] fp32, device (alpha or log alpha)
 *   v          [B,T,H,d_v] io_dtype, device            beta   [B,H,T]   fp32, device
 *   state_in   [B,H,d_k,d_v] fp32, device, or NULL (= zeros: "cached state or zero", Alg. 1 l.9 L338)
 *   out        [B,T,H,d_v] io_dtype, device; must not alias any input
 *   state_out  [B,H,d_k,d_v] fp32, device; may be the same buffer as state_in (streaming use)
 *   Pointers must be 16-byte aligned and token strides multiples of 8 elements, else ALIGNMENT.
 *   Domain: the update is a contraction when beta_n |k_n|^2 <= 1 (G=1) resp. ||K^T B K||_2 <= 1 (G>1);
 *   the library does not check it (reading 21).
 */
gdn_status_t gdn_forward_chunk(gdn_plan_t* plan,
                               const void* q, const void* k, const void* v,
                               const float* alpha, const float* beta,
                               const float* state_in,
                               void* out, float* state_out,
                               gdn_stream_t stream);

/*
 * gdn_forward_chunk_norm: the paper's full readout (plan must carry GDN_FLAG_NORMALIZER):
 *   matrix path with the rotated q_rot,k_rot (Eq. 18-19), vector path z with the un-rotated k_raw
 *   (Eq. 20-21), out_n = scale * q_rot_n S_g / (q_raw_n . z_g + eps) (Eq. 22).
 *   z_in [B,H,d_k] fp32 or NULL; z_out [B,H,d_k] fp32 (may alias z_in).  Other arguments as above.
 *   q_raw has the layout of q_rot (q_token_stride) and k_raw the layout of k_rot (k_token_stride).
 *   Frame-wise bf16 plans (group > 1, d_k = d_v in {64,112,128}) run it on the tensor-core path: the z recurrence goes
 *   through the same summary and scan kernels as column 0 of a matrix state (the z path is the matrix path with v = 1);
 *   the readout of the matrix pass takes z_f from that scan, forms q_raw . z_f per token and divides in its epilogue.
 *   Everything else (token-wise, fp32, d = 32) runs on the fp32 CUDA-core kernel.
 */
gdn_status_t gdn_forward_chunk_norm(gdn_plan_t* plan,
                                    const void* q_rot, const void* k_rot, const void* v,
                                    const void* q_raw, const void* k_raw,
                                    const float* alpha, const float* beta,
                                    const float* S_in, const float* z_in,
                                    void* out, float* S_out, float* z_out,
                                    gdn_stream_t stream);

/*
 * Front end of the GDN block (App. G.2-G.3, G.5; Alg. 1 "Require: qkv, beta, decay alpha, normalization
 * weights, RoPE tables", L325).  bf16 plans only; D = cfg.d_k = cfg.d_v a multiple of 8, at most 128.
 *
 * gdn_featmap_args_t: the operands of the feature map of Eq. 12 (L552) with the key rescale of L554,
 *     x^ = rho_3D(ReLU(RMSNorm(x))),  K and K^ additionally * 1/sqrt(D N),  N = cfg.group tokens per frame.
 *   q, k       [B,T,H,D] bf16 raw projections (Eq. 11), token strides cfg.q_token_stride / cfg.k_token_stride
 *              (a packed qkv [B,T,3,H,D] tensor works), device
 *   rms_wq/wk  [H,D] fp32 RMSNorm weights; RMSNorm is taken over the D channels of one head:
 *              x_i / sqrt(mean_j x_j^2 + rms_eps) * w_i (reading 23), device
 *   rope_cos/sin [T, D/2] fp32: the rotation of the ADJACENT channel pair (2i, 2i+1) of token t (reading 24), device
 */
typedef struct {
    const void *q, *k;
    const float *rms_wq, *rms_wk;
    const float *rope_cos, *rope_sin;
    float rms_eps;
} gdn_featmap_args_t;

/*
 * gdn_feature_map: q_rot, k_rot (for the KV memory, Eq. 18-19, 22) and q_raw, k_raw (un-rotated, for the normaliser,
 *   Eq. 20-22) from ONE read of q and k.  Outputs: dense [B,T,H,D] bf16, device, caller-owned, must not alias the inputs.
 */
gdn_status_t gdn_feature_map(gdn_plan_t* plan, const gdn_featmap_args_t* args,
                             void* q_rot, void* k_rot, void* q_raw, void* k_raw, gdn_stream_t stream);

/*
 * gdn_gate_args_t / gdn_compute_gates: the gates of Eq. 13-15 (L562-L572) from the per-head latent features x:
 *     alpha_f = exp(-e^{A_log} softplus(W_alpha . mean_n x_{f,n} + b_alpha))  per frame (group) and head,
 *     beta_n  = sigmoid(W_beta . x_n + b_beta)                                 per token and head.
 *   x [B,T,H,D] bf16 with token stride x_token_stride (0 = dense); w_alpha, w_beta [H,D] fp32; b_alpha, a_log, b_beta [H]
 *   fp32; all device.  alpha_out [B,H,T/G] fp32 receives alpha, or log(alpha) when the plan carries GDN_FLAG_LOG_ALPHA
 *   (recommended: the path only ever uses differences of cumulative logs); beta_out [B,H,T] fp32.
 *   Sums have a fixed order: results are bit-identical from run to run.
 */
typedef struct {
    const void* x;
    int64_t x_token_stride;
    const float *w_alpha, *b_alpha, *a_log, *w_beta, *b_beta;
} gdn_gate_args_t;

gdn_status_t gdn_compute_gates(gdn_plan_t* plan, const gdn_gate_args_t* args, float* alpha_out, float* beta_out,
                               gdn_stream_t stream);

/*
 * gdn_compute_gates_static: gdn_compute_gates (Eq. 13-15) for callers that must not allocate -- code under CUDA
 *   graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No plan: the problem is given by plain sizes.
 *   The call allocates NOTHING (no cudaMalloc / cudaFree / allocating library routine; it issues one cudaMemsetAsync and one
 *   kernel launch on `stream`): the scratch gdn_compute_gates keeps in a plan-owned buffer (partial frame sums, arrival
 *   counters) lives in a file-scope `static __device__` array of the library, 80 KB that every GPU loading the library holds
 *   until the process exits.
 *   args, alpha_out [B,H,T/group], beta_out [B,H,T]: as gdn_compute_gates (device pointers; the caller owns them);
 *   D = head dim (multiple of 8, <= 128); log_alpha != 0 writes log(alpha) instead of alpha.
 *   LIMIT: B*H*(T/group) <= 4096 frame-heads per call (the paper's chunk: 60); beyond that GDN_ERR_UNSUPPORTED with a
 *   message naming the limit (gdn_last_error(NULL)), nothing is launched.
 *   SHARING: all calls on a device use the same array and find the last call's contents in it; the call clears what must
 *   start at zero in stream order.  Calls that may run concurrently on the GPU (different streams, no ordering between them)
 *   RACE on it and give wrong gates: serialise them.  Results equal gdn_compute_gates' (bit for bit whenever both choose the
 *   same number of token splits per frame, which they do unless B*H*(T/group)*splits would exceed 16384).
 */
gdn_status_t gdn_compute_gates_static(const gdn_gate_args_t* args, int B, int T, int H, int D, int group, int log_alpha,
                                      float* alpha_out, float* beta_out, gdn_stream_t stream);

/*
 * gdn_forward_chunk_full: the operator at the boundary of the paper's kernel (Alg. 1): feature map on q, k
 *   -> [gates from x] -> GDN recurrence with normalised readout (and the bidirectional in-chunk scan when the plan
 *   carries GDN_FLAG_BIDIR) -> output gate, out = G (.) Y (Eq. 23; the projection W_o is outside).
 *   Frame-wise bf16 tensor-core plans created with GDN_FLAG_NORMALIZER only (else UNSUPPORTED).
 *   fm         feature-map operands (required)
 *   v          [B,T,H,D] bf16, token stride cfg.v_token_stride
 *   gates      NULL: alpha [B,H,T/G] and beta [B,H,T] are given; else they are computed into plan-owned buffers
 *              (alpha, beta ignored)
 *   out_gate   G_f = SiLU(W_g X_f + b_g) evaluated (Eq. 16), [B,T,H,D] bf16 with token stride cfg.o_token_stride, or
 *              NULL (no gate)
 *   S_in, z_in, out, S_out, z_out: as gdn_forward_chunk_norm.
 *   The four feature tensors live in plan-owned device buffers (4 x B*T*H*D bf16, allocated at the first call).
 */
gdn_status_t gdn_forward_chunk_full(gdn_plan_t* plan, const gdn_featmap_args_t* fm, const void* v,
                                    const gdn_gate_args_t* gates, const float* alpha, const float* beta,
                                    const void* out_gate,
                                    const float* S_in, const float* z_in,
                                    void* out, float* S_out, float* z_out, gdn_stream_t stream);

/*
 * gdn_forward_chunk_host: the same operator with HOST buffers (dense layouts, strides in the plan are
 *   ignored; pinned memory recommended).  Copies the inputs to plan-owned device staging buffers,
 *   runs gdn_forward_chunk on `stream`, copies out and state_out back on `stream`, and returns without
 *   synchronising: the caller synchronises `stream` before reading the results.  state_in_host may be NULL.
 *   ORDERING of the input copies: q, k, v, alpha, beta must hold their data WHEN THE CALL IS MADE (they are host
 *   memory): they are copied on internal streams that do not wait for work queued earlier on `stream`, so that
 *   in a sequence of calls the copy-in of call i+1 overlaps the compute and copy-out of call i (two staging
 *   sets).  state_in_host IS read in stream order (a stream of chunks hands the state on through host
 *   memory), and so is every input that overlaps out_host / state_out_host of the plan's previous host call.
 *   As before, no host buffer of a call may be overwritten until `stream` has reached the end of that call.
 */
gdn_status_t gdn_forward_chunk_host(gdn_plan_t* plan,
                                    const void* q_host, const void* k_host, const void* v_host,
                                    const float* alpha_host, const float* beta_host,
                                    const float* state_in_host,
                                    void* out_host, float* state_out_host,
                                    gdn_stream_t stream);

/* gdn_destroy: free the plan and its workspace. NULL is allowed. Does not synchronise the stream:
 * the caller makes sure no call using the plan is still in flight. */
gdn_status_t gdn_destroy(gdn_plan_t* plan);

/* gdn_plan_get_info: fill *info. */
gdn_status_t gdn_plan_get_info(const gdn_plan_t* plan, gdn_plan_info_t* info);

/*
 * gdn_plan_set_profiling / gdn_plan_kernel_times: per-kernel device timing for bench.py's roofline.
 *   With profiling enabled every forward call records CUDA events on the launching stream before its
 *   first kernel and after each kernel.  gdn_plan_kernel_times synchronises those events, writes up to
 *   max_n kernel names (static strings) and the AVERAGE duration in milliseconds of each kernel over the
 *   calls made since profiling was enabled, sets *n_out, and clears the accumulated events.
 *   Not meant for the timed region itself (events between launches add a little latency).
 */
gdn_status_t gdn_plan_set_profiling(gdn_plan_t* plan, int enable);
gdn_status_t gdn_plan_kernel_times(gdn_plan_t* plan, int max_n, const char** names, float* avg_ms, int* n_out);

/* gdn_status_string: static name of a status code. */
const char* gdn_status_string(gdn_status_t status);

/* gdn_last_error: detail text of the last failure on this plan (e.g. the CUDA error string);
 * with plan == NULL, of the last failing gdn_plan() call on this thread. Never NULL. */
const char* gdn_last_error(const gdn_plan_t* plan);

/* gdn_version: library version, e.g. "0.1.0". */
const char* gdn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GDN_B200_H_ */
