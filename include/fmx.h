/* fmx.h — C ABI of the B200-native mixed-task vFM forward (FMplex deployment sharing).
 *
 * What the library computes: ONE batched forward pass of a shared foundation-model backbone
 * over a mixed batch whose requests come from many tasks; each request's task id selects that
 * task's LoRA adapter deltas and its output head (the task's "virtual foundation model",
 * PAPER.md §4.1).  This is steps 4-6 of the paper's request path (PAPER.md L123:
 * "The scheduler then selects queued requests for execution on the shared FM and binds
 * task-specific adapters as needed"), executed as "batches the requests across the common
 * backbone first then integrate adapter difference" (§4.2; Fig. 5(c)).
 * Where the paper's runtime LOOPS over adapter sub-batches (its 45 % throughput cost,
 * PAPER.md L335), this library sorts rows by task on the device and applies all adapters as
 * segmented low-rank GEMM steps fused into the backbone projections.
 *
 * Conventions
 *   - Every function returns int: FMX_OK (0) or a negative fmx_status.  No exceptions cross
 *     the ABI.  fmx_last_error() returns a thread-local message for the last failure.
 *   - "DEVICE" pointers are CUDA device memory on the context's device; "HOST" pointers are
 *     ordinary host memory.  All matrices are row-major; bf16 is the 16-bit brain float.
 *   - Linear weights are [out, in] (PyTorch/PEFT orientation, Listing 2).
 *   - Validation happens fully on the host BEFORE any launch; on error nothing is enqueued
 *     on the stream and no library state changes.
 *   - There is no CPU fallback anywhere: without a CUDA device every compute call returns
 *     FMX_E_CUDA.
 */
#ifndef FMX_H
#define FMX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum fmx_status {
  FMX_OK = 0,
  FMX_E_INVALID_ARG = -1,       /* NULL where a pointer is required, bad enum, n < 0 ...      */
  FMX_E_UNKNOWN_BACKBONE = -2,
  FMX_E_UNKNOWN_TASK = -3,      /* task id not currently registered (or bound to another backbone) */
  FMX_E_SHAPE = -4,             /* adapter/head dims do not match the target; rank not in [1,64];
                                   backbone dims not supported (see fmx_register_backbone)    */
  FMX_E_BAD_LENGTH = -5,        /* length < 1, > max_seq, or != tokens_per_request            */
  FMX_E_WORKSPACE = -6,         /* workspace too small / misaligned                            */
  FMX_E_CAPACITY = -7,          /* too many tasks, requests or tokens                          */
  FMX_E_CUDA = -8               /* CUDA runtime/driver failure; code in fmx_last_error()       */
} fmx_status;

typedef struct fmx_ctx fmx_ctx;      /* opaque; one per device                                */
typedef int32_t fmx_backbone_t;      /* small dense handle                                     */
typedef int32_t fmx_task_t;          /* == the task id fmx_forward_mixed and the BFQ builder use */

enum { FMX_MAX_TASKS = 1024, FMX_MAX_REQUESTS = 4096, FMX_MAX_RANK = 64, FMX_N_TARGETS = 7 };

typedef enum { FMX_ACT_GELU_ERF = 0, FMX_ACT_RELU = 1, FMX_ACT_SWIGLU = 2 } fmx_act;
typedef enum { FMX_NORM_LAYERNORM = 0, FMX_NORM_RMSNORM = 1 } fmx_norm;
typedef enum { FMX_INPUT_EMBEDDED = 0,      /* bf16 [n_i, d_model] per request                 */
               FMX_INPUT_PATCH_LINEAR = 1,  /* bf16 patches (or raw image, see img_*) per request */
               FMX_INPUT_TOKEN_IDS = 2      /* int32 [n_i] per request                          */
} fmx_input_kind;
typedef enum { FMX_TGT_Q = 0, FMX_TGT_K, FMX_TGT_V, FMX_TGT_O, FMX_TGT_GATE, FMX_TGT_UP, FMX_TGT_DOWN } fmx_target;
typedef enum { FMX_HEAD_POOL_MEAN = 0,  /* mean over the request's n_i normed rows            */
               FMX_HEAD_POOL_CLS = 1,   /* row 0                                               */
               FMX_HEAD_POOL_LAST = 2,  /* row n_i - 1                                         */
               FMX_HEAD_FLATTEN = 3     /* all rows, token-major then channel (fixed-length backbones only) */
} fmx_head_kind;

/* Backbone: a pre-norm transformer stack.  Plain data, no architecture enum.
 * Per-layer arrays hold n_layers DEVICE pointers each (the arrays themselves are HOST memory).
 * Ownership: the CALLER owns every device buffer named here; they must stay valid and
 * unchanged until fmx_destroy.  The library stores the pointers and builds TMA descriptors
 * over them (it copies only embed_W, into a K-padded layout).
 * Supported shapes: d_model, n_q_heads*head_dim, n_kv_heads*head_dim and d_ffn multiples of
 * 128; head_dim in {32, 64, 128}; n_q_heads a multiple of n_kv_heads; else FMX_E_SHAPE. */
typedef struct fmx_backbone_desc {
  int32_t n_layers, d_model, n_q_heads, n_kv_heads, head_dim, d_ffn;
  int32_t act;                 /* fmx_act                                                     */
  int32_t norm;                /* fmx_norm                                                    */
  float   norm_eps;
  int32_t causal;              /* 0/1                                                         */
  float   rope_theta;          /* 0 = no RoPE; else rotate-half pairing, position = index in request */
  int32_t input_kind;          /* fmx_input_kind                                              */
  int32_t patch_dim;           /* PATCH_LINEAR: values per patch                              */
  int32_t tokens_per_request;  /* fixed token count per request incl. CLS; 0 = variable       */
  int32_t has_cls;             /* PATCH_LINEAR: prepend embed_cls as token 0                  */
  int32_t vocab;               /* TOKEN_IDS                                                   */
  int32_t max_seq;             /* longest request accepted                                    */
  int32_t img_c, img_hw, patch_hw; /* PATCH_LINEAR fed with raw [C,HW,HW] images: the library
                                   patchifies (row-major grid, each patch flattened (c,row,col));
                                   img_c = 0: input is already [n_patches, patch_dim]          */
  const void *embed_W;         /* bf16 [d_model, patch_dim]      (PATCH_LINEAR)               */
  const void *embed_b;         /* bf16 [d_model] or NULL                                      */
  const void *embed_cls;       /* bf16 [d_model]                 (has_cls)                    */
  const void *embed_pos;       /* bf16 [max_seq, d_model] or NULL: added to token p of every request */
  const void *embed_table;     /* bf16 [vocab, d_model]          (TOKEN_IDS)                  */
  const void *const *norm1_g, *const *norm1_b;   /* bf16 [d_model]; *_b NULL array or NULL entries for RMSNorm */
  const void *const *Wq, *const *Wk, *const *Wv, *const *Wo;        /* bf16 [out, in]          */
  const void *const *bq, *const *bk, *const *bv, *const *bo;        /* bf16 [out]; array may be NULL = no bias */
  const void *const *norm2_g, *const *norm2_b;
  const void *const *Wup, *const *Wgate, *const *Wdown;             /* Wgate only for SWIGLU   */
  const void *const *bup, *const *bgate, *const *bdown;
  const void *final_g, *final_b;
} fmx_backbone_desc;

/* One LoRA adapter on one target projection: y += scaling * (x A^T) B^T  (PEFT orientation). */
typedef struct fmx_adapter_desc {
  int32_t target;              /* fmx_target                                                  */
  int32_t rank;                /* 1..FMX_MAX_RANK                                             */
  float   scaling;             /* lora_alpha / rank                                           */
  const void *const *A;        /* HOST array of n_layers DEVICE pointers, each bf16 [rank, d_in]  */
  const void *const *B;        /* HOST array of n_layers DEVICE pointers, each bf16 [d_out, rank] */
} fmx_adapter_desc;

/* A task's extensions: PEFT adapter(s) + decoder head.
 * fmx_register_task copies on the library's own registration stream and does not wait for forwards in flight (adding a
 * task to a serving context costs ~1-2 ms, PAPER.md L92 / L243); the source tensors must be complete (the work that
 * produced them finished) when the call is made.  Growing the LoRA slab arena (rare) synchronises the device.
 * Ownership: the library COPIES adapters and head into its own arena (task-sorted slabs laid
 * out for the segmented kernels); the caller may free its buffers when the call returns. */
typedef struct fmx_task_desc {
  int32_t n_adapters;
  const fmx_adapter_desc *adapters;   /* HOST array; at most one per target                   */
  int32_t head_kind;           /* fmx_head_kind                                               */
  int32_t head_out;            /* o_t >= 1                                                    */
  const void *head_W;          /* DEVICE bf16 [head_out, d_feat]; d_feat = d_model, or
                                  tokens_per_request*d_model for FLATTEN                      */
  const void *head_b;          /* DEVICE bf16 [head_out] or NULL                              */
  /* MLP decoder head (Listing 2: MLPDecoder(input_dim, hidden_dim, output_dim)).
   * head_hidden = 0: the linear head above.  head_hidden > 0 (pooled kinds only, <= 4096):
   *   y = W2 · relu(W · feat + b) + b2   with head_W [head_hidden, d_feat], head_b [head_hidden] or NULL,
   *   head_W2 DEVICE bf16 [head_out, head_hidden] (required), head_b2 DEVICE bf16 [head_out] or NULL.
   * The activation is ReLU (the paper names only the three widths; reading 32). */
  int32_t head_hidden;
  const void *head_W2;
  const void *head_b2;
  /* Per-task input encoder (Listing 2: LinearChannelCombiner(num_channels = 3, new_num_channels = 1);
   * SURVEY.md 8(f) NEXT-1).  enc_channels <= 1: none.  enc_channels = C in [2, 16] (PATCH_LINEAR backbones with series
   * input, img_c = 0, only): a request of this task brings C channels, packed channel-major [C, n_patches * patch_dim], and
   * the series the backbone sees is  sum_c enc_W[c] * x[c, :] + enc_b.  enc_W DEVICE bf16 [C]; enc_b DEVICE bf16 [1] or NULL. */
  int32_t enc_channels;
  const void *enc_W;
  const void *enc_b;
} fmx_task_desc;

/* ---- lifecycle ---------------------------------------------------------------------- */
int fmx_create(fmx_ctx **out, int device_ordinal);
int fmx_destroy(fmx_ctx *ctx);
const char *fmx_last_error(void);                 /* thread-local; "" if none                  */
const char *fmx_version(void);

/* Registers a backbone; *out receives its handle. */
int fmx_register_backbone(fmx_ctx *ctx, const fmx_backbone_desc *desc, fmx_backbone_t *out);

/* Registers a task on a backbone (vFM creation: extensions + state; tasks
 * arrive without redeploying the FM, L92).  *out receives the task id: the lowest free slot.
 * Synchronises the context's copy stream before returning. */
int fmx_register_task(fmx_ctx *ctx, fmx_backbone_t bb, const fmx_task_desc *desc, fmx_task_t *out);

/* Removes a task (remove_adapter).  Other tasks' outputs are unaffected. */
int fmx_unregister_task(fmx_ctx *ctx, fmx_task_t task);

/* HOST.  out_off[i] .. out_off[i+1] is request i's slice of the fp32 output buffer (prefix sum
 * of head_out in ORIGINAL request order); out_off has n_req + 1 entries. */
int fmx_output_layout(fmx_ctx *ctx, const int32_t *task_ids, int32_t n_req, int64_t *out_off);

/* Bytes of DEVICE workspace fmx_forward_mixed needs for up to max_req requests / max_tokens tokens. */
int fmx_workspace_bytes(fmx_ctx *ctx, fmx_backbone_t bb, int32_t max_req, int64_t max_tokens, size_t *bytes);

/* The mixed-task forward.  Asynchronous on cuda_stream (a cudaStream_t; NULL = default
 * stream); the caller synchronises.  One forward in flight per context.
 *   inputs    DEVICE, requests packed back to back in ORIGINAL request order:
 *             EMBEDDED bf16 [n_i, d_model]; PATCH_LINEAR bf16 [n_patches*patch_dim] or image
 *             [img_c, img_hw, img_hw]; TOKEN_IDS int32 [n_i].
 *   task_ids  HOST int32 [n_req], each a currently registered task of this backbone
 *   lengths   HOST int32 [n_req], tokens per request (fixed-length backbones: must equal
 *             tokens_per_request)
 *   outputs   DEVICE fp32, ragged, layout = fmx_output_layout
 *   workspace DEVICE, caller-owned, >= fmx_workspace_bytes(n_req, sum lengths), 1024-B aligned
 * n_req = 0 returns FMX_OK and launches nothing. */
int fmx_forward_mixed(fmx_ctx *ctx, fmx_backbone_t bb, const void *inputs, const int32_t *task_ids,
                      const int32_t *lengths, int32_t n_req, float *outputs, void *workspace,
                      size_t workspace_bytes, void *cuda_stream);

/* Same, end to end from HOST buffers: copies inputs host->device, runs the forward, copies the
 * outputs device->host and synchronises.  inputs_bytes = total bytes of the packed inputs. */
int fmx_forward_mixed_host(fmx_ctx *ctx, fmx_backbone_t bb, const void *inputs_host, size_t inputs_bytes,
                           const int32_t *task_ids, const int32_t *lengths, int32_t n_req,
                           float *outputs_host, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Debug/test: copies the segment tables of the LAST forward to HOST arrays (synchronises).
 * Sizes: perm, inv_perm [n_req]; task_req_off, task_tok_off [n_slots+1]; cu_tok [n_req+1];
 * n_slots = fmx_task_slots().  Any pointer may be NULL. */
int fmx_debug_get_segments(fmx_ctx *ctx, int32_t *perm, int32_t *inv_perm, int32_t *task_req_off,
                           int32_t *cu_tok, int32_t *task_tok_off);
/* Debug/test: the private row-tile table of the last forward (256-row CTA-pair tiles): n_tiles,
 * n_blocks, and per block (tile, task, row_lo, row_hi) into blocks[4*n_blocks] (cap entries available). */
int fmx_debug_get_tiles(fmx_ctx *ctx, int32_t *n_tiles, int32_t *n_blocks, int32_t *blocks, int32_t cap);
/* Debug/test: copies an activation buffer of the LAST forward to HOST (synchronises).  which:
 * 0 X fp32 [N,d] (residual, task-sorted rows)  1 Xn bf16 [N,d]  2 QKV bf16 [N,d_qkv]  3 attention out
 * bf16 [N,d_q]  4 FFN hidden bf16 [N,d_ffn]  5 U bf16 [n_blk_cap*256,192]  6 pooled feature fp32 [B,d]. */
int fmx_debug_read(fmx_ctx *ctx, int which, void *host, size_t bytes);
int fmx_task_slots(fmx_ctx *ctx);                 /* number of task slots (highest id ever live + 1) */

/* Per-kernel-family timing of the next forwards (CUDA events around every launch, on the
 * forward's stream).  Families: see fmx_profile_family_name.  fmx_profile_read synchronises
 * and returns, per family, launches and total milliseconds since the last fmx_profile_enable(1). */
enum { FMX_N_FAMILIES = 12 };
int fmx_profile_enable(fmx_ctx *ctx, int on);
/* Restricts the events to the families whose bit is set (bit f = family f; default all), so a timed
 * region can carry events around its dominant kernels only. */
int fmx_profile_select(fmx_ctx *ctx, uint32_t family_mask);
int fmx_profile_read(fmx_ctx *ctx, int32_t *launches /*[FMX_N_FAMILIES]*/, double *total_ms /*[FMX_N_FAMILIES]*/);
const char *fmx_profile_family_name(int family);
/* Kernels launched by the last forward (the count bench.py reports as gpu_launches). */
int fmx_last_launch_count(fmx_ctx *ctx);
/* Forwards served by replaying the context's cached CUDA graph so far (FMX_OPT_GRAPH; debug / tests). */
long long fmx_graph_replays(fmx_ctx *ctx);

/* Debug/test: one GEMM through the tcgen05 kernel, C[M,N] (fp32) = A[M,K] (bf16) · W[N,K]^T (bf16);
 * N a multiple of 128, K a multiple of 8.  All DEVICE pointers. */
int fmx_debug_gemm(fmx_ctx *ctx, const void *A, const void *W, float *C, int32_t M, int32_t N, int32_t K,
                   void *cuda_stream);

/* Debug/test: the fused variable-length attention step (S3d) alone.  qkv DEVICE bf16
 * [n_tokens, (n_q_heads + 2 n_kv_heads) * head_dim] (q | k | v per row, requests packed back to back),
 * cu_tok HOST int32 [n_req + 1] (prefix sums of the request lengths), out DEVICE bf16
 * [n_tokens, n_q_heads * head_dim].  impl: an FMX_ATTN_* value.  Scale 1/sqrt(head_dim). */
int fmx_debug_attention(fmx_ctx *ctx, const void *qkv, void *out, const int32_t *cu_tok, int32_t n_req,
                        int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, int32_t causal, int32_t impl,
                        void *cuda_stream);

/* Tuning knobs (process-local experiments; defaults are what bench.py measures). */
enum {
  FMX_OPT_ATTENTION_IMPL = 0,    /* FMX_ATTN_AUTO | FMX_ATTN_MMA_SYNC | FMX_ATTN_TCGEN05 | FMX_ATTN_LANES */
  FMX_OPT_ATTENTION_VARIANT = 1, /* tcgen05 attention: 0 = one 128-query tile per CTA; 1 = two q-tiles per CTA
                                    sharing K/V.  FMX_ATTN_LANES: 0 / 1 / 2 = 4 / 2 / 3 lanes per CTA (head_dim 64) */
  FMX_OPT_SHRINK_STAGES = 3,     /* LoRA shrink kernel pipeline: 5 (default) = as deep as ~200 KB allow for the stage size
                                    (8 / 6 / 5 stages for 1 / 2 / 3 targets), 4 = four 40 KB stages */
  FMX_OPT_HALF_TILES = 4,        /* 1 (default): a short last GEMM wave is cut into 256 x 128 half tiles */
  FMX_OPT_ATTN_SHORT = 5,        /* batches whose requests all have <= 64 tokens: 0 = generic kernels, 1 = pipelined
                                    single-tile mma.sync kernel, 2 (default) = tcgen05 head-pair kernel when head_dim is
                                    64 and the head count even (FMX_ATTN_AUTO only), else as 1 */
  FMX_OPT_ROPE_FUSED = 6,        /* 1 (default): head_dim 128 backbones rotate q / k in the QKV GEMM epilogue;
                                    0: separate RoPE kernel over the bf16 QKV buffer */
  FMX_OPT_HEAD_TILED = 7,        /* FLATTEN heads: 0 = one warp per (request, output), 1 = CUDA-core 4 x 4 register tiles,
                                    2 (default) = mma.sync 16-request x 32-output tiles over K chunks */
  FMX_OPT_SHRINK_FUSED = 8,      /* the LoRA shrink runs as the first work items of the GEMM that consumes it: 0 = never
                                    (separate shrink kernel), 1 (default) = when the batch has at most one (tile, task)
                                    block per CTA pair, 2 = always */
  FMX_OPT_GRAPH = 9,             /* 1 (default): fmx_forward_mixed captures a CUDA graph on the 2nd identical call (same
                                    buffers, stream, ids, lengths, registrations, options) and replays it afterwards;
                                    needs a non-default stream; 0: always plain launches */
  FMX_OPT_REVERSE = 10,          /* 1 (default): consecutive kernels of a layer walk the token rows in alternating
                                    directions, so each starts on the rows its producer wrote last (still in L2) */
  FMX_OPT_EXPAND_WIDE = 11,      /* 1 (default): a 256-wide tile whose two chunks share a weight source runs its LoRA
                                    expand as one N = 256 step per block (U loaded once) instead of two N = 128 steps */
  FMX_OPT_DEEP_PIPE = 12,        /* 1 (default): fp32-output GEMMs (residual, embed) run with one more smem pipeline stage
                                    and a single epilogue staging buffer per warpgroup */
  FMX_OPT_PDL = 2                /* programmatic dependent launch of the forward's kernels (process-wide):
                                    0 = off, 1 = always, 2 (default) = only for batches of <= 4096 token rows */
};
enum { FMX_ATTN_AUTO = 0, FMX_ATTN_MMA_SYNC = 1, FMX_ATTN_TCGEN05 = 2, FMX_ATTN_LANES = 3 };
int fmx_set_option(fmx_ctx *ctx, int32_t option, int32_t value);

/* ---- BFQ: host-side batch-aware fair-queue batch builder (§4.2, Eq. 1-3) ------------
 * Pure host code (no CUDA).  It emits the task ids / lengths fmx_forward_mixed consumes. */
typedef struct fmx_bfq fmx_bfq;
typedef struct fmx_bfq_params {
  int32_t n_tasks;             /* task ids 0 .. n_tasks-1                                     */
  int32_t b_max;               /* B_max: max batch size ("profiled throughput knee", L160)    */
  const double *lat_ms;        /* HOST [b_max]: profiled latency (ms) of a batch of b = 1..b_max */
  double l_tok_ms;             /* > 0: token-level charging, a request of n tokens costs l_tok_ms*n (L168) */
} fmx_bfq_params;

int fmx_bfq_create(const fmx_bfq_params *p, fmx_bfq **out);
int fmx_bfq_destroy(fmx_bfq *q);
int fmx_bfq_set_task(fmx_bfq *q, fmx_task_t task, double weight, double slo_ms /* INFINITY = none */);
/* Eq. 1-2: S = max(F_prev, v), F = S + l/w, v = max_i F_i^last at arrival. */
int fmx_bfq_enqueue(fmx_bfq *q, fmx_task_t task, uint64_t req_handle, int32_t length, double arrival_ms);
/* Orders queued requests by (S, F, arrival seq) and extends the batch until min(b_max, cap) or
 * until admitting the next request would push any selected request past arrival + SLO given
 * now + Lat(b+1).  Outputs in admission order; *n_out = 0 if nothing is queued. */
int fmx_bfq_next_batch(fmx_bfq *q, double now_ms, int32_t cap, int32_t *task_ids, int32_t *lengths,
                       uint64_t *req_handles, int32_t *n_out);
/* Eq. 3 retag of the last batch's tasks with the realised per-request service time
 * (measured_batch_ms <= 0: use the profile). */
int fmx_bfq_complete(fmx_bfq *q, double measured_batch_ms);
/* Accounting: per-task dispatched count and charged service time. */
int fmx_bfq_stats(fmx_bfq *q, fmx_task_t task, int64_t *dispatched, double *service_ms, int32_t *queued);
/* Test hook: tags of the j-th queued request of a task: out[0]=S, out[1]=F, out[2]=v_arr. */
int fmx_bfq_peek(fmx_bfq *q, fmx_task_t task, int32_t j, double *out3);

#ifdef __cplusplus
}
#endif
#endif /* FMX_H */
