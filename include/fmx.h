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
 *     on the stream and no library state changes (a registration that fails part-way returns
 *     what it had allocated; the registry is committed only after its last fallible step).
 *   - fmx_forward_mixed allocates nothing and never synchronises: every scratch buffer it
 *     needs is part of the caller's workspace (fmx_workspace_bytes).
 *   - What the host cannot check (token ids living in device memory) is checked on the device:
 *     an id outside [0, vocab) is embedded as a zero row and raises the context's device error
 *     word, which the NEXT call on the context (or fmx_poll_error) reports as FMX_E_INVALID_ARG.
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
               FMX_HEAD_FLATTEN = 3,    /* all rows, token-major then channel (fixed-length backbones only) */
               FMX_HEAD_DENSE = 4       /* dense (per-token) decoder, "dense decoders for ... detection, and
                                           segmentation": the linear head is applied to EVERY normed token row; the request's
                                           output is [n_i, head_out] row-major (token, then class).  d_feat = d_model; no MLP form */
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
  /* Optional T5-style relative-position bias (reading 36): bias[g][a][b] =
   * rel_bias[bucket(b - a)][g] is added to the scaled scores of query head g, query position a, key position b, in every
   * layer.  Buckets as in T5: half per direction when !causal, exact up to n/2 - 1, then logarithmic up to rel_max_distance,
   * the last one open-ended.  rel_bias NULL / rel_buckets 0 = none.  Backbones with a bias do not serve token decode
   * (fmx_register_lm_head: FMX_E_SHAPE). */
  const void *rel_bias;        /* DEVICE bf16 [rel_buckets, n_q_heads] or NULL; copied at registration */
  int32_t rel_buckets;         /* even, 2 .. 256 (causal: 2 .. 256)                                    */
  int32_t rel_max_distance;    /* > rel_buckets                                                        */
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
 * produced them finished) when the call is made.  Growing the LoRA slab arena (rare) builds the wider arena on that
 * stream too and switches descriptors at a forward boundary; nothing synchronises the device.
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
/* Reports (and clears) a device-side error raised by an earlier forward of this context; call after synchronising the
 * stream.  FMX_OK if none. */
int fmx_poll_error(fmx_ctx *ctx);

/* Registers a backbone; *out receives its handle. */
int fmx_register_backbone(fmx_ctx *ctx, const fmx_backbone_desc *desc, fmx_backbone_t *out);

/* Registers a task on a backbone (vFM creation: extensions + state; tasks
 * arrive without redeploying the FM, L92).  *out receives the task id: the lowest free slot.
 * Synchronises the context's copy stream before returning. */
int fmx_register_task(fmx_ctx *ctx, fmx_backbone_t bb, const fmx_task_desc *desc, fmx_task_t *out);

/* Removes a task (remove_adapter).  Other tasks' outputs are unaffected.  Returns at once: forwards already
 * enqueued still serve the task (its buffers are released on the device after them), later forwards reject its id
 * (FMX_E_UNKNOWN_TASK).  A registration that reuses the freed slot or slab columns waits on the device, not on the host. */
int fmx_unregister_task(fmx_ctx *ctx, fmx_task_t task);

/* HOST.  out_off[i] .. out_off[i+1] is request i's slice of the fp32 output buffer (prefix sum
 * of head_out in ORIGINAL request order); out_off has n_req + 1 entries. */
int fmx_output_layout(fmx_ctx *ctx, const int32_t *task_ids, int32_t n_req, int64_t *out_off);
/* The same with the requests' token counts (HOST int32 [n_req]): a FMX_HEAD_DENSE task contributes lengths[i] * head_out values.
 * fmx_output_layout serves dense tasks only on fixed-length backbones (it uses tokens_per_request), else FMX_E_BAD_LENGTH. */
int fmx_output_layout_len(fmx_ctx *ctx, const int32_t *task_ids, const int32_t *lengths, int32_t n_req, int64_t *out_off);

/* Bytes of DEVICE workspace fmx_forward_mixed needs for up to max_req requests / max_tokens tokens (activations, segment
 * tables and the head scratch: the forward itself allocates nothing). */
int fmx_workspace_bytes(fmx_ctx *ctx, fmx_backbone_t bb, int32_t max_req, int64_t max_tokens, size_t *bytes);
/* The same for fmx_forward_mixed_host, which also stages the packed inputs (max_input_bytes) and the outputs
 * (max_output_floats fp32 values) in the workspace. */
int fmx_host_workspace_bytes(fmx_ctx *ctx, fmx_backbone_t bb, int32_t max_req, int64_t max_tokens, size_t max_input_bytes,
                             int64_t max_output_floats, size_t *bytes);

/* The mixed-task forward.  Asynchronous on cuda_stream (a cudaStream_t; NULL = default
 * stream); the caller synchronises.  Calls on one context are serialised by the context's mutex.
 * A stream that is being captured into a CUDA graph by the caller is refused (FMX_E_INVALID_ARG):
 * ids / lengths travel through a pinned staging ring a replay would find overwritten.
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
 * outputs device->host and synchronises.  inputs_bytes = total bytes of the packed inputs.
 * workspace: >= fmx_host_workspace_bytes(...). */
int fmx_forward_mixed_host(fmx_ctx *ctx, fmx_backbone_t bb, const void *inputs_host, size_t inputs_bytes,
                           const int32_t *task_ids, const int32_t *lengths, int32_t n_req,
                           float *outputs_host, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- token decode with a key / value cache ---------------------------------------------------
 * The paper serves "token-based FMs (e.g., LLMs with continuous batching and long-lived decode iterations)" through the
 * same vFM boundary (fourth difference) and charges "token-level work in service-time units" (L168).  What a
 * decode iteration computes (the paper gives no arithmetic; reading 34): the next-token scores of a request that
 * has seen x_0 .. x_{n-1} are  lm_head · FinalNorm(Backbone_t(x_0 .. x_{n-1}))[n-1]  with its task's adapters - the last row
 * of the ordinary causal forward over the whole prefix.  The cache stores every layer's k / v rows (after RoPE) so that a
 * step feeds ONE new token per request; it must not change the value (tests compare with the no-cache definition).
 * Requests of different tasks decode in one batch (task-sorted rows, segmented LoRA as in fmx_forward_mixed), and the batch
 * may change from step to step (continuous batching): a step names, per request, its task, its cache slot and how many
 * tokens the slot already holds.
 *
 * kv_cache: DEVICE, caller-owned, fmx_kv_cache_bytes(n_slots) bytes, 16-byte aligned; layout
 * [slot][layer][k | v][max_seq][n_kv_heads * head_dim] bf16.  The library keeps no per-slot state: `positions` is the
 * caller's.  Causal backbones only (FMX_E_SHAPE otherwise). */

/* The language-model head of a backbone: W DEVICE bf16 [vocab, d_model], caller-owned (not copied), vocab a multiple of
 * 128.  Register it BEFORE sizing workspaces: fmx_workspace_bytes then includes the [max_req, vocab] fp32 score buffer. */
int fmx_register_lm_head(fmx_ctx *ctx, fmx_backbone_t bb, const void *W, int32_t vocab);
int fmx_kv_cache_bytes(fmx_ctx *ctx, fmx_backbone_t bb, int32_t n_slots, size_t *bytes);

/* Prefill: fmx_forward_mixed that also writes every request's k / v rows into cache slot slots[i] (positions 0 .. n_i - 1).
 *   slots        HOST int32 [n_req], distinct, each in [0, n_slots)
 *   outputs      DEVICE fp32 task-head outputs as fmx_forward_mixed, or NULL to skip the heads
 *   scores       DEVICE fp32 [n_req, vocab] next-token scores in ORIGINAL request order, or NULL
 *   next_tokens  DEVICE int32 [n_req] greedy next token (argmax, lowest index on ties), or NULL
 * Asynchronous on cuda_stream.  Decode iterations of one batch shape replay the context's cached CUDA graph on a non-default
 * stream (ids, slots and positions are copied before every launch, as in fmx_forward_mixed). */
int fmx_prefill(fmx_ctx *ctx, fmx_backbone_t bb, const void *inputs, const int32_t *task_ids, const int32_t *lengths,
                const int32_t *slots, int32_t n_req, float *outputs, float *scores, int32_t *next_tokens, void *kv_cache,
                int32_t n_slots, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* One decode iteration: request i appends token tokens[i] at position positions[i] of its slot (the slot must hold exactly
 * positions[i] tokens, < max_seq) and receives the scores / greedy choice of the NEXT token.
 *   tokens     DEVICE int32 [n_req] (e.g. the next_tokens buffer of the previous call), TOKEN_IDS backbones only
 *   positions  HOST int32 [n_req]
 * workspace: >= fmx_workspace_bytes(n_req, n_req tokens).
 * Reproducibility: a request's scores do not depend on which other requests share the iteration, bit for bit, among batches
 * of 1 .. 128 requests, among batches of 129 .. 256 and among larger ones (the three ranges run different projection kernels). */
int fmx_decode_step(fmx_ctx *ctx, fmx_backbone_t bb, const int32_t *tokens, const int32_t *task_ids, const int32_t *slots,
                    const int32_t *positions, int32_t n_req, float *scores, int32_t *next_tokens, void *kv_cache,
                    int32_t n_slots, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- an entry point that allocates nothing ------------------------------------------------------------------------------
 * The small-M projection of a decode iteration alone (NEXT-3: one row per request of the batch, "long-lived
 * decode iterations"):  out[M, N] (fp32) = x[M, K] (bf16) . W[N, K]^T (bf16), fp32 accumulation, the K axis split over CTAs.
 * For callers that cannot call cudaMalloc or hand over a workspace (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid allocation): the per-slice partial sums live in a file-scope __device__ array of 8 MiB that every GPU
 * which loads the library holds until the process exits.  The call allocates and frees nothing and needs no fmx_ctx; it
 * works on the CURRENT device and only enqueues two kernels on cuda_stream (no synchronisation).
 *   x, W, out   DEVICE pointers, caller-owned, 16-byte aligned; rows contiguous (ld = K, K, N)
 *   limits      1 <= M <= 128; N a multiple of 128; K a multiple of 8; round_up(M, 16) * N * 4 bytes <= 8 MiB
 *               (else FMX_E_CAPACITY / FMX_E_INVALID_ARG with a message, nothing launched)
 * Every call shares the array and finds the previous call's contents in it; nothing has to start at zero (a call writes every
 * element it reads).  Calls that OVERLAP on the GPU - different streams, concurrent graphs - race on the array: keep them on
 * one stream or order them with events. */
int fmx_row_gemm_static(const void *x, const void *W, float *out, int32_t M, int32_t N, int32_t K, void *cuda_stream);

/* Debug/test: copies the segment tables of the LAST forward to HOST arrays (synchronises).
 * Sizes: perm, inv_perm [n_req]; task_req_off, task_tok_off [n_slots+1]; cu_tok [n_req+1];
 * n_slots = fmx_task_slots().  Any pointer may be NULL. */
int fmx_debug_get_segments(fmx_ctx *ctx, int32_t *perm, int32_t *inv_perm, int32_t *task_req_off,
                           int32_t *cu_tok, int32_t *task_tok_off);
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

/* Test hooks and tuning knobs (single-kernel entry points, activation read-back, fmx_set_option) are not part of this
 * ABI: they are declared in paper_2606_09643_b200/csrc/fmx_internal.h. */

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
