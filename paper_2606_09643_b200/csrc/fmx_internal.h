/* fmx_internal.h — test hooks and tuning knobs of libfmx.  NOT part of the public C ABI (include/fmx.h): no stability
 * promise; used by the repo's tests, bench.py and profiling runs through the ctypes binding.  Every knob is state of ONE
 * context (nothing is process-global). */
#ifndef FMX_INTERNAL_H
#define FMX_INTERNAL_H

#include "fmx.h"

#ifdef __cplusplus
extern "C" {
#endif

/* The private row-tile table of the last forward (256-row CTA-pair tiles): n_tiles, n_blocks, and per block
 * (tile, task, row_lo, row_hi) into blocks[4*n_blocks] (cap entries available).  Synchronises. */
int fmx_debug_get_tiles(fmx_ctx *ctx, int32_t *n_tiles, int32_t *n_blocks, int32_t *blocks, int32_t cap);
/* Copies an activation buffer of the LAST forward to HOST (synchronises).  which:
 * 0 X fp32 [N,d] (residual, task-sorted rows)  1 Xn bf16 [N,d]  2 QKV bf16 [N,d_qkv]  3 attention out
 * bf16 [N,d_q]  4 FFN hidden bf16 [N,d_ffn]  5 U bf16 [n_blk_cap*256,192]  6 pooled feature fp32 [B,d].
 * The buffers hold what the LAST layer left there (layer L-1's norm-2 output, QKV, attention output, FFN hidden; the final
 * residual stream). */
int fmx_debug_read(fmx_ctx *ctx, int which, void *host, size_t bytes);
/* Forwards served by replaying the context's cached CUDA graph so far (FMX_OPT_GRAPH). */
long long fmx_graph_replays(fmx_ctx *ctx);

/* One GEMM through the tcgen05 kernel, C[M,N] (fp32) = A[M,K] (bf16) · W[N,K]^T (bf16);
 * N a multiple of 128, K a multiple of 8.  All DEVICE pointers. */
int fmx_debug_gemm(fmx_ctx *ctx, const void *A, const void *W, float *C, int32_t M, int32_t N, int32_t K,
                   void *cuda_stream);

/* The fused variable-length attention step (S3d) alone.  qkv DEVICE bf16
 * [n_tokens, (n_q_heads + 2 n_kv_heads) * head_dim] (q | k | v per row, requests packed back to back),
 * cu_tok HOST int32 [n_req + 1] (prefix sums of the request lengths), out DEVICE bf16
 * [n_tokens, n_q_heads * head_dim].  impl: an FMX_ATTN_* value.  Scale 1/sqrt(head_dim). */
int fmx_debug_attention(fmx_ctx *ctx, const void *qkv, void *out, const int32_t *cu_tok, int32_t n_req,
                        int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, int32_t causal, int32_t impl,
                        void *cuda_stream);

/* Tuning knobs of one context (experiments; the defaults are what bench.py measures). */
enum {
  FMX_OPT_ATTENTION_IMPL = 0,    /* FMX_ATTN_AUTO | FMX_ATTN_MMA_SYNC | FMX_ATTN_TCGEN05 (head_dim 64 / 128 only) */
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
  FMX_OPT_SHRINK_FUSED = 8,      /* the LoRA shrink runs as the first work items of the GEMM that consumes it: 0 (default) = never
                                    (separate shrink kernel), 1 = when the batch has at most one (tile, task) block per CTA pair,
                                    2 = always.  Opt-in: a pair waits for blocks computed by OTHER pairs, so every cluster of the
                                    grid must be resident at once - true only when no other kernel holds SMs of the device.  A wait
                                    that times out (~2 s) raises the device error word (fmx_poll_error); it does not trap. */
  FMX_OPT_GRAPH = 9,             /* 1 (default): fmx_forward_mixed captures a CUDA graph on the 2nd identical call (same
                                    buffers, stream, ids, lengths, registrations, options) and replays it afterwards;
                                    needs a non-default stream; 0: always plain launches */
  FMX_OPT_REVERSE = 10,          /* 1 (default): consecutive kernels of a layer walk the token rows in alternating
                                    directions, so each starts on the rows its producer wrote last (still in L2) */
  FMX_OPT_EXPAND_WIDE = 11,      /* 1 (default): a 256-wide tile whose two chunks share a weight source runs its LoRA
                                    expand as one N = 256 step per block (U loaded once) instead of two N = 128 steps */
  FMX_OPT_DEEP_PIPE = 12,        /* 1 (default): fp32-output GEMMs (residual, embed) run with one more smem pipeline stage
                                    and a single epilogue staging buffer per warpgroup */
  FMX_OPT_DECODE_FORK = 13,      /* 1 (default): in a decode iteration the row-wise LoRA kernels of a projection run on the
                                    context's auxiliary stream beside the projection GEMM (both are latency-bound) and join
                                    before the reduction; set 0 when the serving stream belongs to an SM partition */
  FMX_OPT_DECODE_ROWGEMM = 14,   /* 1 (default): decode iterations of <= 128 rows run their projections on the lean mma.sync
                                    kernel (row_gemm.cuh); 0 = the pair GEMM in partial-output mode */
  FMX_OPT_EMBED_SMALL = 15,      /* 1 (default): patch embeddings with patch_dim <= 8 run on a CUDA-core kernel; 0 = the GEMM */
  FMX_OPT_PDL = 2                /* programmatic dependent launch of the forward's kernels:
                                    0 = off, 1 = always, 2 (default) = only for batches of <= 4096 token rows */
};
enum { FMX_ATTN_AUTO = 0, FMX_ATTN_MMA_SYNC = 1, FMX_ATTN_TCGEN05 = 2 };
int fmx_set_option(fmx_ctx *ctx, int32_t option, int32_t value);

#ifdef __cplusplus
}
#endif
#endif /* FMX_INTERNAL_H */
