// libfmx host runtime: context, backbone/task registry, LoRA slab arena, workspace carving and
// the launch sequence of fmx_forward_mixed.  All compute runs in the kernels of
// gemm.cuh / attention.cuh / kernels.cuh; there is no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <mutex>
#include <vector>

#include "attention.cuh"
#include "attention_pair64.cuh"
#include "attention_fa.cuh"
#include "common.h"
#include "fmx.h"
#include "fmx_internal.h"
#include "gemm.cuh"
#include "kernels.cuh"
#include "pair_gemm.cuh"
#include "row_gemm.cuh"

using namespace fmx;
typedef __nv_bfloat16 bf16;

#define CU_OK(expr)                                                                                   \
  do {                                                                                                \
    cudaError_t _e = (expr);                                                                          \
    if (_e != cudaSuccess)                                                                            \
      return fmx_fail(FMX_E_CUDA, "%s failed: %s (%d) at %s:%d", #expr, cudaGetErrorString(_e), (int)_e, __FILE__, __LINE__); \
  } while (0)

namespace {

enum Family { F_SORT = 0, F_EMBED, F_NORM, F_SHRINK, F_GEMM_QKV, F_ATTN, F_GEMM_O, F_GEMM_FFN_IN, F_GEMM_FFN_OUT,
              F_ROPE, F_POOL, F_HEAD };
const char *kFamilyNames[FMX_N_FAMILIES] = {"task_sort", "embed", "norm", "lora_shrink", "gemm_qkv", "attention",
                                            "gemm_o", "gemm_ffn_in", "gemm_ffn_out", "rope", "final_pool", "head"};

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TaskRec {
  bool live = false;
  unsigned long long freed_seq = 0;       // retirement after which this slot's device-table entries may be rewritten
  int bb = -1;
  int coff = 0, rpad = 0;                 // slab columns [coff, coff + rpad)
  unsigned char trpad[7] = {0};
  float scale[7] = {0};
  int head_kind = 0, head_out = 0, head_hidden = 0;   // head_hidden > 0: MLP head, head_W is [head_hidden, d_feat]
  bf16 *head_W = nullptr, *head_b = nullptr;   // library-owned copies
  bf16 *head_W2 = nullptr, *head_b2 = nullptr; // MLP heads: [head_out, head_hidden], [head_out]
  int enc_channels = 0;                        // per-task input encoder (channel combiner), 0 / 1 = none
  bf16 *enc_W = nullptr, *enc_b = nullptr;     // [enc_channels], [1]
};

struct Backbone {
  fmx_backbone_desc d;
  // deep copies of the caller's per-layer pointer arrays
  std::vector<const void *> norm1_g, norm1_b, Wq, Wk, Wv, Wo, bq, bk, bv, bo, norm2_g, norm2_b, Wup, Wgate, Wdown, bup, bgate, bdown;
  int d_q = 0, d_kv = 0, d_qkv = 0;
  int Kp = 0;                              // padded patch_dim
  bf16 *embed_Wpad = nullptr;              // [d, Kp]
  float *posb = nullptr;                   // [n_pos, d]
  float2 *rope_cs = nullptr;               // [max_seq, dh/2]
  float2 *rope_cs_t = nullptr;             // [dh/2, max_seq] (the fused-RoPE GEMM epilogue reads this one)
  float *relb = nullptr;                   // relative-position bias by distance: [n_q_heads, relb_ld] fp32, times log2(e); index (key - query) + relb_off;
  int relb_ld = 0, relb_off = 0;           //   padded by 128 / 127 zeros so that a tile's padding rows / keys index inside the table
  // weight maps, [0] = box {64,128} (pair tile 256x256: one CTA loads a whole chunk), [1] = box {64,64} (256x128 tiles)
  std::vector<CUtensorMap> mWq[2], mWk[2], mWv[2], mWo[2], mWup[2], mWgate[2], mWdown[2];
  CUtensorMap mEmbedW[2];
  // language-model head for token decode (NEXT-3): caller-owned bf16 [lm_vocab, d_model]
  const bf16 *lm_head = nullptr;
  int lm_vocab = 0;
  CUtensorMap mLm[2];
  // LoRA slabs
  int Rcap = 0;
  std::vector<unsigned char> col_used;     // units of 16 columns
  std::vector<unsigned long long> col_freed_seq;   // retirement after which a freed unit may be rewritten
  bf16 *slabA[7] = {nullptr};              // per target: [L][Rcap, d_in]
  bf16 *slabB[7] = {nullptr};              // per target: [L][d_out, Rcap]
  bf16 *slabBt[7] = {nullptr};             // decoder backbones only (row_bt): the same B, rank-major [L][Rcap, d_out] - a task's rank rows are
                                           //   contiguous, which is what the row-wise expand of a decode iteration streams
  bool row_bt = false;
  std::vector<CUtensorMap> mA[7], mB[7];   // per target, per layer
  int n_adapters[7] = {0};                 // live adapters per target
  int din[7], dout[7];
};

struct ProfEvent { int family; cudaEvent_t e0, e1; };

// Tuning state of ONE context (fmx_set_option, csrc/fmx_internal.h); nothing tunable lives at file scope.
struct Opts {
  int pdl = 2;            // programmatic dependent launch: 0 off, 1 always, 2 = only for batches of <= kPdlAutoRows token rows
  int shrink_stages = 5;
  int half_tiles = 1;
  int deep_pipe = 1;
  int expand_wide = 1;
  int rope_fused = 1;
  int head_tiled = 2;     // FLATTEN heads: 0 = one warp per output, 1 = CUDA-core 4 x 4 tiles, 2 = mma.sync 16 x 32 tiles
  int shrink_fused = 0;   // 1 / 2: the LoRA shrink runs as the first work items of the GEMM that consumes it (see pair_gemm.cuh);
                          // opt-in: it needs every CTA pair of the grid resident at once, i.e. the GPU to itself
  int reverse = 1;        // consecutive kernels of a layer walk the rows in alternating directions (L2 reuse)
  int attn_short = 2;     // 0: generic kernel, 1: pipelined mma.sync kernel, 2: tcgen05 head-pair kernel where it applies
  int graph = 1;
  int attn_impl = FMX_ATTN_AUTO;
  int embed_small = 1;    // PATCH_LINEAR with patch_dim <= 8: CUDA-core embed kernel instead of the one-k-block GEMM
  int decode_rowgemm = 1; // decode iterations of <= 128 rows: projections on the lean mma.sync kernel (row_gemm.cuh) instead of the pair GEMM
  int decode_fork = 1;    // decode iterations: row-wise LoRA kernels on the auxiliary stream beside the projection GEMM
};

// A launch target: the stream and whether the launch carries the programmatic-stream-serialization attribute.
struct Strm { cudaStream_t s; int pdl; };

}  // namespace

struct BatchShape {
  long long N = 0;
  int max_len = 0, max_out = 0, max_hidden = 0, max_out2 = 0, max_out_flat = 0, n_blk = 0;
  bool any_flat = false, any_pooled = false, any_dense = false;
  int max_out_dense = 0;
  bool operator==(const BatchShape &o) const {
    return N == o.N && max_len == o.max_len && max_out == o.max_out && max_hidden == o.max_hidden && max_out2 == o.max_out2 &&
           max_out_flat == o.max_out_flat && any_flat == o.any_flat && any_pooled == o.any_pooled && any_dense == o.any_dense &&
           max_out_dense == o.max_out_dense;
  }
};

struct fmx_ctx {
  int device = 0, sm_count = 0;
  bool pairs_resident = false;             // sm_count / 2 clusters of the pair GEMM fit the device at once (fused shrink needs it)
  EncodeTiledFn encode = nullptr;
  std::vector<std::unique_ptr<Backbone>> bbs;
  std::vector<TaskRec> tasks;              // slot = task id
  int n_slots = 0;
  // device task tables (FMX_MAX_TASKS entries)
  int *d_task_coff = nullptr, *d_task_head_kind = nullptr, *d_task_head_out = nullptr;
  unsigned char *d_task_trpad = nullptr;
  float *d_task_scale = nullptr;
  const bf16 **d_task_head_W = nullptr, **d_task_head_b = nullptr, **d_task_head_W2 = nullptr, **d_task_head_b2 = nullptr;
  int *d_task_head_w1 = nullptr;           // first-layer width of the head (= head_out for linear heads)
  int *d_task_enc_ch = nullptr;            // input-encoder channels by task
  const bf16 **d_task_enc_W = nullptr, **d_task_enc_b = nullptr;
  // pinned staging for ids / lengths: a ring (a slot is rewritten only after the copy that read it has run)
  static constexpr int kStageSlots = 4;
  int *h_stage = nullptr;                  // [kStageSlots][4 * FMX_MAX_REQUESTS]: ids, lengths, cache slots, cache positions
  cudaEvent_t stage_ev[kStageSlots] = {nullptr, nullptr, nullptr, nullptr};
  bool stage_used[kStageSlots] = {false, false, false, false};
  int stage_next = 0;
  // CUDA-graph cache of the forward (FMX_OPT_GRAPH): keyed by buffers + BatchShape, not by the ids (see forward_cached)
  struct CallKey {
    int bb = -1, B = 0; const void *inputs = nullptr; float *outputs = nullptr; void *workspace = nullptr; size_t ws_bytes = 0;
    cudaStream_t stream = nullptr; unsigned long long gen = 0; BatchShape shape; bool fuse = false;
    const void *kv_cache = nullptr, *scores = nullptr, *next_tokens = nullptr; int kv_mode = 0, n_slots = 0;   // 0 plain, 1 prefill, 2 decode
    bool operator==(const CallKey &o) const {
      return bb == o.bb && B == o.B && inputs == o.inputs && outputs == o.outputs && workspace == o.workspace && ws_bytes == o.ws_bytes &&
             stream == o.stream && gen == o.gen && shape == o.shape && fuse == o.fuse && kv_cache == o.kv_cache && scores == o.scores &&
             next_tokens == o.next_tokens && kv_mode == o.kv_mode && n_slots == o.n_slots;
    }
  };
  // registration runs on its own non-blocking stream: adding a task never waits for (or stalls) forwards in flight
  cudaStream_t side = nullptr;
  // retirement stream: frees of what forwards in flight may still read happen here, after those forwards (see retire())
  cudaStream_t side2 = nullptr;
  cudaEvent_t side_ev = nullptr, retire_ev = nullptr;
  cudaStream_t aux = nullptr;              // decode iterations fork the row-wise LoRA kernels onto this stream (FMX_OPT_DECODE_FORK)
  cudaEvent_t fork_ev = nullptr, join_ev = nullptr;
  unsigned long long retire_seq = 0, retire_done = 0;   // retirements issued / known complete
  struct TaskStage { int coff, head_kind, head_out, w1, enc_ch; unsigned char trpad[8]; float scale[7]; const void *ptr[6]; };
  TaskStage *h_task_stage = nullptr;       // pinned
  Opts o;
  unsigned long long config_gen = 0;       // bumped by every registration change and option change
  CallKey last_key, graph_key;
  cudaGraphExec_t graph_exec = nullptr;
  int graph_launches = 0;                  // kernels inside the cached graph
  unsigned long long graph_replays = 0;
  // Where forwards are in flight: the end-of-forward event of the latest forward on each serving stream seen (a few
  // entries, least recently used replaced).  fmx_unregister_task and a slab growth make the registration stream wait for
  // these events before it frees or reuses what those forwards may still read - the host never waits (NEXT-2).
  static constexpr int kServe = 8;
  struct Serving { cudaStream_t stream = nullptr; cudaEvent_t ev = nullptr; bool used = false; unsigned long long tick = 0; };
  Serving serving[kServe];
  unsigned long long serve_tick = 0;
  // device-side error word (mapped pinned host memory): bit 0 = a TOKEN_IDS request carried an id outside [0, vocab)
  unsigned *h_err = nullptr, *d_err = nullptr;
  // last forward (debug)
  SegTables last_t{};
  int last_B = 0, last_T = 0, last_n_tiles = 0, last_launches = 0;
  cudaStream_t last_stream = nullptr;
  void *last_buf[7] = {nullptr}; size_t last_buf_bytes[7] = {0};
  // profiling
  bool prof_on = false;
  uint32_t prof_mask = 0xFFFFFFFFu;        // families that get events while prof_on
  std::vector<ProfEvent> prof;
  std::vector<cudaEvent_t> ev_pool;        // recycled events
  int *d_dbg_cu = nullptr;                 // fmx_debug_attention's device copy of cu_tok [FMX_MAX_REQUESTS + 1]
  std::mutex mu;
};

namespace {

int encode_2d(fmx_ctx *c, CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, uint64_t ld_elems,
              uint32_t box_rows, bool f32 = false) {
  const uint64_t esz = f32 ? 4 : 2;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {ld_elems * esz};
  cuuint32_t box[2] = {f32 ? 32u : 64u, box_rows};          // 128-byte inner box = one swizzle row
  cuuint32_t estr[2] = {1, 1};
  if ((reinterpret_cast<uintptr_t>(base) & 15) || (strides[0] & 15))
    return fmx_fail(FMX_E_INVALID_ARG, "tensor map: base %p / row stride %llu B not 16-byte aligned", base,
                    (unsigned long long)strides[0]);
  CUresult r = c->encode(m, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fmx_fail(FMX_E_CUDA, "cuTensorMapEncodeTiled failed (%d) rows=%llu cols=%llu ld=%llu", (int)r,
                                         (unsigned long long)rows, (unsigned long long)cols, (unsigned long long)ld_elems);
  return FMX_OK;
}

void target_dims(const fmx_backbone_desc &d, int tg, int &din, int &dout) {
  const int dq = d.n_q_heads * d.head_dim, dkv = d.n_kv_heads * d.head_dim;
  switch (tg) {
    case FMX_TGT_Q: din = d.d_model; dout = dq; break;
    case FMX_TGT_K: case FMX_TGT_V: din = d.d_model; dout = dkv; break;
    case FMX_TGT_O: din = dq; dout = d.d_model; break;
    case FMX_TGT_GATE: case FMX_TGT_UP: din = d.d_model; dout = d.d_ffn; break;
    default: din = d.d_ffn; dout = d.d_model; break;
  }
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---------------------------------------------------------------- workspace layout
struct Workspace {
  SegTables t{};
  float *X = nullptr, *feat = nullptr;
  bf16 *Xn = nullptr, *QKV = nullptr, *AttnO = nullptr, *Hid = nullptr, *U = nullptr;
  unsigned *u_flag = nullptr;            // completion counter of the fused-shrink items
  float *head_hid = nullptr;             // hidden activations of MLP heads [B, kMaxHeadHidden]
  float *head_part = nullptr;            // K-chunk partials of the tensor-core FLATTEN head: kHeadPartFloats per request
  size_t head_part_floats = 0;
  // token decode (NEXT-3): cache slot / position per request (original order) and per token row; LM-head operands
  int *slots = nullptr, *pos0 = nullptr, *row_slot = nullptr, *row_cpos = nullptr;
  bf16 *Fl = nullptr;                    // [B, d] final-normed last rows, sorted request order
  float *lm_scores = nullptr;            // [B, lm_vocab] sorted request order
  float *splitk = nullptr;               // partials of the small-M (decode) projections: [k_split, 256, N] fp32, k_split * N <= splitk_cols
  float *delta = nullptr;                // row-wise LoRA deltas of a projection group: [256, proj_max_n] fp32
  float *dec_part = nullptr;             // decode attention: per (request, q head, chunk) partial (o, m, l)
  unsigned *dec_cnt = nullptr;           // decode attention: chunks finished per (request, KV head)
  float *rowu = nullptr;                 // row-wise shrink partial sums [nkc, 256, 3, 64] fp32 (nkc = 512-column chunks of the widest input)
  int n_tiles = 0, n_blk_cap = 0;
  size_t bytes = 0;
};

// The head scratch is part of the caller's workspace (no allocation inside the forward): an MLP head's hidden layer is at
// most kMaxHeadHidden wide (fmx_register_task enforces it); the FLATTEN-head partials get a fixed budget per request and
// the launcher picks the K split that fits it.
constexpr int kMaxHeadHidden = 4096;
constexpr int kSplitMax = 16;            // most K splits of a small-M projection
// widest projection output of a backbone (SwiGLU: gate and up interleaved), and the columns of the split-K partial buffer:
// k_split * N <= (CTA pairs) * 256 by construction, or N itself when the projection is not split
int proj_max_n(const Backbone &bb) { return std::max(std::max(bb.d_qkv, bb.d.d_model), (bb.d.act == FMX_ACT_SWIGLU ? 2 : 1) * bb.d.d_ffn); }
size_t splitk_cols(const Backbone &bb) { return (size_t)std::max(80 * 256, proj_max_n(bb)); }
constexpr size_t kHeadPartFloats = 2048;
int row_shrink_chunks(int K) { return (K + kRowShrinkK - 1) / kRowShrinkK; }
// Decode attention splits a sequence's cached positions into chunks of kc_keys (a property of the backbone: the longest sequence
// has at most 16 chunks), one CTA each.
int dec_chunk_keys(int max_seq) { int kc = kDecKeys; while (kc * 16 < max_seq) kc *= 2; return kc; }
int dec_chunks_cap(int max_seq) { const int kc = dec_chunk_keys(max_seq); return (max_seq + kc - 1) / kc; }
Workspace carve(const Backbone &bb, void *base, int B, long long N, int T) {
  Workspace w;
  uint8_t *p = static_cast<uint8_t *>(base);
  size_t off = 0;
  auto take = [&](size_t bytes) { void *r = p ? p + off : nullptr; off = align_up(off + bytes, 1024); return r; };
  w.n_tiles = (int)((N + kPairRows - 1) / kPairRows);        // 256-row pair tiles
  w.n_blk_cap = w.n_tiles + std::min(T, B);
  const fmx_backbone_desc &d = bb.d;
  w.t.task_ids = (int *)take(sizeof(int) * B);
  w.t.lengths = (int *)take(sizeof(int) * B);
  w.t.perm = (int *)take(sizeof(int) * B);
  w.t.inv_perm = (int *)take(sizeof(int) * B);
  w.t.task_sorted = (int *)take(sizeof(int) * B);
  w.t.task_req_off = (int *)take(sizeof(int) * (T + 1));
  w.t.task_tok_off = (int *)take(sizeof(int) * (T + 1));
  w.t.cu_tok = (int *)take(sizeof(int) * (B + 1));
  w.t.in_off = (long long *)take(sizeof(long long) * (B + 1));
  w.t.out_off = (long long *)take(sizeof(long long) * (B + 1));
  w.t.tile_blk_off = (int *)take(sizeof(int) * (w.n_tiles + 1));
  w.t.blk_tile = (int *)take(sizeof(int) * w.n_blk_cap);
  w.t.blk_task = (int *)take(sizeof(int) * w.n_blk_cap);
  w.t.blk_lo = (int *)take(sizeof(int) * w.n_blk_cap);
  w.t.blk_hi = (int *)take(sizeof(int) * w.n_blk_cap);
  w.t.n_blk = (int *)take(sizeof(int));
  w.t.row_req = (int *)take(sizeof(int) * N);
  w.t.row_pos = (int *)take(sizeof(int) * N);
  w.X = (float *)take(sizeof(float) * N * d.d_model);
  w.Xn = (bf16 *)take(sizeof(bf16) * N * d.d_model);
  w.QKV = (bf16 *)take(sizeof(bf16) * N * bb.d_qkv);
  w.AttnO = (bf16 *)take(sizeof(bf16) * N * bb.d_q);
  w.Hid = (bf16 *)take(sizeof(bf16) * N * std::max(d.d_ffn, bb.Kp));     // also the patch-pack buffer
  w.U = (bf16 *)take(sizeof(bf16) * (size_t)w.n_blk_cap * kPairRows * 192);
  w.feat = (float *)take(sizeof(float) * (size_t)B * d.d_model);
  w.u_flag = (unsigned *)take(sizeof(unsigned));
  w.head_hid = (float *)take(sizeof(float) * (size_t)B * kMaxHeadHidden);
  w.head_part_floats = (size_t)((B + 15) / 16) * 16 * kHeadPartFloats;
  w.head_part = (float *)take(sizeof(float) * w.head_part_floats);
  w.slots = (int *)take(sizeof(int) * B);
  w.pos0 = (int *)take(sizeof(int) * B);
  w.row_slot = (int *)take(sizeof(int) * N);
  w.row_cpos = (int *)take(sizeof(int) * N);
  if (bb.lm_head) {
    w.Fl = (bf16 *)take(sizeof(bf16) * (size_t)B * d.d_model);
    w.lm_scores = (float *)take(sizeof(float) * (size_t)B * bb.lm_vocab);
    w.splitk = (float *)take(sizeof(float) * kPairRows * splitk_cols(bb));
    w.delta = (float *)take(sizeof(float) * (size_t)kPairRows * proj_max_n(bb));
    w.dec_part = (float *)take(sizeof(float) * (size_t)B * d.n_q_heads * dec_chunks_cap(d.max_seq) * (d.head_dim + 2));
    w.dec_cnt = (unsigned *)take(sizeof(unsigned) * (size_t)B * d.n_kv_heads);
    w.rowu = (float *)take(sizeof(float) * (size_t)row_shrink_chunks(std::max({d.d_model, d.d_ffn, bb.d_q})) * kPairRows * 3 * 64);
  }
  w.bytes = off;
  return w;
}

// ---------------------------------------------------------------- launch bookkeeping
struct Launcher {
  fmx_ctx *c;
  cudaStream_t s;
  int count = 0;
  bool rec = false;
  int get_event(cudaEvent_t *e) {
    if (!c->ev_pool.empty()) { *e = c->ev_pool.back(); c->ev_pool.pop_back(); return FMX_OK; }
    CU_OK(cudaEventCreate(e));
    return FMX_OK;
  }
  int begin(int family) {
    ++count;
    rec = c->prof_on && ((c->prof_mask >> family) & 1u);
    if (rec) {
      ProfEvent pe{family, nullptr, nullptr};
      if (int e = get_event(&pe.e0)) return e;
      if (int e = get_event(&pe.e1)) return e;
      CU_OK(cudaEventRecord(pe.e0, s));
      c->prof.push_back(pe);
    }
    return FMX_OK;
  }
  int end() {
    CU_OK(cudaGetLastError());
    if (rec) CU_OK(cudaEventRecord(c->prof.back().e1, s));
    return FMX_OK;
  }
};
#define LAUNCH(L, family, ...)                    \
  do {                                            \
    if (int _e = (L).begin(family)) return _e;    \
    __VA_ARGS__;                                  \
    if (int _e = (L).end()) return _e;            \
  } while (0)


// Every forward-path kernel is launched with the programmatic-stream-serialization attribute (PDL, see ptx.cuh):
// the next kernel's CTAs become resident and run their prologue while this one drains; each kernel blocks in
// griddepcontrol.wait before it touches global memory.  FMX_OPT_PDL: 0 = plain stream order, 1 = always, 2 (default) =
// only for small batches (<= kPdlAutoRows token rows), where the step is bound by launch latency: measured on B200 it
// takes cfg1 from 0.208 to 0.163 ms per forward and is neutral to slightly negative (< 1 %) on the large configs.
constexpr int kPdlAutoRows = 4096;
template <typename... KArgs, typename... Args>
void launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Strm st, Args &&...args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st.s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = st.pdl;
  cfg.attrs = at; cfg.numAttrs = 1;
  cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <int kVec>
void launch_norm(Strm s, const float *X, bf16 *Y, const bf16 *g, const bf16 *b, int N, float eps, int rms, int rev) {
  launch_k(norm_kernel<kVec>, (N + 7) / 8, 256, 0, s, X, Y, g, b, N, eps, rms, rev);
}
bool dispatch_norm(Strm s, int d, const float *X, bf16 *Y, const bf16 *g, const bf16 *b, int N, float eps, int rms, int rev) {
  switch (d / 128) {
    case 1: launch_norm<1>(s, X, Y, g, b, N, eps, rms, rev); return true;
    case 2: launch_norm<2>(s, X, Y, g, b, N, eps, rms, rev); return true;
    case 4: launch_norm<4>(s, X, Y, g, b, N, eps, rms, rev); return true;
    case 6: launch_norm<6>(s, X, Y, g, b, N, eps, rms, rev); return true;
    case 8: launch_norm<8>(s, X, Y, g, b, N, eps, rms, rev); return true;
    case 12: launch_norm<12>(s, X, Y, g, b, N, eps, rms, rev); return true;
    case 16: launch_norm<16>(s, X, Y, g, b, N, eps, rms, rev); return true;
  }
  return false;
}
bool dispatch_pool(Strm s, int d, int B, const PoolArgs &a) {
  switch (d / 128) {
    case 1: launch_k(final_pool_kernel<1>, B, 128, 0, s, a); return true;
    case 2: launch_k(final_pool_kernel<2>, B, 128, 0, s, a); return true;
    case 4: launch_k(final_pool_kernel<4>, B, 128, 0, s, a); return true;
    case 6: launch_k(final_pool_kernel<6>, B, 128, 0, s, a); return true;
    case 8: launch_k(final_pool_kernel<8>, B, 128, 0, s, a); return true;
    case 12: launch_k(final_pool_kernel<12>, B, 128, 0, s, a); return true;
    case 16: launch_k(final_pool_kernel<16>, B, 128, 0, s, a); return true;
  }
  return false;
}
bool norm_dim_supported(int d) {
  const int v = d / 128;
  return d % 128 == 0 && (v == 1 || v == 2 || v == 4 || v == 6 || v == 8 || v == 12 || v == 16);
}

void launch_shrink(fmx_ctx *c, Strm s, const GemmParams &p) {
  if (c->o.shrink_stages == 4) launch_k((shrink_kernel<4, 3>), c->sm_count, kGemmThreads, (shrink_smem_bytes<4, 3>()), s, p);
  else if (p.n_tg == 1) launch_k((shrink_kernel<8, 1>), c->sm_count, kGemmThreads, (shrink_smem_bytes<8, 1>()), s, p);
  else if (p.n_tg == 2) launch_k((shrink_kernel<6, 2>), c->sm_count, kGemmThreads, (shrink_smem_bytes<6, 2>()), s, p);
  else launch_k((shrink_kernel<5, 3>), c->sm_count, kGemmThreads, (shrink_smem_bytes<5, 3>()), s, p);
}

// Pair tiles 256 x 256 when the chunk count is even, else 256 x 128; one cluster of 2 CTAs per SM pair.
bool pair_wide(const PairGemmParams &p) { return p.n_chunks % 2 == 0; }
void launch_pair_gemm(fmx_ctx *c, Strm s, const PairGemmParams &p) {
  const int pairs = c->sm_count / 2;
  // fp32-output modes (residual reduce-add, embed) take the deep variant: one more pipeline stage, one staging buffer
  const bool deep = c->o.deep_pipe && (p.mode == GM_RESID_F32 || p.mode == GM_EMBED_F32 || p.mode == GM_OUT_F32 || p.k_split > 0);
  if (pair_wide(p)) {
    const int tiles = p.n_ptiles * (p.n_chunks / 2);
    // Wave quantisation: when the last wave would hold at most half as many tiles as there are pairs, its tiles are cut
    // into 256 x 128 halves so that it lasts half a tile time (cfg2 O / FFN-out: 256 tiles on 74 pairs, 4 -> 3.5 waves).
    PairGemmParams q = p;
    q.expand_wide = c->o.expand_wide;
    const int rem = tiles % pairs;
    q.n_full = (c->o.half_tiles && p.k_split == 0 && p.mode != GM_OUT_BF16_SWIGLU && !p.rope_cs && tiles > pairs && rem > 0 && 2 * rem <= pairs) ? tiles - rem : -1;
    const int items = p.k_split > 0 ? tiles * p.k_split : (q.n_full >= 0 ? q.n_full + 2 * rem : tiles);
    const int grid = 2 * (p.n_sh > 0 ? pairs : std::min(items, pairs));
    if (deep) launch_k((pair_gemm_kernel<256, true>), grid, kGemmThreads, (pair_smem_bytes<256, true>()), s, q);
    else launch_k((pair_gemm_kernel<256, false>), grid, kGemmThreads, (pair_smem_bytes<256, false>()), s, q);
  } else {
    const int tiles = p.n_ptiles * p.n_chunks * std::max(p.k_split, 1);
    const int grid = 2 * (p.n_sh > 0 ? pairs : std::min(tiles, pairs));
    if (deep) launch_k((pair_gemm_kernel<128, true>), grid, kGemmThreads, (pair_smem_bytes<128, true>()), s, p);
    else launch_k((pair_gemm_kernel<128, false>), grid, kGemmThreads, (pair_smem_bytes<128, false>()), s, p);
  }
}

// Every request <= 64 tokens: the pipelined single-tile kernel (4 CTAs per SM, each walking a strided item list).
bool attn_pair64_ok(const Opts &o, int dh, int n_q_heads, int max_len) { return o.attn_short == 2 && dh == 64 && n_q_heads % 2 == 0 && max_len <= 64; }
void launch_attention_pair64(Strm s, int sm_count, const AttnPairArgs &a) {
  const int items = a.n_req * (a.n_q_heads / 2);
  const int grid = std::min(sm_count, (items + kP64Lanes - 1) / kP64Lanes);
  launch_k(attention_pair64_kernel, grid, kP64Threads, attn_pair64_smem_bytes(), s, a);
}
void launch_attention_short(Strm s, int sm_count, int dh, int n_req, const AttnArgs &a) {
  const int items = n_req * a.n_q_heads;
  const int grid = std::min(items, sm_count * 4);
  if (dh == 32) launch_k(attention_short_kernel<32>, grid, kAttnThreads, attn_short_smem_bytes<32>(), s, a, n_req);
  else if (dh == 64) launch_k(attention_short_kernel<64>, grid, kAttnThreads, attn_short_smem_bytes<64>(), s, a, n_req);
  else launch_k(attention_short_kernel<128>, std::min(items, sm_count * 2), kAttnThreads, attn_short_smem_bytes<128>(), s, a, n_req);
}
void launch_attention(Strm s, int dh, dim3 grid, const AttnArgs &a) {
  if (dh == 32) launch_k(attention_kernel<32>, grid, kAttnThreads, attn_smem_bytes<32>(), s, a);
  else if (dh == 64) launch_k(attention_kernel<64>, grid, kAttnThreads, attn_smem_bytes<64>(), s, a);
  else launch_k(attention_kernel<128>, grid, kAttnThreads, attn_smem_bytes<128>(), s, a);
}

// The tcgen05 kernel serves head_dim 64 / 128 (a TMA box is 64 columns wide); head_dim 32 stays on mma.sync.
// Variant v: 0 = one q-tile (128 queries) per CTA, two CTAs per SM; 1 = two q-tiles per CTA sharing K/V, one CTA per SM.
// AUTO: short sequences (one KV tile per request, cfg2/cfg5's 64 tokens) are bound by per-CTA latency, where the
// lighter mma.sync kernel measured faster (47 vs 65 us per layer on cfg2); everything longer goes to tcgen05.
bool attn_use_tc(int impl, int dh, int max_len) {
  if (dh != 64 && dh != 128) return false;
  if (impl == FMX_ATTN_AUTO) return max_len > 64;
  return impl != FMX_ATTN_MMA_SYNC;
}
// head_dim 64: four light CTAs per SM (single S buffer, two-pass softmax: 80 registers); head_dim 128: TMEM (2 x 64 + 128
// columns) allows two CTAs per SM, which double-buffer S and keep a tile's 64 scores in registers.  Measured against the other
// trades (profiles/r2_02): head_dim 64 one-pass at 3 CTAs per SM 5.2 vs 3.5 ms per cfg3 step; head_dim 128 two-pass 6.7 vs 6.4 ms.
void launch_attention_tc(Strm s, int dh, int max_len, int n_heads, int B, const AttnTcArgs &a) {
  dim3 grid((max_len + kAtBQ - 1) / kAtBQ, n_heads, B);
  if (a.relb) {              // relative-position bias: the same kernels with the bias added to each score (d_h 64: 3 CTAs per SM for the registers)
    if (dh == 64) launch_k((attention_fa_kernel<64, 1, 3, false, true>), grid, kFaThreads, attn_fa_smem_bytes<64>(), s, a);
    else launch_k((attention_fa_kernel<128, 2, 2, true, true>), grid, kFaThreads, attn_fa_smem_bytes<128>(), s, a);
    return;
  }
  if (dh == 64) launch_k((attention_fa_kernel<64, 1, 4, false>), grid, kFaThreads, attn_fa_smem_bytes<64>(), s, a);
  else launch_k((attention_fa_kernel<128, 2, 2, true>), grid, kFaThreads, attn_fa_smem_bytes<128>(), s, a);
}
template <int DH, int kSBuf, int kMinB, bool kOne, bool kBias = false>
cudaError_t set_attn_fa_attr() {
  cudaError_t e = cudaFuncSetAttribute(attention_fa_kernel<DH, kSBuf, kMinB, kOne, kBias>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_fa_smem_bytes<DH>());
  // without this the driver sizes the L1/shared split for ONE block and further CTAs never become resident
  if (e == cudaSuccess) e = cudaFuncSetAttribute(attention_fa_kernel<DH, kSBuf, kMinB, kOne, kBias>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  if (e == cudaSuccess && getenv("FMX_DEBUG")) {
    int nb = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, attention_fa_kernel<DH, kSBuf, kMinB, kOne, kBias>, kFaThreads, attn_fa_smem_bytes<DH>());
    cudaFuncAttributes fa{};
    cudaFuncGetAttributes(&fa, attention_fa_kernel<DH, kSBuf, kMinB, kOne, kBias>);
    fprintf(stderr, "fmx: attention_fa<%d,%d,%d,%d>: %d B smem, %d CTA/SM, %d regs\n", DH, kSBuf, kMinB, (int)kOne, attn_fa_smem_bytes<DH>(), nb, fa.numRegs);
  }
  return e;
}

int set_kernel_attrs() {
  CU_OK((set_attn_fa_attr<64, 1, 4, false>()));
  CU_OK((set_attn_fa_attr<128, 2, 2, true>()));
  CU_OK((set_attn_fa_attr<64, 1, 3, false, true>()));
  CU_OK((set_attn_fa_attr<128, 2, 2, true, true>()));
  CU_OK((cudaFuncSetAttribute(pair_gemm_kernel<256, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, pair_smem_bytes<256, false>())));
  CU_OK((cudaFuncSetAttribute(pair_gemm_kernel<256, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, pair_smem_bytes<256, true>())));
  CU_OK((cudaFuncSetAttribute(pair_gemm_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, pair_smem_bytes<128, false>())));
  CU_OK((cudaFuncSetAttribute(pair_gemm_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, pair_smem_bytes<128, true>())));
  CU_OK((cudaFuncSetAttribute(row_gemm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, row_gemm_smem<1>())));
  CU_OK((cudaFuncSetAttribute(row_gemm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, row_gemm_smem<2>())));
  CU_OK((cudaFuncSetAttribute(row_gemm_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, row_gemm_smem<4>())));
  CU_OK((cudaFuncSetAttribute(row_gemm_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, row_gemm_smem<8>())));
  CU_OK((cudaFuncSetAttribute(decode_attention_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, decode_attention_smem<32>())));
  CU_OK((cudaFuncSetAttribute(decode_attention_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, decode_attention_smem<64>())));
  CU_OK((cudaFuncSetAttribute(decode_attention_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, decode_attention_smem<128>())));
  CU_OK((cudaFuncSetAttribute(shrink_kernel<4, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, shrink_smem_bytes<4, 3>())));
  CU_OK((cudaFuncSetAttribute(shrink_kernel<5, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, shrink_smem_bytes<5, 3>())));
  CU_OK((cudaFuncSetAttribute(shrink_kernel<6, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, shrink_smem_bytes<6, 2>())));
  CU_OK((cudaFuncSetAttribute(shrink_kernel<8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, shrink_smem_bytes<8, 1>())));
  CU_OK(cudaFuncSetAttribute(attention_pair64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_pair64_smem_bytes()));
  CU_OK(cudaFuncSetAttribute(attention_short_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_short_smem_bytes<32>()));
  CU_OK(cudaFuncSetAttribute(attention_short_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_short_smem_bytes<64>()));
  CU_OK(cudaFuncSetAttribute(attention_short_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_short_smem_bytes<128>()));
  CU_OK(cudaFuncSetAttribute(attention_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_smem_bytes<32>()));
  CU_OK(cudaFuncSetAttribute(attention_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_smem_bytes<64>()));
  CU_OK(cudaFuncSetAttribute(attention_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_smem_bytes<128>()));
  return FMX_OK;
}

std::vector<const void *> copy_ptrs(const void *const *arr, int n) {
  std::vector<const void *> v(n, nullptr);
  if (arr) for (int i = 0; i < n; ++i) v[i] = arr[i];
  return v;
}

// ---------------------------------------------------------------- LoRA slab arena
int rebuild_slab_maps(fmx_ctx *c, Backbone &bb, int tg) {
  const int L = bb.d.n_layers;
  bb.mA[tg].resize(L);
  bb.mB[tg].resize(L);
  for (int l = 0; l < L; ++l) {
    bf16 *A = bb.slabA[tg] + (size_t)l * bb.Rcap * bb.din[tg];
    bf16 *B = bb.slabB[tg] + (size_t)l * bb.dout[tg] * bb.Rcap;
    if (int e = encode_2d(c, &bb.mA[tg][l], A, bb.Rcap, bb.din[tg], bb.din[tg], 64)) return e;
    if (int e = encode_2d(c, &bb.mB[tg][l], B, bb.dout[tg], bb.Rcap, bb.Rcap, 64)) return e;
  }
  return FMX_OK;
}

// Forwards in flight may still read what an unregister or a slab growth is about to free.  The retirement stream waits
// (on the device) for the registration stream and for the latest forward of every serving stream, then frees; the host
// never waits.  Every retirement gets a sequence number; a later registration that wants to REUSE a freed task slot or
// freed slab columns makes the registration stream wait for that retirement first (wait_retired).
int retire(fmx_ctx *c, const std::vector<void *> &ptrs) {
  CU_OK(cudaEventRecord(c->side_ev, c->side));
  CU_OK(cudaStreamWaitEvent(c->side2, c->side_ev, 0));
  for (auto &sv : c->serving)
    if (sv.used) CU_OK(cudaStreamWaitEvent(c->side2, sv.ev, 0));
  for (void *q : ptrs) if (q) CU_OK(cudaFreeAsync(q, c->side2));
  CU_OK(cudaEventRecord(c->retire_ev, c->side2));
  ++c->retire_seq;
  return FMX_OK;
}
int wait_retired(fmx_ctx *c, unsigned long long seq) {
  if (seq <= c->retire_done) return FMX_OK;
  if (cudaEventQuery(c->retire_ev) == cudaSuccess) { c->retire_done = c->retire_seq; return FMX_OK; }
  cudaGetLastError();                                    // cudaErrorNotReady is not an error
  CU_OK(cudaStreamWaitEvent(c->side, c->retire_ev, 0));   // covers every earlier retirement: the stream is ordered
  return FMX_OK;
}

// Called at the end of every forward enqueued on `s` (not while capturing).
int note_forward(fmx_ctx *c, cudaStream_t s) {
  fmx_ctx::Serving *slot = nullptr;
  for (auto &sv : c->serving) if (sv.used && sv.stream == s) { slot = &sv; break; }
  if (!slot) {
    for (auto &sv : c->serving) if (!sv.used) { slot = &sv; break; }
    if (!slot) {                                        // all entries taken: the least recently used one is replaced; the
      slot = &c->serving[0];                            // retirement stream inherits its dependency first
      for (auto &sv : c->serving) if (sv.tick < slot->tick) slot = &sv;
      CU_OK(cudaStreamWaitEvent(c->side2, slot->ev, 0));
    }
    if (!slot->ev) CU_OK(cudaEventCreateWithFlags(&slot->ev, cudaEventDisableTiming));
    slot->stream = s; slot->used = true;
  }
  slot->tick = ++c->serve_tick;
  CU_OK(cudaEventRecord(slot->ev, s));
  return FMX_OK;
}

// First adapter on a target: its slabs, zero-filled, from the stream-ordered pool on the registration stream.
int alloc_slab(fmx_ctx *c, Backbone &bb, int tg) {
  const size_t L = bb.d.n_layers;
  const size_t na = L * bb.Rcap * bb.din[tg], nb = L * bb.dout[tg] * bb.Rcap;
  bf16 *A = nullptr, *B = nullptr, *Bt = nullptr;
  CU_OK(cudaMallocAsync(&A, na * sizeof(bf16), c->side));
  cudaError_t e = cudaMallocAsync(&B, nb * sizeof(bf16), c->side);
  if (e == cudaSuccess && bb.row_bt) e = cudaMallocAsync(&Bt, nb * sizeof(bf16), c->side);
  if (e != cudaSuccess) {
    cudaFreeAsync(A, c->side);
    if (B) cudaFreeAsync(B, c->side);
    return fmx_fail(FMX_E_CUDA, "register_task: LoRA slab allocation failed: %s", cudaGetErrorString(e));
  }
  CU_OK(cudaMemsetAsync(A, 0, na * sizeof(bf16), c->side));
  CU_OK(cudaMemsetAsync(B, 0, nb * sizeof(bf16), c->side));
  if (Bt) CU_OK(cudaMemsetAsync(Bt, 0, nb * sizeof(bf16), c->side));
  bb.slabA[tg] = A; bb.slabB[tg] = B; bb.slabBt[tg] = Bt;
  return rebuild_slab_maps(c, bb, tg);
}

// The arena is full: a twice as wide one is built on the registration stream (the old columns copied over) while forwards
// keep reading the old one; the descriptors switch at a forward boundary (forwards enqueued from now on take the new maps)
// and the old arena is released once the forwards that were in flight are done - no device-wide synchronisation.
int grow_slabs(fmx_ctx *c, Backbone &bb, int new_cap) {
  const size_t L = bb.d.n_layers;
  const int old = bb.Rcap;
  bf16 *nA[7] = {nullptr}, *nB[7] = {nullptr}, *nBt[7] = {nullptr};
  auto undo = [&]() {
    for (int tg = 0; tg < 7; ++tg) { if (nA[tg]) cudaFreeAsync(nA[tg], c->side); if (nB[tg]) cudaFreeAsync(nB[tg], c->side); if (nBt[tg]) cudaFreeAsync(nBt[tg], c->side); }
  };
  for (int tg = 0; tg < 7; ++tg) {
    if (!bb.slabA[tg]) continue;
    const size_t na = L * new_cap * bb.din[tg], nb = L * bb.dout[tg] * (size_t)new_cap;
    cudaError_t e = cudaMallocAsync(&nA[tg], na * sizeof(bf16), c->side);
    if (e == cudaSuccess) e = cudaMallocAsync(&nB[tg], nb * sizeof(bf16), c->side);
    if (e == cudaSuccess) e = cudaMemsetAsync(nA[tg], 0, na * sizeof(bf16), c->side);
    if (e == cudaSuccess) e = cudaMemsetAsync(nB[tg], 0, nb * sizeof(bf16), c->side);
    if (e == cudaSuccess)
      e = cudaMemcpy2DAsync(nA[tg], (size_t)new_cap * bb.din[tg] * sizeof(bf16), bb.slabA[tg], (size_t)old * bb.din[tg] * sizeof(bf16),
                            (size_t)old * bb.din[tg] * sizeof(bf16), L, cudaMemcpyDeviceToDevice, c->side);
    if (e == cudaSuccess)
      e = cudaMemcpy2DAsync(nB[tg], (size_t)new_cap * sizeof(bf16), bb.slabB[tg], (size_t)old * sizeof(bf16), (size_t)old * sizeof(bf16),
                            L * bb.dout[tg], cudaMemcpyDeviceToDevice, c->side);
    if (e == cudaSuccess && bb.slabBt[tg]) {
      e = cudaMallocAsync(&nBt[tg], nb * sizeof(bf16), c->side);
      if (e == cudaSuccess) e = cudaMemsetAsync(nBt[tg], 0, nb * sizeof(bf16), c->side);
      if (e == cudaSuccess)
        e = cudaMemcpy2DAsync(nBt[tg], (size_t)new_cap * bb.dout[tg] * sizeof(bf16), bb.slabBt[tg], (size_t)old * bb.dout[tg] * sizeof(bf16),
                              (size_t)old * bb.dout[tg] * sizeof(bf16), L, cudaMemcpyDeviceToDevice, c->side);
    }
    if (e != cudaSuccess) { undo(); return fmx_fail(FMX_E_CUDA, "register_task: growing the LoRA slabs to %d columns failed: %s", new_cap, cudaGetErrorString(e)); }
  }
  // commit: nothing below fails short of a broken context
  std::vector<void *> old_slabs;
  for (int tg = 0; tg < 7; ++tg) if (bb.slabA[tg]) { old_slabs.push_back(bb.slabA[tg]); old_slabs.push_back(bb.slabB[tg]); old_slabs.push_back(bb.slabBt[tg]); }
  if (int e = retire(c, old_slabs)) { undo(); return e; }
  for (int tg = 0; tg < 7; ++tg) {
    if (!bb.slabA[tg]) continue;
    bb.slabA[tg] = nA[tg];
    bb.slabB[tg] = nB[tg];
    bb.slabBt[tg] = nBt[tg];
  }
  bb.Rcap = new_cap;
  bb.col_used.resize(new_cap / 16, 0);
  bb.col_freed_seq.resize(new_cap / 16, 0);
  for (int tg = 0; tg < 7; ++tg)
    if (bb.slabA[tg]) if (int e = rebuild_slab_maps(c, bb, tg)) return e;
  return FMX_OK;
}

int find_columns(const Backbone &bb, int units) {        // first fit, units of 16 columns
  const int n = (int)bb.col_used.size();
  for (int i = 0; i + units <= n; ++i) {
    int j = 0;
    while (j < units && !bb.col_used[i + j]) ++j;
    if (j == units) return i;
    i += j;
  }
  return -1;
}

int upload_task_tables(fmx_ctx *c, int t, const TaskRec &r) {
  // One task's entries of the device tables, through a pinned staging struct on the registration stream (no legacy-stream
  // cudaMemcpy: that would wait for forwards running on the default stream).  The caller synchronises c->side afterwards.
  fmx_ctx::TaskStage &h = *c->h_task_stage;                // free: every registration ends with a synchronise of c->side
  h.coff = r.coff; h.head_kind = r.head_kind; h.head_out = r.head_out; h.w1 = r.head_hidden > 0 ? r.head_hidden : r.head_out;
  h.enc_ch = r.enc_channels;
  memcpy(h.trpad, r.trpad, 7); memcpy(h.scale, r.scale, sizeof(r.scale));
  h.ptr[0] = r.head_W; h.ptr[1] = r.head_b; h.ptr[2] = r.head_W2; h.ptr[3] = r.head_b2; h.ptr[4] = r.enc_W; h.ptr[5] = r.enc_b;
  auto put = [&](void *dst, const void *src, size_t n) { return cudaMemcpyAsync(dst, src, n, cudaMemcpyHostToDevice, c->side); };
  CU_OK(put(c->d_task_coff + t, &h.coff, sizeof(int)));
  CU_OK(put(c->d_task_trpad + t * 7, h.trpad, 7));
  CU_OK(put(c->d_task_scale + t * 7, h.scale, 7 * sizeof(float)));
  CU_OK(put(c->d_task_head_kind + t, &h.head_kind, sizeof(int)));
  CU_OK(put(c->d_task_head_out + t, &h.head_out, sizeof(int)));
  CU_OK(put(c->d_task_head_w1 + t, &h.w1, sizeof(int)));
  CU_OK(put(c->d_task_enc_ch + t, &h.enc_ch, sizeof(int)));
  CU_OK(put(c->d_task_head_W + t, &h.ptr[0], sizeof(void *)));
  CU_OK(put(c->d_task_head_b + t, &h.ptr[1], sizeof(void *)));
  CU_OK(put(c->d_task_head_W2 + t, &h.ptr[2], sizeof(void *)));
  CU_OK(put(c->d_task_head_b2 + t, &h.ptr[3], sizeof(void *)));
  CU_OK(put(c->d_task_enc_W + t, &h.ptr[4], sizeof(void *)));
  CU_OK(put(c->d_task_enc_b + t, &h.ptr[5], sizeof(void *)));
  return FMX_OK;
}

Backbone *get_bb(fmx_ctx *c, fmx_backbone_t h) {
  if (h < 0 || h >= (int)c->bbs.size() || !c->bbs[h]) return nullptr;
  return c->bbs[h].get();
}

}  // namespace

// =====================================================================================
extern "C" {

int fmx_create(fmx_ctx **out, int device_ordinal) {
  if (!out) return fmx_fail(FMX_E_INVALID_ARG, "fmx_create: out is NULL");
  *out = nullptr;
  int n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess || n_dev == 0)
    return fmx_fail(FMX_E_CUDA, "fmx_create: no CUDA device (%s); libfmx has no CPU fallback", cudaGetErrorString(e));
  if (device_ordinal < 0 || device_ordinal >= n_dev) return fmx_fail(FMX_E_INVALID_ARG, "fmx_create: device %d of %d", device_ordinal, n_dev);
  CU_OK(cudaSetDevice(device_ordinal));
  cudaDeviceProp prop;
  CU_OK(cudaGetDeviceProperties(&prop, device_ordinal));
  if (prop.major != 10) return fmx_fail(FMX_E_CUDA, "fmx_create: device is sm_%d%d; libfmx is built for sm_100a only", prop.major, prop.minor);
  std::unique_ptr<fmx_ctx> c(new fmx_ctx());
  c->device = device_ordinal;
  c->sm_count = prop.multiProcessorCount;
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  CU_OK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
  if (!fn || qres != cudaDriverEntryPointSuccess) return fmx_fail(FMX_E_CUDA, "fmx_create: cuTensorMapEncodeTiled not available");
  c->encode = reinterpret_cast<EncodeTiledFn>(fn);
  if (int err = set_kernel_attrs()) return err;
  {
    // The fused LoRA shrink makes one CTA pair wait for another pair's work item: every cluster of the persistent grid
    // must be resident at the same time.
    auto max_clusters = [&](auto kern, int smem) {
      cudaLaunchConfig_t cfg{};
      cfg.gridDim = dim3(c->sm_count, 1, 1); cfg.blockDim = dim3(kGemmThreads, 1, 1); cfg.dynamicSmemBytes = smem;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      int n = 0;
      if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) { cudaGetLastError(); n = 0; }
      return n;
    };
    const int n256 = std::min(max_clusters(pair_gemm_kernel<256, false>, pair_smem_bytes<256, false>()), max_clusters(pair_gemm_kernel<256, true>, pair_smem_bytes<256, true>()));
    const int n128 = std::min(max_clusters(pair_gemm_kernel<128, false>, pair_smem_bytes<128, false>()), max_clusters(pair_gemm_kernel<128, true>, pair_smem_bytes<128, true>()));
    c->pairs_resident = n256 >= c->sm_count / 2 && n128 >= c->sm_count / 2;
    if (getenv("FMX_DEBUG")) fprintf(stderr, "fmx: max active pair-GEMM clusters %d / %d (need %d): fused shrink %s\n", n256, n128, c->sm_count / 2, c->pairs_resident ? "on" : "off");
  }
  c->tasks.resize(FMX_MAX_TASKS);
  CU_OK(cudaMalloc(&c->d_task_coff, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_kind, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_out, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_trpad, 7 * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_scale, sizeof(float) * 7 * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_W, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_b, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_W2, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_b2, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_head_w1, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_enc_ch, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_enc_W, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMalloc(&c->d_task_enc_b, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_coff, 0, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_kind, 0, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_out, 0, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_trpad, 0, 7 * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_scale, 0, sizeof(float) * 7 * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_W, 0, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_b, 0, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_W2, 0, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_b2, 0, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_head_w1, 0, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_enc_ch, 0, sizeof(int) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_enc_W, 0, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMemset(c->d_task_enc_b, 0, sizeof(void *) * FMX_MAX_TASKS));
  CU_OK(cudaMallocHost(&c->h_stage, sizeof(int) * 4 * FMX_MAX_REQUESTS * fmx_ctx::kStageSlots));
  for (int i = 0; i < fmx_ctx::kStageSlots; ++i) CU_OK(cudaEventCreateWithFlags(&c->stage_ev[i], cudaEventDisableTiming));
  CU_OK(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
  CU_OK(cudaStreamCreateWithFlags(&c->side2, cudaStreamNonBlocking));
  CU_OK(cudaEventCreateWithFlags(&c->side_ev, cudaEventDisableTiming));
  CU_OK(cudaStreamCreateWithFlags(&c->aux, cudaStreamNonBlocking));
  CU_OK(cudaEventCreateWithFlags(&c->fork_ev, cudaEventDisableTiming));
  CU_OK(cudaEventCreateWithFlags(&c->join_ev, cudaEventDisableTiming));
  CU_OK(cudaEventCreateWithFlags(&c->retire_ev, cudaEventDisableTiming));
  CU_OK(cudaMallocHost(&c->h_task_stage, sizeof(fmx_ctx::TaskStage)));
  CU_OK(cudaHostAlloc(&c->h_err, sizeof(unsigned), cudaHostAllocMapped));
  *c->h_err = 0;
  CU_OK(cudaHostGetDevicePointer(&c->d_err, c->h_err, 0));
  CU_OK(cudaMalloc(&c->d_dbg_cu, sizeof(int) * (FMX_MAX_REQUESTS + 1)));
  {
    // task tensors and LoRA slabs come from the device's stream-ordered pool on the registration stream (cudaFree would
    // synchronise the whole device; cudaFreeAsync does not); keep freed memory cached in the pool
    cudaMemPool_t pool = nullptr;
    CU_OK(cudaDeviceGetDefaultMemPool(&pool, device_ordinal));
    unsigned long long keep = ~0ull;
    CU_OK(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
  }
  *out = c.release();
  fmx_clear_error();
  return FMX_OK;
}

int fmx_destroy(fmx_ctx *c) {
  if (!c) return FMX_OK;
  cudaSetDevice(c->device);
  cudaDeviceSynchronize();
  for (auto &pe : c->prof) { cudaEventDestroy(pe.e0); cudaEventDestroy(pe.e1); }
  for (auto e : c->ev_pool) cudaEventDestroy(e);
  for (auto &bp : c->bbs) {
    if (!bp) continue;
    cudaFree(bp->embed_Wpad); cudaFree(bp->posb); cudaFree(bp->rope_cs); cudaFree(bp->rope_cs_t); cudaFree(bp->relb);
    for (int tg = 0; tg < 7; ++tg) { if (bp->slabA[tg]) cudaFreeAsync(bp->slabA[tg], c->side); if (bp->slabB[tg]) cudaFreeAsync(bp->slabB[tg], c->side); if (bp->slabBt[tg]) cudaFreeAsync(bp->slabBt[tg], c->side); }
  }
  for (auto &t : c->tasks)
    for (bf16 *q : {t.head_W, t.head_b, t.head_W2, t.head_b2, t.enc_W, t.enc_b}) if (q) cudaFreeAsync(q, c->side);
  cudaStreamSynchronize(c->side);
  cudaStreamSynchronize(c->side2);
  cudaFree(c->d_task_coff); cudaFree(c->d_task_head_kind); cudaFree(c->d_task_head_out); cudaFree(c->d_task_trpad);
  cudaFree(c->d_task_scale); cudaFree(c->d_task_head_W); cudaFree(c->d_task_head_b);
  cudaFree(c->d_task_head_W2); cudaFree(c->d_task_head_b2); cudaFree(c->d_task_head_w1);
  cudaFree(c->d_task_enc_ch); cudaFree(c->d_task_enc_W); cudaFree(c->d_task_enc_b);
  cudaFree(c->d_dbg_cu);
  for (auto &sv : c->serving) if (sv.ev) cudaEventDestroy(sv.ev);
  cudaFreeHost(c->h_err);
  if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
  for (int i = 0; i < fmx_ctx::kStageSlots; ++i) if (c->stage_ev[i]) cudaEventDestroy(c->stage_ev[i]);
  cudaFreeHost(c->h_stage);
  cudaFreeHost(c->h_task_stage);
  if (c->side_ev) cudaEventDestroy(c->side_ev);
  if (c->retire_ev) cudaEventDestroy(c->retire_ev);
  if (c->fork_ev) cudaEventDestroy(c->fork_ev);
  if (c->join_ev) cudaEventDestroy(c->join_ev);
  if (c->aux) cudaStreamDestroy(c->aux);
  if (c->side) cudaStreamDestroy(c->side);
  if (c->side2) cudaStreamDestroy(c->side2);
  delete c;
  return FMX_OK;
}

int fmx_task_slots(fmx_ctx *c) { return c ? c->n_slots : 0; }

int fmx_register_backbone(fmx_ctx *c, const fmx_backbone_desc *desc, fmx_backbone_t *out) {
  if (!c || !desc || !out) return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: NULL argument");
  std::lock_guard<std::mutex> lk(c->mu);
  ++c->config_gen;                      // invalidates the cached forward graph
  CU_OK(cudaSetDevice(c->device));
  const fmx_backbone_desc &d = *desc;
  if (d.n_layers < 1 || d.d_model < 128 || d.n_q_heads < 1 || d.n_kv_heads < 1 || d.d_ffn < 128 || d.max_seq < 1)
    return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: non-positive dimension");
  const int dq = d.n_q_heads * d.head_dim, dkv = d.n_kv_heads * d.head_dim;
  if (!norm_dim_supported(d.d_model) || dq % 128 || dkv % 128 || d.d_ffn % 128 || d.n_q_heads % d.n_kv_heads ||
      !(d.head_dim == 32 || d.head_dim == 64 || d.head_dim == 128))
    return fmx_fail(FMX_E_SHAPE, "register_backbone: unsupported dims (d_model=%d d_q=%d d_kv=%d d_ffn=%d head_dim=%d)", d.d_model, dq, dkv, d.d_ffn, d.head_dim);
  if (d.act < 0 || d.act > 2 || d.norm < 0 || d.norm > 1 || d.input_kind < 0 || d.input_kind > 2)
    return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: bad enum");
  if (d.tokens_per_request < 0 || d.tokens_per_request > d.max_seq) return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: tokens_per_request > max_seq");
  if (!d.norm1_g || !d.norm2_g || !d.Wq || !d.Wk || !d.Wv || !d.Wo || !d.Wup || !d.Wdown || !d.final_g ||
      (d.act == FMX_ACT_SWIGLU && !d.Wgate))
    return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: missing weight array");
  if (d.norm == FMX_NORM_LAYERNORM && (!d.norm1_b || !d.norm2_b || !d.final_b)) return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: LayerNorm needs *_b");
  if (d.input_kind == FMX_INPUT_PATCH_LINEAR) {
    if (!d.embed_W || d.patch_dim < 1 || d.tokens_per_request < 1) return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: PATCH_LINEAR needs embed_W, patch_dim, tokens_per_request");
    if (d.has_cls && !d.embed_cls) return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: has_cls needs embed_cls");
    if (d.img_c) {
      const int g = d.patch_hw > 0 ? d.img_hw / d.patch_hw : 0;
      if (d.patch_hw < 1 || d.img_hw % d.patch_hw || d.img_c * d.patch_hw * d.patch_hw != d.patch_dim ||
          g * g != d.tokens_per_request - (d.has_cls ? 1 : 0))
        return fmx_fail(FMX_E_SHAPE, "register_backbone: image geometry inconsistent with patch_dim / tokens_per_request");
    }
  }
  if (d.input_kind == FMX_INPUT_TOKEN_IDS && (!d.embed_table || d.vocab < 1)) return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: TOKEN_IDS needs embed_table, vocab");
  if (d.rope_theta > 0 && d.head_dim % 2) return fmx_fail(FMX_E_SHAPE, "register_backbone: RoPE needs even head_dim");
  if (d.rel_bias && d.rel_buckets != 0) {
    const int side = d.causal ? d.rel_buckets : d.rel_buckets / 2;           // buckets per direction
    if (d.rel_buckets < 2 || d.rel_buckets > 256 || d.rel_buckets % 2 || side < 2 || d.rel_max_distance <= side / 2)
      return fmx_fail(FMX_E_SHAPE, "register_backbone: relative-position bias needs an even rel_buckets in 2..256 (>= 4 when not causal) and rel_max_distance > buckets-per-side / 2 (got %d, %d)",
                      d.rel_buckets, d.rel_max_distance);
  }

  std::unique_ptr<Backbone> b(new Backbone());
  b->d = d;
  const int L = d.n_layers;
  b->norm1_g = copy_ptrs(d.norm1_g, L); b->norm1_b = copy_ptrs(d.norm1_b, L);
  b->norm2_g = copy_ptrs(d.norm2_g, L); b->norm2_b = copy_ptrs(d.norm2_b, L);
  b->Wq = copy_ptrs(d.Wq, L); b->Wk = copy_ptrs(d.Wk, L); b->Wv = copy_ptrs(d.Wv, L); b->Wo = copy_ptrs(d.Wo, L);
  b->bq = copy_ptrs(d.bq, L); b->bk = copy_ptrs(d.bk, L); b->bv = copy_ptrs(d.bv, L); b->bo = copy_ptrs(d.bo, L);
  b->Wup = copy_ptrs(d.Wup, L); b->Wgate = copy_ptrs(d.Wgate, L); b->Wdown = copy_ptrs(d.Wdown, L);
  b->bup = copy_ptrs(d.bup, L); b->bgate = copy_ptrs(d.bgate, L); b->bdown = copy_ptrs(d.bdown, L);
  b->d_q = dq; b->d_kv = dkv; b->d_qkv = dq + 2 * dkv;
  for (int tg = 0; tg < 7; ++tg) target_dims(d, tg, b->din[tg], b->dout[tg]);
  for (int l = 0; l < L; ++l) {
    if (!b->norm1_g[l] || !b->norm2_g[l] || !b->Wq[l] || !b->Wk[l] || !b->Wv[l] || !b->Wo[l] || !b->Wup[l] || !b->Wdown[l] ||
        (d.act == FMX_ACT_SWIGLU && !b->Wgate[l]))
      return fmx_fail(FMX_E_INVALID_ARG, "register_backbone: NULL weight pointer in layer %d", l);
  }
  for (int v = 0; v < 2; ++v) {
    const uint32_t br = v == 0 ? 128 : 64;
    b->mWq[v].resize(L); b->mWk[v].resize(L); b->mWv[v].resize(L); b->mWo[v].resize(L); b->mWup[v].resize(L); b->mWgate[v].resize(L); b->mWdown[v].resize(L);
    for (int l = 0; l < L; ++l) {
      int e;
      if ((e = encode_2d(c, &b->mWq[v][l], b->Wq[l], dq, d.d_model, d.d_model, br))) return e;
      if ((e = encode_2d(c, &b->mWk[v][l], b->Wk[l], dkv, d.d_model, d.d_model, br))) return e;
      if ((e = encode_2d(c, &b->mWv[v][l], b->Wv[l], dkv, d.d_model, d.d_model, br))) return e;
      if ((e = encode_2d(c, &b->mWo[v][l], b->Wo[l], d.d_model, dq, dq, br))) return e;
      if ((e = encode_2d(c, &b->mWup[v][l], b->Wup[l], d.d_ffn, d.d_model, d.d_model, br))) return e;
      if (d.act == FMX_ACT_SWIGLU && (e = encode_2d(c, &b->mWgate[v][l], b->Wgate[l], d.d_ffn, d.d_model, d.d_model, br))) return e;
      if ((e = encode_2d(c, &b->mWdown[v][l], b->Wdown[l], d.d_model, d.d_ffn, d.d_ffn, br))) return e;
    }
  }
  if (d.input_kind == FMX_INPUT_PATCH_LINEAR) {
    b->Kp = (d.patch_dim + 7) / 8 * 8;
    CU_OK(cudaMalloc(&b->embed_Wpad, sizeof(bf16) * d.d_model * b->Kp));
    const int n = d.d_model * b->Kp;
    pad_rows_kernel<<<(n + 255) / 256, 256>>>((const bf16 *)d.embed_W, b->embed_Wpad, d.d_model, d.patch_dim, b->Kp);
    const int n_pos = d.tokens_per_request;
    CU_OK(cudaMalloc(&b->posb, sizeof(float) * n_pos * d.d_model));
    build_posb_kernel<<<(n_pos * d.d_model + 255) / 256, 256>>>(b->posb, (const bf16 *)d.embed_b, (const bf16 *)d.embed_cls,
                                                                   (const bf16 *)d.embed_pos, n_pos, d.d_model, d.has_cls);
    CU_OK(cudaGetLastError());
    if (int e = encode_2d(c, &b->mEmbedW[0], b->embed_Wpad, d.d_model, b->Kp, b->Kp, 128)) return e;
    if (int e = encode_2d(c, &b->mEmbedW[1], b->embed_Wpad, d.d_model, b->Kp, b->Kp, 64)) return e;
  }
  if (d.rope_theta > 0) {
    const int n = d.max_seq * (d.head_dim / 2);
    CU_OK(cudaMalloc(&b->rope_cs, sizeof(float2) * n));
    build_rope_table_kernel<<<(n + 255) / 256, 256>>>(b->rope_cs, d.max_seq, d.head_dim, (double)d.rope_theta);
    CU_OK(cudaMalloc(&b->rope_cs_t, sizeof(float2) * n));
    transpose_rope_table_kernel<<<(n + 255) / 256, 256>>>(b->rope_cs, b->rope_cs_t, d.max_seq, d.head_dim / 2);
    CU_OK(cudaGetLastError());
  }
  if (d.rel_bias && d.rel_buckets > 0) {
    // bias by relative distance, for every head: the bucket of each distance is taken here on the host (T5's bucket function in
    // double precision, reading 36), the table row is the caller's bf16 value; stored times log2(e) for the exp2 softmax
    const int nb = d.rel_buckets, H = d.n_q_heads, S = d.max_seq, off = S - 1 + 128, ld = 2 * S - 1 + 255;
    std::vector<uint16_t> tab((size_t)nb * H);
    CU_OK(cudaMemcpy(tab.data(), d.rel_bias, tab.size() * sizeof(uint16_t), cudaMemcpyDeviceToHost));
    std::vector<float> dense((size_t)H * ld, 0.0f);
    for (int rel = -(S - 1); rel <= S - 1; ++rel) {
      int n = nb, bucket = 0, dist;
      if (!d.causal) { n /= 2; if (rel > 0) bucket += n; dist = rel < 0 ? -rel : rel; }
      else dist = rel < 0 ? -rel : 0;
      const int max_exact = n / 2;
      if (dist < max_exact) bucket += dist;
      else bucket += std::min(max_exact + (int)(std::log((double)dist / max_exact) / std::log((double)d.rel_max_distance / max_exact) * (n - max_exact)), n - 1);
      for (int g = 0; g < H; ++g) {
        const uint32_t bits = (uint32_t)tab[(size_t)bucket * H + g] << 16;
        float v;
        memcpy(&v, &bits, sizeof(v));
        dense[(size_t)g * ld + rel + off] = v * 1.4426950408889634f;
      }
    }
    CU_OK(cudaMalloc(&b->relb, dense.size() * sizeof(float)));
    CU_OK(cudaMemcpy(b->relb, dense.data(), dense.size() * sizeof(float), cudaMemcpyHostToDevice));
    b->relb_ld = ld; b->relb_off = off;
  }
  CU_OK(cudaDeviceSynchronize());
  b->Rcap = 256;
  b->row_bt = d.input_kind == FMX_INPUT_TOKEN_IDS && d.causal;      // a decoder: may serve decode iterations (row-wise LoRA reads B rank-major)
  b->col_used.assign(b->Rcap / 16, 0);
  b->col_freed_seq.assign(b->Rcap / 16, 0);
  c->bbs.push_back(std::move(b));
  *out = (int)c->bbs.size() - 1;
  return FMX_OK;
}

int fmx_register_task(fmx_ctx *c, fmx_backbone_t h, const fmx_task_desc *desc, fmx_task_t *out) {
  if (!c || !desc || !out) return fmx_fail(FMX_E_INVALID_ARG, "register_task: NULL argument");
  std::lock_guard<std::mutex> lk(c->mu);
  CU_OK(cudaSetDevice(c->device));
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "register_task: unknown backbone %d", h);
  const fmx_backbone_desc &d = bb->d;
  const int L = d.n_layers;
  // ---- validate everything before touching state ----
  if (desc->n_adapters < 0 || desc->n_adapters > 7 || (desc->n_adapters && !desc->adapters)) return fmx_fail(FMX_E_INVALID_ARG, "register_task: bad n_adapters");
  if (desc->head_kind < 0 || desc->head_kind > FMX_HEAD_DENSE || desc->head_out < 1 || !desc->head_W) return fmx_fail(FMX_E_INVALID_ARG, "register_task: bad head");
  if (desc->head_kind == FMX_HEAD_FLATTEN && d.tokens_per_request < 1) return fmx_fail(FMX_E_SHAPE, "register_task: FLATTEN head needs a fixed-length backbone");
  if (desc->head_hidden < 0 || desc->head_hidden > kMaxHeadHidden) return fmx_fail(FMX_E_SHAPE, "register_task: head_hidden %d not in [0,%d]", desc->head_hidden, kMaxHeadHidden);
  if (desc->head_hidden > 0 && (desc->head_kind == FMX_HEAD_FLATTEN || desc->head_kind == FMX_HEAD_DENSE))
    return fmx_fail(FMX_E_SHAPE, "register_task: an MLP head needs a pooled feature (mean / cls / last)");
  if (desc->head_hidden > 0 && !desc->head_W2) return fmx_fail(FMX_E_INVALID_ARG, "register_task: MLP head without head_W2");
  if (desc->enc_channels < 0 || desc->enc_channels > 16) return fmx_fail(FMX_E_SHAPE, "register_task: enc_channels %d not in [0,16]", desc->enc_channels);
  if (desc->enc_channels > 1 && (d.input_kind != FMX_INPUT_PATCH_LINEAR || d.img_c))
    return fmx_fail(FMX_E_SHAPE, "register_task: an input encoder needs a PATCH_LINEAR backbone with series input");
  if (desc->enc_channels > 1 && !desc->enc_W) return fmx_fail(FMX_E_INVALID_ARG, "register_task: input encoder without enc_W");
  bool seen[7] = {false};
  int rpad = 0;
  for (int i = 0; i < desc->n_adapters; ++i) {
    const fmx_adapter_desc &a = desc->adapters[i];
    if (a.target < 0 || a.target > 6) return fmx_fail(FMX_E_INVALID_ARG, "register_task: adapter %d: bad target", i);
    if (seen[a.target]) return fmx_fail(FMX_E_INVALID_ARG, "register_task: two adapters on target %d", a.target);
    seen[a.target] = true;
    if (a.rank < 1 || a.rank > FMX_MAX_RANK) return fmx_fail(FMX_E_SHAPE, "register_task: adapter %d: rank %d not in [1,%d]", i, a.rank, FMX_MAX_RANK);
    if ((a.target == FMX_TGT_GATE) && d.act != FMX_ACT_SWIGLU) return fmx_fail(FMX_E_SHAPE, "register_task: gate adapter on a backbone without a gate projection");
    if (!a.A || !a.B) return fmx_fail(FMX_E_INVALID_ARG, "register_task: adapter %d: NULL A/B array", i);
    for (int l = 0; l < L; ++l) if (!a.A[l] || !a.B[l]) return fmx_fail(FMX_E_INVALID_ARG, "register_task: adapter %d: NULL A/B in layer %d", i, l);
    rpad = std::max(rpad, (a.rank + 15) / 16 * 16);
  }
  int slot = -1;
  for (int t = 0; t < FMX_MAX_TASKS; ++t) if (!c->tasks[t].live) { slot = t; break; }
  if (slot < 0) return fmx_fail(FMX_E_CAPACITY, "register_task: all %d task slots in use", FMX_MAX_TASKS);

  // Nothing below changes the registry until the last fallible call has succeeded: buffers are allocated first, the slab
  // arena may grow (a grown arena is a valid state by itself), the copies are enqueued, and only then are the columns, the
  // adapter counts and the task record committed.  On failure the buffers allocated here go back to the pool.
  TaskRec r;
  r.live = true; r.bb = h; r.head_kind = desc->head_kind; r.head_out = desc->head_out; r.head_hidden = desc->head_hidden; r.rpad = rpad;
  r.freed_seq = c->tasks[slot].freed_seq;
  std::vector<void *> mine;
  auto fail = [&](int code) { for (void *q : mine) cudaFreeAsync(q, c->side); return code; };
  auto dup = [&](bf16 **dst, const void *src, size_t n) -> int {           // device -> device copy into a pool allocation
    cudaError_t e = cudaMallocAsync(dst, n * sizeof(bf16), c->side);
    if (e != cudaSuccess) { *dst = nullptr; return fmx_fail(FMX_E_CUDA, "register_task: cudaMallocAsync(%zu B) failed: %s", n * sizeof(bf16), cudaGetErrorString(e)); }
    mine.push_back(*dst);
    e = cudaMemcpyAsync(*dst, src, n * sizeof(bf16), cudaMemcpyDeviceToDevice, c->side);
    if (e != cudaSuccess) return fmx_fail(FMX_E_CUDA, "register_task: copy failed: %s", cudaGetErrorString(e));
    return FMX_OK;
  };
  // ---- head / encoder buffers ----
  const size_t d_feat = desc->head_kind == FMX_HEAD_FLATTEN ? (size_t)d.tokens_per_request * d.d_model : (size_t)d.d_model;
  const size_t w1 = desc->head_hidden > 0 ? (size_t)desc->head_hidden : (size_t)desc->head_out;     // rows of the first layer
  if (int e = dup(&r.head_W, desc->head_W, d_feat * w1)) return fail(e);
  if (desc->head_b) if (int e = dup(&r.head_b, desc->head_b, w1)) return fail(e);
  if (desc->enc_channels > 1) {
    r.enc_channels = desc->enc_channels;
    if (int e = dup(&r.enc_W, desc->enc_W, desc->enc_channels)) return fail(e);
    if (desc->enc_b) if (int e = dup(&r.enc_b, desc->enc_b, 1)) return fail(e);
  }
  if (desc->head_hidden > 0) {
    if (int e = dup(&r.head_W2, desc->head_W2, (size_t)desc->head_out * desc->head_hidden)) return fail(e);
    if (desc->head_b2) if (int e = dup(&r.head_b2, desc->head_b2, desc->head_out)) return fail(e);
  }
  // ---- slab columns ----
  int pos = -1, units = rpad / 16;
  if (rpad) {
    pos = find_columns(*bb, units);
    int new_cap = bb->Rcap;
    while (pos < 0) {
      new_cap *= 2;
      if (new_cap > 16 * 65536) return fail(fmx_fail(FMX_E_CAPACITY, "register_task: LoRA slab capacity exceeded"));
      if (int e = grow_slabs(c, *bb, new_cap)) return fail(e);
      pos = find_columns(*bb, units);
    }
    r.coff = pos * 16;
    for (int i = 0; i < desc->n_adapters; ++i)
      if (!bb->slabA[desc->adapters[i].target]) if (int e = alloc_slab(c, *bb, desc->adapters[i].target)) return fail(e);
    // a slot or columns handed back by a recent fmx_unregister_task may still be read by forwards that were in flight then
    unsigned long long seq = r.freed_seq;
    for (int u = 0; u < units; ++u) seq = std::max(seq, bb->col_freed_seq[pos + u]);
    if (int e = wait_retired(c, seq)) return fail(e);
    for (int i = 0; i < desc->n_adapters; ++i) {
      const fmx_adapter_desc &a = desc->adapters[i];
      const int tg = a.target, rp = (a.rank + 15) / 16 * 16;
      const int din = bb->din[tg], dout = bb->dout[tg];
      for (int l = 0; l < L; ++l) {
        bf16 *A = bb->slabA[tg] + ((size_t)l * bb->Rcap + r.coff) * din;
        bf16 *B = bb->slabB[tg] + (size_t)l * dout * bb->Rcap + r.coff;
        cudaError_t e = cudaSuccess;
        if (rp > a.rank) {                 // the zero padding of the rank (exact): whatever a previous owner left there goes
          e = cudaMemsetAsync(A + (size_t)a.rank * din, 0, (size_t)(rp - a.rank) * din * sizeof(bf16), c->side);
          if (e == cudaSuccess) e = cudaMemset2DAsync(B + a.rank, (size_t)bb->Rcap * sizeof(bf16), 0, (size_t)(rp - a.rank) * sizeof(bf16), dout, c->side);
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(A, a.A[l], (size_t)a.rank * din * sizeof(bf16), cudaMemcpyDeviceToDevice, c->side);
        if (e == cudaSuccess)
          e = cudaMemcpy2DAsync(B, (size_t)bb->Rcap * sizeof(bf16), a.B[l], (size_t)a.rank * sizeof(bf16), (size_t)a.rank * sizeof(bf16),
                                dout, cudaMemcpyDeviceToDevice, c->side);
        if (e == cudaSuccess && bb->slabBt[tg]) {          // rank-major copy, padding rows zeroed
          bf16 *Bt = bb->slabBt[tg] + ((size_t)l * bb->Rcap + r.coff) * dout;
          lora_bt_fill_kernel<<<(unsigned)(((size_t)dout * rp + 255) / 256), 256, 0, c->side>>>((const bf16 *)a.B[l], Bt, dout, a.rank, rp);
          e = cudaGetLastError();
        }
        if (e != cudaSuccess) return fail(fmx_fail(FMX_E_CUDA, "register_task: adapter copy failed: %s", cudaGetErrorString(e)));
      }
      r.trpad[tg] = (unsigned char)rp;
      r.scale[tg] = a.scaling;
    }
  } else if (int e = wait_retired(c, r.freed_seq)) {
    return fail(e);
  }
  // ---- device tables, then commit ----
  if (int e = upload_task_tables(c, slot, r)) return fail(e);
  if (cudaError_t e = cudaStreamSynchronize(c->side))      // the caller may free its buffers; forwards in flight are not waited for
    return fail(fmx_fail(FMX_E_CUDA, "register_task: %s", cudaGetErrorString(e)));
  for (int u = 0; u < units; ++u) bb->col_used[pos + u] = 1;
  for (int tg = 0; tg < 7; ++tg) if (r.trpad[tg]) bb->n_adapters[tg]++;
  c->tasks[slot] = r;
  c->n_slots = std::max(c->n_slots, slot + 1);
  ++c->config_gen;                      // invalidates the cached forward graph
  *out = slot;
  return FMX_OK;
}

// No device-wide synchronisation: the task leaves the registry at once (later forwards reject its id), its buffers are freed
// on the retirement stream after the forwards in flight, and its slot / slab columns carry the retirement's sequence number
// so that a registration reusing them waits for it on the device.  Slab columns are not cleared: no live task reads them
// (a registration zero-fills the padding of its own columns).
int fmx_unregister_task(fmx_ctx *c, fmx_task_t t) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "unregister_task: NULL ctx");
  std::lock_guard<std::mutex> lk(c->mu);
  if (t < 0 || t >= FMX_MAX_TASKS || !c->tasks[t].live) return fmx_fail(FMX_E_UNKNOWN_TASK, "unregister_task: task %d is not registered", t);
  CU_OK(cudaSetDevice(c->device));
  TaskRec &r = c->tasks[t];
  Backbone *bb = get_bb(c, r.bb);
  if (int e = retire(c, {r.head_W, r.head_b, r.head_W2, r.head_b2, r.enc_W, r.enc_b})) return e;
  for (int tg = 0; tg < 7; ++tg) if (r.trpad[tg]) bb->n_adapters[tg]--;
  for (int u = 0; u < r.rpad / 16; ++u) { bb->col_used[r.coff / 16 + u] = 0; bb->col_freed_seq[r.coff / 16 + u] = c->retire_seq; }
  r = TaskRec();
  r.freed_seq = c->retire_seq;
  ++c->config_gen;                      // invalidates the cached forward graph
  return FMX_OK;
}

static int output_layout_locked(fmx_ctx *c, const int32_t *task_ids, const int32_t *lengths, int32_t n_req, int64_t *out_off);
int fmx_output_layout(fmx_ctx *c, const int32_t *task_ids, int32_t n_req, int64_t *out_off) {
  if (!c || !out_off || (n_req > 0 && !task_ids) || n_req < 0) return fmx_fail(FMX_E_INVALID_ARG, "output_layout: bad argument");
  std::lock_guard<std::mutex> lk(c->mu);
  return output_layout_locked(c, task_ids, nullptr, n_req, out_off);
}
int fmx_output_layout_len(fmx_ctx *c, const int32_t *task_ids, const int32_t *lengths, int32_t n_req, int64_t *out_off) {
  if (!c || !out_off || (n_req > 0 && (!task_ids || !lengths)) || n_req < 0) return fmx_fail(FMX_E_INVALID_ARG, "output_layout_len: bad argument");
  std::lock_guard<std::mutex> lk(c->mu);
  return output_layout_locked(c, task_ids, lengths, n_req, out_off);
}

static int output_layout_locked(fmx_ctx *c, const int32_t *task_ids, const int32_t *lengths, int32_t n_req, int64_t *out_off) {
  int64_t run = 0;
  for (int i = 0; i < n_req; ++i) {
    const int t = task_ids[i];
    if (t < 0 || t >= FMX_MAX_TASKS || !c->tasks[t].live) return fmx_fail(FMX_E_UNKNOWN_TASK, "output_layout: request %d: task %d is not registered", i, t);
    out_off[i] = run;
    int64_t rows = 1;
    if (c->tasks[t].head_kind == FMX_HEAD_DENSE) {                  // one output row per token
      rows = lengths ? lengths[i] : get_bb(c, c->tasks[t].bb)->d.tokens_per_request;
      if (rows < 1) return fmx_fail(FMX_E_BAD_LENGTH, "output_layout: request %d: a dense head on a variable-length backbone needs fmx_output_layout_len", i);
    }
    run += rows * c->tasks[t].head_out;
  }
  out_off[n_req] = run;
  return FMX_OK;
}

int fmx_workspace_bytes(fmx_ctx *c, fmx_backbone_t h, int32_t max_req, int64_t max_tokens, size_t *bytes) {
  if (!c || !bytes) return fmx_fail(FMX_E_INVALID_ARG, "workspace_bytes: NULL argument");
  std::lock_guard<std::mutex> lk(c->mu);
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "workspace_bytes: unknown backbone %d", h);
  if (max_req < 1 || max_req > FMX_MAX_REQUESTS || max_tokens < 1 || max_tokens > (1ll << 24))
    return fmx_fail(FMX_E_CAPACITY, "workspace_bytes: max_req in [1,%d], max_tokens in [1,2^24]", FMX_MAX_REQUESTS);
  *bytes = carve(*bb, nullptr, max_req, max_tokens, FMX_MAX_TASKS).bytes;
  return FMX_OK;
}

int fmx_host_workspace_bytes(fmx_ctx *c, fmx_backbone_t h, int32_t max_req, int64_t max_tokens, size_t max_input_bytes,
                             int64_t max_output_floats, size_t *bytes) {
  if (max_output_floats < 0) return fmx_fail(FMX_E_INVALID_ARG, "host_workspace_bytes: max_output_floats < 0");
  if (int e = fmx_workspace_bytes(c, h, max_req, max_tokens, bytes)) return e;
  *bytes += align_up(max_input_bytes, 1024) + align_up((size_t)max_output_floats * sizeof(float), 1024);
  return FMX_OK;
}

// ---------------------------------------------------------------- the forward
// What the launch sequence of a forward depends on, beyond the buffers: everything the host derives from the caller's
// ids / lengths.  Two batches with the same BatchShape run the SAME kernels with the same grids (the ids / lengths
// themselves travel to the device tables), so one captured CUDA graph serves both.
// Host validation of a batch (nothing is enqueued on failure) and its BatchShape.
static int batch_shape(fmx_ctx *c, const Backbone &bb, const int32_t *task_ids, const int32_t *lengths, int32_t B, BatchShape &bs) {
  const fmx_backbone_desc &d = bb.d;
  int bb_index = -1;
  for (size_t i = 0; i < c->bbs.size(); ++i) if (c->bbs[i].get() == &bb) bb_index = (int)i;
  bs = BatchShape();
  for (int i = 0; i < B; ++i) {
    const int t = task_ids[i];
    if (t < 0 || t >= FMX_MAX_TASKS || !c->tasks[t].live || c->tasks[t].bb != bb_index)
      return fmx_fail(FMX_E_UNKNOWN_TASK, "forward_mixed: request %d: task %d is not registered on this backbone", i, t);
    const int n = lengths[i];
    if (n < 1 || n > d.max_seq || (d.tokens_per_request && n != d.tokens_per_request))
      return fmx_fail(FMX_E_BAD_LENGTH, "forward_mixed: request %d: length %d (max_seq %d, fixed %d)", i, n, d.max_seq, d.tokens_per_request);
    const TaskRec &tr = c->tasks[t];
    bs.N += n;
    bs.max_len = std::max(bs.max_len, n);
    bs.max_out = std::max(bs.max_out, tr.head_hidden > 0 ? tr.head_hidden : tr.head_out);   // first-layer width
    if (tr.head_hidden > 0) { bs.max_hidden = std::max(bs.max_hidden, tr.head_hidden); bs.max_out2 = std::max(bs.max_out2, tr.head_out); }
    if (tr.head_kind == FMX_HEAD_FLATTEN) { bs.any_flat = true; bs.max_out_flat = std::max(bs.max_out_flat, tr.head_out); }
    else if (tr.head_kind == FMX_HEAD_DENSE) { bs.any_dense = true; bs.max_out_dense = std::max(bs.max_out_dense, tr.head_out); }
    else bs.any_pooled = true;
  }
  if (bs.N > (1ll << 24)) return fmx_fail(FMX_E_CAPACITY, "forward_mixed: %lld tokens > 2^24", bs.N);
  // (tile, task) blocks of the task-sorted batch (the device computes the same number in S1)
  const int T = c->n_slots;
  std::vector<long long> tok(T + 1, 0);
  for (int i = 0; i < B; ++i) tok[task_ids[i]] += lengths[i];
  long long lo = 0;
  for (int t = 0; t < T; ++t) {
    if (tok[t] == 0) continue;
    const long long hi = lo + tok[t];
    bs.n_blk += (int)((hi - 1) / kPairRows - lo / kPairRows + 1);
    lo = hi;
  }
  return FMX_OK;
}

// ids / lengths -> the device tables, through the pinned staging ring (a slot is rewritten only after the copy that read it
// has run).  Never part of a captured graph: a replay serves a NEW batch, so these copies are enqueued before every launch.
static int stage_ids(fmx_ctx *c, const Workspace &w, const int32_t *task_ids, const int32_t *lengths, int32_t B, cudaStream_t s,
                     const int32_t *slots = nullptr, const int32_t *pos0 = nullptr) {
  const int slot = c->stage_next;
  c->stage_next = (c->stage_next + 1) % fmx_ctx::kStageSlots;
  if (c->stage_used[slot]) CU_OK(cudaEventSynchronize(c->stage_ev[slot]));
  int *stage = c->h_stage + (size_t)slot * 4 * FMX_MAX_REQUESTS;
  memcpy(stage, task_ids, sizeof(int) * B);
  memcpy(stage + FMX_MAX_REQUESTS, lengths, sizeof(int) * B);
  CU_OK(cudaMemcpyAsync(w.t.task_ids, stage, sizeof(int) * B, cudaMemcpyHostToDevice, s));
  CU_OK(cudaMemcpyAsync(w.t.lengths, stage + FMX_MAX_REQUESTS, sizeof(int) * B, cudaMemcpyHostToDevice, s));
  if (slots) {
    memcpy(stage + 2 * FMX_MAX_REQUESTS, slots, sizeof(int) * B);
    CU_OK(cudaMemcpyAsync(w.slots, stage + 2 * FMX_MAX_REQUESTS, sizeof(int) * B, cudaMemcpyHostToDevice, s));
  }
  if (pos0) {
    memcpy(stage + 3 * FMX_MAX_REQUESTS, pos0, sizeof(int) * B);
    CU_OK(cudaMemcpyAsync(w.pos0, stage + 3 * FMX_MAX_REQUESTS, sizeof(int) * B, cudaMemcpyHostToDevice, s));
  }
  CU_OK(cudaEventRecord(c->stage_ev[slot], s));
  c->stage_used[slot] = true;
  return FMX_OK;
}

// A forward that also maintains a key / value cache (NEXT-3): prefill writes every request's k / v rows into its slot,
// a decode step appends ONE token per request and attends the cached positions.
struct KvCall {
  bf16 *cache = nullptr;
  int n_slots = 0;
  const int32_t *slots = nullptr;        // HOST [B]
  const int32_t *pos0 = nullptr;         // HOST [B] tokens already cached per request (decode); NULL = prefill from 0
  float *scores = nullptr;               // DEVICE fp32 [B, lm_vocab] or NULL
  int32_t *next_tokens = nullptr;        // DEVICE int32 [B] or NULL
  bool decode = false;
};

// graph_capture: the stream is being captured into the context's cached graph: ids / lengths go through the graph's own
// pinned buffer and no event is recorded.
static int forward_impl(fmx_ctx *c, Backbone &bb, const void *inputs, const int32_t *task_ids, const int32_t *lengths,
                        int32_t B, float *outputs, void *workspace, size_t workspace_bytes, cudaStream_t s, const BatchShape &bs,
                        bool graph_capture = false, const KvCall *kv = nullptr) {
  const fmx_backbone_desc &d = bb.d;
  const long long N = bs.N;
  const int max_len = bs.max_len, max_out = bs.max_out;
  const int T = c->n_slots;
  if (reinterpret_cast<uintptr_t>(workspace) & 1023) return fmx_fail(FMX_E_WORKSPACE, "forward_mixed: workspace must be 1024-byte aligned");
  Workspace w = carve(bb, workspace, B, N, T);
  if (w.bytes > workspace_bytes) return fmx_fail(FMX_E_WORKSPACE, "forward_mixed: workspace %zu B < required %zu B", workspace_bytes, w.bytes);

  const int Ni = (int)N;
  const Strm S{s, (c->o.pdl == 1 || (c->o.pdl == 2 && Ni <= kPdlAutoRows)) ? 1 : 0};
  Launcher Lh{c, s};
  // Every kernel of the layer chain streams over all N rows and the next one reads what it wrote.  Walking the rows in
  // alternating directions lets each kernel start on the rows its producer wrote last, which are the ones still in L2.
  int dir = 0;
  auto rev = [&]() { const int r = c->o.reverse ? dir : 0; dir ^= 1; return r; };
  // ---- S1: ids/lengths to the device, counting sort, tables ----
  if (!graph_capture) {
    // ids / lengths reach the device through the library's pinned staging ring, whose slots are rewritten a few calls later:
    // a graph the CALLER captures would replay stale copies, so a capturing stream is refused (the library keeps its own
    // graph cache, FMX_OPT_GRAPH).
    cudaStreamCaptureStatus cap_status = cudaStreamCaptureStatusNone;
    CU_OK(cudaStreamIsCapturing(s, &cap_status));
    if (cap_status != cudaStreamCaptureStatusNone)
      return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed: the stream is being captured; capture is not supported (the library caches its own CUDA graph)");
    if (int e = stage_ids(c, w, task_ids, lengths, B, s, kv ? kv->slots : nullptr, kv ? kv->pos0 : nullptr)) return e;
  }
  SortArgs sa{};
  sa.t = w.t; sa.B = B; sa.T = T; sa.n_tiles = w.n_tiles; sa.tile_rows = kPairRows; sa.task_head_out = c->d_task_head_out; sa.task_head_kind = c->d_task_head_kind;
  sa.task_enc_ch = (d.input_kind == FMX_INPUT_PATCH_LINEAR && !d.img_c) ? c->d_task_enc_ch : nullptr;
  if (d.input_kind == FMX_INPUT_EMBEDDED) { sa.in_per_tok = d.d_model; sa.in_per_req = 0; }
  else if (d.input_kind == FMX_INPUT_TOKEN_IDS) { sa.in_per_tok = 1; sa.in_per_req = 0; }
  else if (d.img_c) { sa.in_per_tok = 0; sa.in_per_req = (long long)d.img_c * d.img_hw * d.img_hw; }
  else { sa.in_per_tok = 0; sa.in_per_req = (long long)(d.tokens_per_request - (d.has_cls ? 1 : 0)) * d.patch_dim; }
  LAUNCH(Lh, F_SORT, (launch_k(task_sort_kernel, 1, kSortThreads, 0, S, sa)));
  LAUNCH(Lh, F_SORT, (launch_k(row_tables_kernel, (Ni + 255) / 256, 256, 0, S, w.t.cu_tok, B, Ni, w.t.row_req, w.t.row_pos)));
  KvArgs ka{};
  if (kv) {
    ka.cache = kv->cache; ka.d_kv = bb.d_kv; ka.max_seq = d.max_seq;
    ka.kv_stride = (long long)d.max_seq * bb.d_kv; ka.layer_stride = 2 * ka.kv_stride; ka.slot_stride = (long long)d.n_layers * ka.layer_stride;
    ka.row_slot = w.row_slot; ka.row_cpos = w.row_cpos;
    LAUNCH(Lh, F_SORT, (launch_k(kv_rows_kernel, (Ni + 255) / 256, 256, 0, S, (const int *)w.t.row_req, (const int *)w.t.row_pos, (const int *)w.t.perm,
                                 (const int *)w.slots, kv->pos0 ? (const int *)w.pos0 : (const int *)nullptr, Ni, w.row_slot, w.row_cpos)));
  }
  const int *rope_pos = kv ? w.row_cpos : w.t.row_pos;        // RoPE position of a row = its position in the request's WHOLE sequence

  // ---- common GEMM parameter pieces ----
  GemmParams sbase{};                       // segmented shrink
  sbase.M = Ni; sbase.n_mtiles = w.n_tiles;
  sbase.tile_blk_off = w.t.tile_blk_off; sbase.blk_task = w.t.blk_task; sbase.blk_lo = w.t.blk_lo; sbase.blk_hi = w.t.blk_hi;
  sbase.blk_tile = w.t.blk_tile; sbase.n_blk = w.t.n_blk;
  sbase.task_coff = c->d_task_coff; sbase.task_trpad = c->d_task_trpad; sbase.task_scale = c->d_task_scale;
  PairGemmParams base{};                    // projections
  base.M = Ni; base.n_ptiles = w.n_tiles;
  base.tile_blk_off = w.t.tile_blk_off; base.blk_task = w.t.blk_task;
  base.task_coff = c->d_task_coff; base.task_trpad = c->d_task_trpad;
  base.row_pos = w.t.row_pos;
  for (int i = 0; i < 3; ++i) { base.lora_tgt[i] = -1; base.src_end[i] = 1 << 30; }
  CUtensorMap mXn, mAttnO, mHid, mU, mPk, oQKV, oHid, oX, mQKV64;
  int e;
  if ((e = encode_2d(c, &mXn, w.Xn, Ni, d.d_model, d.d_model, 128))) return e;
  if ((e = encode_2d(c, &mAttnO, w.AttnO, Ni, bb.d_q, bb.d_q, 128))) return e;
  if ((e = encode_2d(c, &mHid, w.Hid, Ni, d.d_ffn, d.d_ffn, 128))) return e;
  if ((e = encode_2d(c, &mU, w.U, (uint64_t)w.n_blk_cap * kPairRows, 192, 192, 128))) return e;
  if ((e = encode_2d(c, &oQKV, w.QKV, Ni, bb.d_qkv, bb.d_qkv, 128))) return e;
  if ((e = encode_2d(c, &mQKV64, w.QKV, Ni, bb.d_qkv, bb.d_qkv, 64))) return e;     // attention: box {64, 64}
  oHid = mHid;                              // same bf16 {64,128} box serves loads and stores
  if ((e = encode_2d(c, &oX, w.X, Ni, d.d_model, d.d_model, 128, true))) return e;
  base.umap = mU;
  auto wv = [](const PairGemmParams &p) { return p.n_chunks % 2 == 0 ? 0 : 1; };   // weight-map variant (box rows 128 / 64)

  // shrink over an input group: targets tgs[0..n) that currently have adapters; fills uslot_of[tg]
  int uslot_of[7] = {-1, -1, -1, -1, -1, -1, -1};
  auto shrink = [&](const CUtensorMap &amap, int K, const int *tgs, int n, int layer) -> int {
    if (kv && kv->decode && w.splitk && bb.row_bt && w.n_tiles == 1) return FMX_OK;     // row_mode: row_shrink_kernel + row_expand_kernel do shrink and expand
    GemmParams p = sbase;
    p.mode = GM_SHRINK; p.amap = amap; p.K = K; p.out = w.U; p.ld_out = 192; p.n_tg = 0;
    for (int i = 0; i < n; ++i) {
      const int tg = tgs[i];
      uslot_of[tg] = -1;
      if (bb.n_adapters[tg] <= 0) continue;
      p.wmap[p.n_tg] = bb.mA[tg][layer];
      p.tg_ids[p.n_tg] = tg;
      uslot_of[tg] = p.n_tg++;
    }
    if (p.n_tg == 0) return FMX_OK;
    p.reverse = rev();
    LAUNCH(Lh, F_SHRINK, launch_shrink(c, S, p));
    return FMX_OK;
  };
  // fused form: no launch; the GEMM that reads the same input computes U in its first work items
  unsigned u_epoch = 0;
  auto shrink_fused = [&](PairGemmParams &p, const int *tgs, int n, int layer) {
    p.n_sh = 0;
    for (int i = 0; i < n; ++i) {
      const int tg = tgs[i];
      uslot_of[tg] = -1;
      if (bb.n_adapters[tg] <= 0) continue;
      p.smap[p.n_sh] = bb.mA[tg][layer];
      p.sh_tg[p.n_sh] = tg;
      uslot_of[tg] = p.n_sh++;
    }
    if (p.n_sh == 0) return;
    p.blk_tile = w.t.blk_tile; p.blk_lo = w.t.blk_lo; p.blk_hi = w.t.blk_hi; p.n_blk = w.t.n_blk;
    p.task_scale = c->d_task_scale; p.U = w.U; p.u_flag = w.u_flag; p.u_epoch = ++u_epoch; p.err = c->d_err;
  };
  // (tile, task) blocks of the sorted batch (bs.n_blk, counted on the host).  Measured on B200: fusing pays when the shrink
  // items fit ONE wave of the persistent grid (cfg2: 73 blocks on 74 pairs, -0.4 ms per step); with more blocks the items'
  // low arithmetic intensity costs as much as the separate shrink launches (cfg3 / cfg4 / cfg5 at 92 tasks: +-0).
  const int n_blk_host = bs.n_blk;
  const bool fuse_ok = !(kv && kv->decode && w.splitk && bb.row_bt && w.n_tiles == 1) && c->o.shrink_fused && c->pairs_resident && (c->o.shrink_fused == 2 || n_blk_host <= c->sm_count / 2);
  if (fuse_ok) CU_OK(cudaMemsetAsync(w.u_flag, 0, sizeof(unsigned), s));
  if (kv && kv->decode) CU_OK(cudaMemsetAsync(w.dec_cnt, 0, sizeof(unsigned) * (size_t)B * d.n_kv_heads, s));   // the last chunk's CTA resets its counter; this covers an aborted launch
  // fusable: all CTA pairs of the persistent grid are co-resident (the expand steps spin on another pair's result) and
  // a 3-target group needs the 256-wide kernel
  auto can_fuse = [&](const PairGemmParams &p, int n_targets) {
    return fuse_ok && (n_targets < 3 || pair_wide(p));
  };

  auto set_lora = [&](PairGemmParams &p, int src, int tg, int layer) {
    if (kv && kv->decode && w.splitk && bb.row_bt && w.n_tiles == 1) return;
    if (bb.n_adapters[tg] > 0 && uslot_of[tg] >= 0) {
      p.lora_tgt[src] = tg; p.uslot[src] = uslot_of[tg]; p.lmap[src] = bb.mB[tg][layer]; p.has_lora = 1;
    }
  };

  // Decode iterations (one row tile of <= 256 rows, a few rows per task).  The segmented tensor-core LoRA path would load a 256-row U
  // tile and a slab block per (tile, task) for a few rows of work, and a projection with few N tiles would be streamed by a handful
  // of CTA pairs.  So in this mode (row_mode): (1) row_shrink_kernel + row_expand_kernel compute every row's LoRA delta on CUDA cores,
  // on the auxiliary stream beside (2) the projection without shrink / expand, which stores raw fp32 partials of K slices:
  // row_gemm_kernel for <= 128 rows, else the pair GEMM in partial-output mode with its K axis split over the CTA pairs; (3) a
  // reduction adds the partials in split order, the delta and the bias and applies what follows (RoPE + cache append, SwiGLU /
  // activation, residual update + the next norm).  Within each of the two size classes every choice depends on the projection's
  // shape only, never on the batch, so a request decodes to the same bits alone and in a batch of its class.  (Prefill keeps the
  // fused path: its outputs must not depend on the batch size.)
  const bool row_mode = kv && kv->decode && w.splitk && bb.row_bt && w.n_tiles == 1;
  // row mode fuses what follows a reduction into it: RoPE + the cache append after q / k / v, the next norm after a residual update
  const bool row_norm_fused = row_mode && d.d_model <= 4096;
  const bf16 *next_norm_g = nullptr, *next_norm_b = nullptr;
  auto project = [&](PairGemmParams &p, int family, __nv_bfloat16 *out_bf16, int ld_out, const __nv_bfloat16 *x, const int *tgs, int n_tg, int layer,
                     const void *W0, const void *W1, const void *W2) -> int {
    if (!row_mode) { LAUNCH(Lh, family, launch_pair_gemm(c, S, p)); return FMX_OK; }
    const int Nn = p.n_chunks * 128;
    bool any = false;
    for (int i = 0; i < n_tg; ++i) any = any || bb.n_adapters[tgs[i]] > 0;
    // the LoRA kernels and the GEMM are independent until the reduction: fork them (not while per-launch profiling events are on)
    const bool fork = any && c->o.decode_fork && !c->prof_on;
    if (any) {
      RowLoraArgs la{};
      la.x = x; la.M = Ni; la.K = p.K; la.ld_delta = Nn; la.delta = w.delta; la.n_tg = n_tg; la.interleave2 = p.interleave2; la.Rcap = bb.Rcap;
      la.row_req = w.t.row_req; la.task_sorted = w.t.task_sorted; la.task_coff = c->d_task_coff; la.task_trpad = c->d_task_trpad; la.task_scale = c->d_task_scale;
      int col = 0;
      for (int i = 0; i < n_tg; ++i) {
        const int tg = tgs[i];
        la.tg[i] = tg; la.d_out[i] = bb.dout[tg]; la.col0[i] = col; col += bb.dout[tg];
        la.slabA[i] = bb.slabA[tg] ? bb.slabA[tg] + (size_t)layer * bb.Rcap * bb.din[tg] : nullptr;
        la.slabB[i] = bb.slabBt[tg] ? bb.slabBt[tg] + (size_t)layer * bb.Rcap * bb.dout[tg] : nullptr;
      }
      int max_dout = 0;
      for (int i = 0; i < n_tg; ++i) max_dout = std::max(max_dout, bb.dout[tgs[i]]);
      const int nkc = row_shrink_chunks(p.K), k_range = ((p.K + nkc - 1) / nkc + 255) / 256 * 256;
      const Strm SL = fork ? Strm{c->aux, 0} : S;
      if (fork) { CU_OK(cudaEventRecord(c->fork_ev, s)); CU_OK(cudaStreamWaitEvent(c->aux, c->fork_ev, 0)); }
      LAUNCH(Lh, F_SHRINK, (launch_k(row_shrink_kernel, dim3(Ni, n_tg, nkc), 256, 0, SL, la, w.rowu, k_range)));
      LAUNCH(Lh, F_SHRINK, (launch_k(row_expand_kernel, dim3(Ni, n_tg, (max_dout + kRowExpandCols - 1) / kRowExpandCols), 256, 0, SL, la, (const float *)w.rowu, nkc)));
      if (fork) CU_OK(cudaEventRecord(c->join_ev, c->aux));
    }
    const int nK = (p.K + kBK - 1) / kBK;
    int ks = 1, split_rows = kPairRows;
    if (Ni <= 128 && c->o.decode_rowgemm) {
      // the lean small-M kernel (row_gemm.cuh): 128-column slices x K slices, ~2 CTAs per SM, at least two 64-wide chunks per slice
      RowGemmArgs ga{};
      ga.x = x; ga.M = Ni; ga.K = p.K; ga.N = Nn; ga.interleave2 = p.interleave2;
      ga.W[0] = (const bf16 *)W0; ga.W[1] = (const bf16 *)W1; ga.W[2] = (const bf16 *)W2;
      for (int i = 0; i < 3; ++i) ga.src_end_col[i] = p.src_end[i] >= (1 << 20) ? (1 << 30) : p.src_end[i] * 128;
      const int n_slices = Nn / kRgCols;
      split_rows = (Ni + 15) / 16 * 16;
      ks = std::max(1, std::min(2 * c->sm_count / n_slices, nK / 2));      // one wave at two CTAs per SM
      while (ks > 1 && (size_t)ks * split_rows * Nn > (size_t)kPairRows * splitk_cols(bb)) --ks;      // the partials' workspace
      const int cps = (nK + ks - 1) / ks;
      ks = (nK + cps - 1) / cps;
      ga.chunks_per_split = cps; ga.split_rows = split_rows; ga.partial = w.splitk;
      const dim3 grid(n_slices, ks);
      if (Ni <= 16) LAUNCH(Lh, family, (launch_k(row_gemm_kernel<1>, grid, 256, row_gemm_smem<1>(), S, ga)));
      else if (Ni <= 32) LAUNCH(Lh, family, (launch_k(row_gemm_kernel<2>, grid, 256, row_gemm_smem<2>(), S, ga)));
      else if (Ni <= 64) LAUNCH(Lh, family, (launch_k(row_gemm_kernel<4>, grid, 256, row_gemm_smem<4>(), S, ga)));
      else LAUNCH(Lh, family, (launch_k(row_gemm_kernel<8>, grid, 256, row_gemm_smem<8>(), S, ga)));
    } else {
      const int tiles = pair_wide(p) ? p.n_chunks / 2 : p.n_chunks, pairs = c->sm_count / 2;
      int kbps = nK;
      if (2 * tiles <= pairs) {
        ks = std::min(kSplitMax, pairs / tiles);
        kbps = (nK + ks - 1) / ks;
        ks = (nK + kbps - 1) / kbps;
      }
      if (int e2 = encode_2d(c, &p.pmap, w.splitk, (uint64_t)ks * kPairRows, Nn, Nn, 128, true)) return e2;
      p.k_split = ks; p.kb_per_split = kbps; p.split_rows = kPairRows;
      LAUNCH(Lh, family, launch_pair_gemm(c, S, p));
    }
    if (fork) CU_OK(cudaStreamWaitEvent(s, c->join_ev, 0));
    if (family == F_GEMM_QKV) {                              // + RoPE at the cache position + append k / v to the cache
      QkvReduceArgs qa{};
      qa.partial = w.splitk; qa.k_split = ks; qa.split_rows = split_rows; qa.M = Ni; qa.N = Nn; qa.delta = any ? w.delta : nullptr;
      for (int i = 0; i < 3; ++i) qa.bias[i] = p.bias[i];
      qa.qkv = out_bf16; qa.n_q_heads = d.n_q_heads; qa.n_kv_heads = d.n_kv_heads; qa.dh = d.head_dim; qa.layer = layer;
      qa.rope_cs = d.rope_theta > 0 ? bb.rope_cs : nullptr;
      const long long n_thr = (long long)Ni * (d.n_q_heads + 2 * d.n_kv_heads) * (d.head_dim / 8);
      LAUNCH(Lh, family, (launch_k(qkv_reduce_rope_kernel, (unsigned)((n_thr + 255) / 256), 256, 0, S, qa, ka)));
      return FMX_OK;
    }
    if (p.mode == GM_RESID_F32 && row_norm_fused) {          // + the norm that follows the residual update
      ReduceNormArgs na{};
      na.partial = w.splitk; na.k_split = ks; na.split_rows = split_rows; na.N = Nn; na.delta = any ? w.delta : nullptr; na.bias = p.bias[0];
      na.X = w.X; na.Y = w.Xn; na.g = next_norm_g; na.b = next_norm_b; na.eps = d.norm_eps; na.rms = d.norm == FMX_NORM_RMSNORM;
      LAUNCH(Lh, family, (launch_k(reduce_resid_norm_kernel, (unsigned)Ni, (unsigned)((Nn / 4 + 31) / 32 * 32), 0, S, na)));
      return FMX_OK;
    }
    SplitKReduceArgs ra{};
    ra.partial = w.splitk; ra.k_split = ks; ra.split_rows = split_rows; ra.M = Ni; ra.N = Nn; ra.delta = any ? w.delta : nullptr;
    ra.mode = p.mode == GM_RESID_F32 ? 3 : p.mode == GM_OUT_BF16_SWIGLU ? 4 : p.mode == GM_OUT_BF16_GELU ? 1 : p.mode == GM_OUT_BF16_RELU ? 2 : 0;
    for (int i = 0; i < 3; ++i) { ra.bias[i] = p.bias[i]; ra.src_end_col[i] = p.src_end[i] >= (1 << 20) ? (1 << 30) : p.src_end[i] * 128; }
    ra.out_bf16 = out_bf16; ra.X = w.X; ra.ld_out = ld_out;
    const long long n_thr = (long long)Ni * (ra.mode == 4 ? Nn / 8 : Nn / 4);
    LAUNCH(Lh, family, (launch_k(splitk_reduce_kernel, (unsigned)((n_thr + 255) / 256), 256, 0, S, ra)));
    return FMX_OK;
  };

  // ---- S2: embed ----
  if (d.input_kind == FMX_INPUT_PATCH_LINEAR) {
    PackArgs pa{};
    pa.inputs = (const bf16 *)inputs; pa.perm = w.t.perm; pa.row_req = w.t.row_req; pa.row_pos = w.t.row_pos; pa.in_off = w.t.in_off;
    pa.N = Ni; pa.patch_dim = d.patch_dim; pa.Kp = bb.Kp; pa.has_cls = d.has_cls; pa.img_c = d.img_c; pa.img_hw = d.img_hw; pa.patch_hw = d.patch_hw;
    pa.task_ids = w.t.task_ids; pa.task_enc_ch = c->d_task_enc_ch;
    pa.task_enc_W = (const bf16 *const *)c->d_task_enc_W; pa.task_enc_b = (const bf16 *const *)c->d_task_enc_b;
    pa.series_len = (d.tokens_per_request - (d.has_cls ? 1 : 0)) * d.patch_dim;
    pa.A = w.Hid;
    pa.tpr = 128;
    while (pa.tpr > 8 && pa.tpr / 2 >= bb.Kp) pa.tpr /= 2;          // 8 .. 128 threads per row: tiny patches share a block
    LAUNCH(Lh, F_EMBED, (launch_k(pack_patches_kernel, (Ni + 128 / pa.tpr - 1) / (128 / pa.tpr), 128, 0, S, pa)));
    if (bb.Kp == 8 && c->o.embed_small) {
      // a one-k-block GEMM is all epilogue: tiny patches go through the CUDA-core kernel (kernels.cuh)
      LAUNCH(Lh, F_EMBED, (launch_k(embed_small_patch_kernel, dim3((Ni + kEmbRows - 1) / kEmbRows, (d.d_model / 4 + 255) / 256), 256, 0, S,
                                    (const bf16 *)w.Hid, (const bf16 *)bb.embed_Wpad, (const float *)bb.posb, (const int *)w.t.row_pos, Ni, d.d_model, w.X)));
    } else {
      if ((e = encode_2d(c, &mPk, w.Hid, Ni, bb.Kp, bb.Kp, 128))) return e;
      PairGemmParams p = base;
      p.mode = GM_EMBED_F32; p.amap = mPk; p.K = bb.Kp; p.n_chunks = d.d_model / 128;
      p.wmap[0] = bb.mEmbedW[wv(p)]; p.wmap_h[0] = bb.mEmbedW[1]; p.omap = oX; p.posb = bb.posb; p.ld_pos = d.d_model;
      LAUNCH(Lh, F_EMBED, launch_pair_gemm(c, S, p));
    }
  } else {
    EmbedArgs ea{};
    ea.inputs = inputs; ea.perm = w.t.perm; ea.row_req = w.t.row_req; ea.row_pos = w.t.row_pos; ea.in_off = w.t.in_off;
    ea.N = Ni; ea.d = d.d_model; ea.X = w.X; ea.table = (const bf16 *)d.embed_table; ea.pos = (const bf16 *)d.embed_pos;
    ea.vocab = d.vocab; ea.err = c->d_err;
    LAUNCH(Lh, F_EMBED, (launch_k(embed_rows_kernel, (Ni + 7) / 8, 256, 0, S, ea, d.input_kind == FMX_INPUT_TOKEN_IDS)));
  }

  // ---- layers ----
  const int rms = d.norm == FMX_NORM_RMSNORM;
  const float scale_log2 = 1.4426950408889634f / sqrtf((float)d.head_dim);
  bool rope_fused = false;
  for (int l = 0; l < d.n_layers; ++l) {
    if (!(row_norm_fused && l > 0))                          // (row mode: the previous layer's FFN-down reduction wrote Xn)
      LAUNCH(Lh, F_NORM, dispatch_norm(S, d.d_model, w.X, w.Xn, (const bf16 *)bb.norm1_g[l], (const bf16 *)bb.norm1_b[l], Ni, d.norm_eps, rms, rev()));
    {
      const int tgs[3] = {FMX_TGT_Q, FMX_TGT_K, FMX_TGT_V};
      PairGemmParams p = base;
      p.mode = GM_OUT_BF16; p.amap = mXn; p.K = d.d_model; p.n_chunks = bb.d_qkv / 128;
      if (can_fuse(p, 3)) shrink_fused(p, tgs, 3, l);
      else if ((e = shrink(mXn, d.d_model, tgs, 3, l))) return e;
      const int v = wv(p);
      p.wmap[0] = bb.mWq[v][l]; p.wmap[1] = bb.mWk[v][l]; p.wmap[2] = bb.mWv[v][l];
      p.wmap_h[0] = bb.mWq[1][l]; p.wmap_h[1] = bb.mWk[1][l]; p.wmap_h[2] = bb.mWv[1][l];
      p.src_end[0] = bb.d_q / 128; p.src_end[1] = (bb.d_q + bb.d_kv) / 128; p.src_end[2] = 1 << 30;
      p.bias[0] = (const bf16 *)bb.bq[l]; p.bias[1] = (const bf16 *)bb.bk[l]; p.bias[2] = (const bf16 *)bb.bv[l];
      set_lora(p, 0, FMX_TGT_Q, l); set_lora(p, 1, FMX_TGT_K, l); set_lora(p, 2, FMX_TGT_V, l);
      p.omap = oQKV;
      // head_dim 128: a 128-column chunk is one head, so RoPE is applied in the GEMM epilogue (fp32, one rounding)
      // (a decode iteration splits the K axis of this GEMM and rotates q / k with rope_kernel after the reduction)
      rope_fused = c->o.rope_fused && d.rope_theta > 0 && d.head_dim == 128 && pair_wide(p) && !(kv && kv->decode && w.splitk && bb.row_bt && w.n_tiles == 1);
      if (rope_fused) { p.rope_cs = bb.rope_cs_t; p.rope_ld = d.max_seq; p.rope_src_mask = 3; p.row_pos = rope_pos; }
      p.reverse = rev();
      if ((e = project(p, F_GEMM_QKV, w.QKV, bb.d_qkv, w.Xn, tgs, 3, l, bb.Wq[l], bb.Wk[l], bb.Wv[l]))) return e;
    }
    if (d.rope_theta > 0 && !rope_fused && !row_mode) {
      const int nh = d.n_q_heads + d.n_kv_heads;
      const long long total = (long long)Ni * nh * (d.head_dim / 16);
      LAUNCH(Lh, F_ROPE, (launch_k(rope_kernel, (unsigned)((total + 255) / 256), 256, 0, S, w.QKV, bb.d_qkv, rope_pos, bb.rope_cs, Ni, nh, d.head_dim)));
    }
    if (kv && !row_mode) LAUNCH(Lh, F_ATTN, (launch_k(kv_append_kernel, (Ni + 7) / 8, 256, 0, S, (const bf16 *)w.QKV, bb.d_qkv, bb.d_q, bb.d_q + bb.d_kv, Ni, l, ka)));
    if (kv && kv->decode) {
      DecAttnArgs da{};
      da.qkv = w.QKV; da.out = w.AttnO; da.ld_qkv = bb.d_qkv; da.ld_out = bb.d_q; da.n_q_heads = d.n_q_heads; da.n_kv_heads = d.n_kv_heads;
      da.layer = l; da.scale_log2 = scale_log2; da.kc_keys = dec_chunk_keys(d.max_seq); da.part = w.dec_part; da.cnt = w.dec_cnt;
      dim3 grid(B, d.n_kv_heads, dec_chunks_cap(d.max_seq));
      if (d.head_dim == 32) LAUNCH(Lh, F_ATTN, (launch_k(decode_attention_kernel<32>, grid, 128, decode_attention_smem<32>(), S, da, ka)));
      else if (d.head_dim == 64) LAUNCH(Lh, F_ATTN, (launch_k(decode_attention_kernel<64>, grid, 128, decode_attention_smem<64>(), S, da, ka)));
      else LAUNCH(Lh, F_ATTN, (launch_k(decode_attention_kernel<128>, grid, 128, decode_attention_smem<128>(), S, da, ka)));
      rev();
    } else if (!bb.relb && c->o.attn_impl == FMX_ATTN_AUTO && attn_pair64_ok(c->o, d.head_dim, d.n_q_heads, max_len)) {
      AttnPairArgs pa2{};
      pa2.qkv_map = mQKV64; pa2.out = w.AttnO; pa2.cu_tok = w.t.cu_tok; pa2.ld_out = bb.d_q; pa2.n_req = B;
      pa2.n_q_heads = d.n_q_heads; pa2.n_kv_heads = d.n_kv_heads; pa2.causal = d.causal; pa2.scale_log2 = scale_log2;
      pa2.reverse = rev();
      LAUNCH(Lh, F_ATTN, launch_attention_pair64(S, c->sm_count, pa2));
    } else if (attn_use_tc(c->o.attn_impl, d.head_dim, max_len)) {
      AttnTcArgs ta{};
      ta.relb = bb.relb; ta.relb_ld = bb.relb_ld; ta.relb_off = bb.relb_off;
      ta.qkv_map = mQKV64; ta.out = w.AttnO; ta.cu_tok = w.t.cu_tok; ta.ld_out = bb.d_q;
      ta.n_q_heads = d.n_q_heads; ta.n_kv_heads = d.n_kv_heads; ta.causal = d.causal; ta.scale_log2 = scale_log2;
      ta.reverse = rev();
      LAUNCH(Lh, F_ATTN, launch_attention_tc(S, d.head_dim, max_len, d.n_q_heads, B, ta));
    } else {
      AttnArgs aa{};
      aa.qkv = w.QKV; aa.out = w.AttnO; aa.cu_tok = w.t.cu_tok; aa.ld_qkv = bb.d_qkv; aa.ld_out = bb.d_q;
      aa.n_q_heads = d.n_q_heads; aa.n_kv_heads = d.n_kv_heads; aa.causal = d.causal; aa.scale_log2 = scale_log2;
      aa.relb = bb.relb; aa.relb_ld = bb.relb_ld; aa.relb_off = bb.relb_off;
      dim3 grid((max_len + kAttnBQ - 1) / kAttnBQ, d.n_q_heads, B);
      if (max_len <= 64 && c->o.attn_short && !bb.relb) LAUNCH(Lh, F_ATTN, launch_attention_short(S, c->sm_count, d.head_dim, B, aa));
      else LAUNCH(Lh, F_ATTN, launch_attention(S, d.head_dim, grid, aa));
    }
    {
      const int tgs[1] = {FMX_TGT_O};
      PairGemmParams p = base;
      p.mode = GM_RESID_F32; p.amap = mAttnO; p.K = bb.d_q; p.n_chunks = d.d_model / 128;
      if (can_fuse(p, 1)) shrink_fused(p, tgs, 1, l);
      else if ((e = shrink(mAttnO, bb.d_q, tgs, 1, l))) return e;
      p.wmap[0] = bb.mWo[wv(p)][l]; p.wmap_h[0] = bb.mWo[1][l]; p.bias[0] = (const bf16 *)bb.bo[l];
      set_lora(p, 0, FMX_TGT_O, l);
      p.omap = oX;
      p.reverse = rev();
      next_norm_g = (const bf16 *)bb.norm2_g[l]; next_norm_b = (const bf16 *)bb.norm2_b[l];
      if ((e = project(p, F_GEMM_O, nullptr, d.d_model, w.AttnO, tgs, 1, l, bb.Wo[l], nullptr, nullptr))) return e;
    }
    if (!row_norm_fused)
      LAUNCH(Lh, F_NORM, dispatch_norm(S, d.d_model, w.X, w.Xn, (const bf16 *)bb.norm2_g[l], (const bf16 *)bb.norm2_b[l], Ni, d.norm_eps, rms, rev()));
    if (d.act == FMX_ACT_SWIGLU) {
      const int tgs[2] = {FMX_TGT_GATE, FMX_TGT_UP};
      PairGemmParams p = base;
      p.mode = GM_OUT_BF16_SWIGLU; p.amap = mXn; p.K = d.d_model; p.n_chunks = 2 * d.d_ffn / 128; p.interleave2 = 1;
      if (can_fuse(p, 2)) shrink_fused(p, tgs, 2, l);
      else if ((e = shrink(mXn, d.d_model, tgs, 2, l))) return e;
      p.wmap[0] = bb.mWgate[0][l]; p.wmap[1] = bb.mWup[0][l];
      p.bias[0] = (const bf16 *)bb.bgate[l]; p.bias[1] = (const bf16 *)bb.bup[l];
      set_lora(p, 0, FMX_TGT_GATE, l); set_lora(p, 1, FMX_TGT_UP, l);
      p.omap = oHid;
      p.reverse = rev();
      if ((e = project(p, F_GEMM_FFN_IN, w.Hid, d.d_ffn, w.Xn, tgs, 2, l, bb.Wgate[l], bb.Wup[l], nullptr))) return e;
    } else {
      const int tgs[1] = {FMX_TGT_UP};
      PairGemmParams p = base;
      p.mode = d.act == FMX_ACT_GELU_ERF ? GM_OUT_BF16_GELU : GM_OUT_BF16_RELU; p.amap = mXn; p.K = d.d_model; p.n_chunks = d.d_ffn / 128;
      if (can_fuse(p, 1)) shrink_fused(p, tgs, 1, l);
      else if ((e = shrink(mXn, d.d_model, tgs, 1, l))) return e;
      p.wmap[0] = bb.mWup[wv(p)][l]; p.wmap_h[0] = bb.mWup[1][l]; p.bias[0] = (const bf16 *)bb.bup[l];
      set_lora(p, 0, FMX_TGT_UP, l);
      p.omap = oHid;
      p.reverse = rev();
      if ((e = project(p, F_GEMM_FFN_IN, w.Hid, d.d_ffn, w.Xn, tgs, 1, l, bb.Wup[l], nullptr, nullptr))) return e;
    }
    {
      const int tgs[1] = {FMX_TGT_DOWN};
      PairGemmParams p = base;
      p.mode = GM_RESID_F32; p.amap = mHid; p.K = d.d_ffn; p.n_chunks = d.d_model / 128;
      if (can_fuse(p, 1)) shrink_fused(p, tgs, 1, l);
      else if ((e = shrink(mHid, d.d_ffn, tgs, 1, l))) return e;
      p.wmap[0] = bb.mWdown[wv(p)][l]; p.wmap_h[0] = bb.mWdown[1][l]; p.bias[0] = (const bf16 *)bb.bdown[l];
      set_lora(p, 0, FMX_TGT_DOWN, l);
      p.omap = oX;
      p.reverse = rev();
      next_norm_g = l + 1 < d.n_layers ? (const bf16 *)bb.norm1_g[l + 1] : nullptr;
      next_norm_b = l + 1 < d.n_layers ? (const bf16 *)bb.norm1_b[l + 1] : nullptr;
      if ((e = project(p, F_GEMM_FFN_OUT, nullptr, d.d_model, w.Hid, tgs, 1, l, bb.Wdown[l], nullptr, nullptr))) return e;
    }
  }
  // ---- S4-S6 (skipped by a decode step that wants LM scores only) ----
  if (outputs != nullptr) {
  PoolArgs pa{};
  pa.X = w.X; pa.g = (const bf16 *)d.final_g; pa.b = (const bf16 *)d.final_b; pa.cu_tok = w.t.cu_tok; pa.task_sorted = w.t.task_sorted;
  pa.task_head_kind = c->d_task_head_kind; pa.feat = w.feat; pa.Fn = w.Xn; pa.d = d.d_model; pa.eps = d.norm_eps; pa.rms = rms;
  LAUNCH(Lh, F_POOL, dispatch_pool(S, d.d_model, B, pa));
  HeadArgs ha{};
  ha.feat = w.feat; ha.Fn = w.Xn; ha.cu_tok = w.t.cu_tok; ha.task_sorted = w.t.task_sorted; ha.perm = w.t.perm; ha.out_off = w.t.out_off;
  ha.task_head_kind = c->d_task_head_kind; ha.task_head_out = c->d_task_head_out;
  ha.task_head_W = (const bf16 *const *)c->d_task_head_W; ha.task_head_b = (const bf16 *const *)c->d_task_head_b;
  ha.out = outputs; ha.d = d.d_model;
  ha.task_head_w1 = c->d_task_head_w1;
  ha.task_head_W2 = (const bf16 *const *)c->d_task_head_W2; ha.task_head_b2 = (const bf16 *const *)c->d_task_head_b2;
  const int max_hidden = bs.max_hidden, max_out2 = bs.max_out2;      // MLP heads in this batch
  if (max_hidden > 0) { ha.hid = w.head_hid; ha.ld_hid = max_hidden; }      // max_hidden <= kMaxHeadHidden by registration
  const bool any_flat = bs.any_flat, any_pooled = bs.any_pooled;
  const int max_out_flat = bs.max_out_flat;
  ha.skip_flatten = (any_flat && c->o.head_tiled) ? 1 : 0;
  if (any_pooled || !ha.skip_flatten) LAUNCH(Lh, F_HEAD, (launch_k(head_kernel, dim3(B, (max_out + 7) / 8), 256, 0, S, ha)));
  if (ha.skip_flatten) {
    // tensor-core path: K (= tokens x d_model, the same for every FLATTEN task of a fixed-length backbone) must split into
    // n_kc chunks x 8 warps x multiples of 32 features; the chunk partials live in the caller's workspace
    const long long Kf = (long long)d.tokens_per_request * d.d_model;
    const int groups = (B + 15) / 16, ogs = (max_out_flat + 31) / 32;
    int n_kc = 0;
    if (c->o.head_tiled == 2 && d.tokens_per_request > 0)
      for (int k = 1; k <= 16; k *= 2)
        if (Kf % (256ll * k) == 0) { n_kc = k; if ((long long)groups * ogs * k >= 8ll * c->sm_count) break; }   // >= 8 CTAs per SM, i.e. four rounds of the two resident ones: a CTA streams one task's weights per pass at single-SM bandwidth (measured on cfg5: 1 / 2 / 4 / 8 per SM = 0.46 / 0.32 / 0.27 / 0.24 ms)
    while (n_kc > 0 && (size_t)groups * ogs * n_kc * 512 > w.head_part_floats) n_kc /= 2;     // fit the workspace's partial budget
    if (n_kc > 0) {
      LAUNCH(Lh, F_HEAD, (launch_k(head_flatten_mma_kernel, dim3(groups, ogs, n_kc), 256, 0, S, ha, B, n_kc, w.head_part)));
      LAUNCH(Lh, F_HEAD, (launch_k(head_flatten_reduce_kernel, dim3(groups, ogs), 512, 0, S, ha, B, n_kc, (const float *)w.head_part)));
    } else {
      LAUNCH(Lh, F_HEAD, (launch_k(head_flatten_kernel, dim3((B + 3) / 4, (max_out + 3) / 4), 256, 0, S, ha, B)));
    }
  }

  if (bs.any_dense)                                      // dense (per-token) heads: one warp per token row of a dense task's request
    LAUNCH(Lh, F_HEAD, (launch_k(head_dense_kernel, (Ni + 7) / 8, 256, 0, S, ha, Ni, (const int *)w.t.row_req, (const int *)w.t.row_pos)));
  if (max_hidden > 0)                                    // second layer of the MLP heads (the first wrote relu(W feat + b) to hid)
    LAUNCH(Lh, F_HEAD, (launch_k(head_mlp2_kernel, dim3(B, (max_out2 + 7) / 8), 256, 0, S, ha)));
  }

  // ---- LM head (NEXT-3): scores of every request's last token, greedy next token; original request order ----
  if (kv && (kv->scores || kv->next_tokens)) {
    switch (d.d_model / 128) {
#define FMX_LRN(V) case V: LAUNCH(Lh, F_POOL, (launch_k(last_row_norm_kernel<V>, (B + 7) / 8, 256, 0, S, (const float *)w.X, (const int *)w.t.cu_tok, w.Fl, (const bf16 *)d.final_g, (const bf16 *)d.final_b, B, d.norm_eps, rms))); break;
      FMX_LRN(1) FMX_LRN(2) FMX_LRN(4) FMX_LRN(6) FMX_LRN(8) FMX_LRN(12) FMX_LRN(16)
#undef FMX_LRN
    }
    PairGemmParams p{};
    p.M = B; p.K = d.d_model; p.n_chunks = bb.lm_vocab / 128; p.n_ptiles = (B + kPairRows - 1) / kPairRows; p.mode = GM_OUT_F32;
    for (int i = 0; i < 3; ++i) { p.lora_tgt[i] = -1; p.src_end[i] = 1 << 30; }
    CUtensorMap mFl, oLm;
    if ((e = encode_2d(c, &mFl, w.Fl, B, d.d_model, d.d_model, 128))) return e;
    if ((e = encode_2d(c, &oLm, w.lm_scores, B, bb.lm_vocab, bb.lm_vocab, 128, true))) return e;
    p.amap = mFl; p.omap = oLm; p.wmap[0] = bb.mLm[pair_wide(p) ? 0 : 1]; p.wmap_h[0] = bb.mLm[1];
    LAUNCH(Lh, F_HEAD, launch_pair_gemm(c, S, p));
    LAUNCH(Lh, F_HEAD, (launch_k(scores_out_kernel, B, 256, 0, S, (const float *)w.lm_scores, (const int *)w.t.perm, bb.lm_vocab, kv->scores, kv->next_tokens)));
  }

  {
    void *bufs[7] = {w.X, w.Xn, w.QKV, w.AttnO, w.Hid, w.U, w.feat};
    size_t sz[7] = {sizeof(float) * N * d.d_model, sizeof(bf16) * N * d.d_model, sizeof(bf16) * N * bb.d_qkv, sizeof(bf16) * N * bb.d_q,
                    sizeof(bf16) * N * d.d_ffn, sizeof(bf16) * (size_t)w.n_blk_cap * kPairRows * 192, sizeof(float) * (size_t)B * d.d_model};
    for (int i = 0; i < 7; ++i) { c->last_buf[i] = bufs[i]; c->last_buf_bytes[i] = sz[i]; }
  }
  c->last_t = w.t; c->last_B = B; c->last_T = T; c->last_n_tiles = w.n_tiles; c->last_stream = s; c->last_launches = Lh.count;
  return graph_capture ? FMX_OK : note_forward(c, s);
}

// The forward with the context's one-entry CUDA-graph cache in front of it (c->mu held by the caller).  The graph holds the
// kernels only; ids / lengths are copied to the device tables before every launch, so the graph is keyed by the call's
// buffers and BatchShape, not by the ids: a serving loop whose batches change but keep their shape (a fixed-length backbone
// at a fixed batch size) replays it on every step.  The 2nd call with the same key is captured, later ones replay; a step
// of ~200 short kernels loses ~4 % to launch gaps otherwise (cfg2: 11.55 -> 11.09 ms).
static int forward_cached(fmx_ctx *c, Backbone *bb, fmx_backbone_t h, const void *inputs, const int32_t *task_ids, const int32_t *lengths,
                          int32_t n_req, float *outputs, void *workspace, size_t workspace_bytes, cudaStream_t s, const KvCall *kv = nullptr) {
  BatchShape bs;
  if (int e = batch_shape(c, *bb, task_ids, lengths, n_req, bs)) return e;
  const bool graphable = c->o.graph && !c->prof_on && s != nullptr && s != cudaStreamLegacy && s != cudaStreamPerThread;
  if (graphable) {
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    CU_OK(cudaStreamIsCapturing(s, &st));
    if (st == cudaStreamCaptureStatusNone) {
      fmx_ctx::CallKey key;
      key.bb = h; key.B = n_req; key.inputs = inputs; key.outputs = outputs; key.workspace = workspace; key.ws_bytes = workspace_bytes;
      key.stream = s; key.gen = c->config_gen; key.shape = bs;
      key.fuse = c->o.shrink_fused == 2 || (c->o.shrink_fused == 1 && bs.n_blk <= c->sm_count / 2);
      if (kv) { key.kv_cache = kv->cache; key.scores = kv->scores; key.next_tokens = kv->next_tokens; key.kv_mode = kv->decode ? 2 : 1; key.n_slots = kv->n_slots; }
      const bool hit = c->graph_exec && key == c->graph_key;
      if (hit || key == c->last_key) {
        if (reinterpret_cast<uintptr_t>(workspace) & 1023) return fmx_fail(FMX_E_WORKSPACE, "forward_mixed: workspace must be 1024-byte aligned");
        const Workspace w = carve(*bb, workspace, n_req, bs.N, c->n_slots);
        if (w.bytes > workspace_bytes) return fmx_fail(FMX_E_WORKSPACE, "forward_mixed: workspace %zu B < required %zu B", workspace_bytes, w.bytes);
        if (hit) {
          if (int e = stage_ids(c, w, task_ids, lengths, n_req, s, kv ? kv->slots : nullptr, kv ? kv->pos0 : nullptr)) return e;
          CU_OK(cudaGraphLaunch(c->graph_exec, s));
          c->last_launches = c->graph_launches; c->last_stream = s;
          c->last_t = w.t; c->last_B = n_req; c->last_T = c->n_slots; c->last_n_tiles = w.n_tiles;
          ++c->graph_replays;
          return note_forward(c, s);
        }
        if (c->graph_exec) {                          // the old graph may still be running
          CU_OK(cudaStreamSynchronize(c->graph_key.stream));
          cudaGraphExecDestroy(c->graph_exec);
          c->graph_exec = nullptr;
        }
        if (int e = stage_ids(c, w, task_ids, lengths, n_req, s, kv ? kv->slots : nullptr, kv ? kv->pos0 : nullptr)) return e;
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
          const int e = forward_impl(c, *bb, inputs, task_ids, lengths, n_req, outputs, workspace, workspace_bytes, s, bs, true, kv);
          const cudaError_t ce = cudaStreamEndCapture(s, &graph);
          if (e == FMX_OK && ce == cudaSuccess && graph && cudaGraphInstantiate(&c->graph_exec, graph, 0) == cudaSuccess) {
            cudaGraphDestroy(graph);
            c->graph_key = key;
            c->graph_launches = c->last_launches;
            CU_OK(cudaGraphLaunch(c->graph_exec, s));
            return note_forward(c, s);
          }
          if (graph) cudaGraphDestroy(graph);
          c->graph_exec = nullptr;
          cudaGetLastError();
          if (e != FMX_OK) return e;
        } else {
          cudaGetLastError();
        }
        // capture failed: the ids are staged already; run the kernels plainly (graph_capture = true skips the staging only)
        if (int e = forward_impl(c, *bb, inputs, task_ids, lengths, n_req, outputs, workspace, workspace_bytes, s, bs, true, kv)) return e;
        return note_forward(c, s);
      }
      c->last_key = std::move(key);
    }
  }
  return forward_impl(c, *bb, inputs, task_ids, lengths, n_req, outputs, workspace, workspace_bytes, s, bs, false, kv);
}

// A device-side error of an EARLIER forward (the word is mapped host memory the kernels write): reported by the next call.
static int poll_device_error(fmx_ctx *c) {
  const unsigned e = *(volatile unsigned *)c->h_err;
  if (!e) return FMX_OK;
  *(volatile unsigned *)c->h_err = 0;
  if (e & 2u)
    return fmx_fail(FMX_E_CUDA, "an earlier forward's fused LoRA shrink timed out waiting for CTA pairs that never became resident (another "
                                "kernel held their SMs); its outputs are invalid.  FMX_OPT_SHRINK_FUSED needs the GPU to itself (device error word 0x%x)", e);
  return fmx_fail(FMX_E_INVALID_ARG, "an earlier forward read token ids outside [0, vocab): those rows were embedded as zeros (device error word 0x%x)", e);
}

int fmx_poll_error(fmx_ctx *c) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "poll_error: NULL ctx");
  std::lock_guard<std::mutex> lk(c->mu);
  return poll_device_error(c);
}

int fmx_forward_mixed(fmx_ctx *c, fmx_backbone_t h, const void *inputs, const int32_t *task_ids, const int32_t *lengths,
                      int32_t n_req, float *outputs, void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed: NULL ctx");
  if (n_req < 0) return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed: n_req < 0");
  std::lock_guard<std::mutex> lk(c->mu);
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "forward_mixed: unknown backbone %d", h);
  if (n_req == 0) return FMX_OK;
  if (n_req > FMX_MAX_REQUESTS) return fmx_fail(FMX_E_CAPACITY, "forward_mixed: %d requests > %d", n_req, FMX_MAX_REQUESTS);
  if (!inputs || !task_ids || !lengths || !outputs || !workspace) return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed: NULL pointer");
  CU_OK(cudaSetDevice(c->device));
  if (int e = poll_device_error(c)) return e;
  return forward_cached(c, bb, h, inputs, task_ids, lengths, n_req, outputs, workspace, workspace_bytes, (cudaStream_t)cuda_stream);
}

// Layout of the host-path workspace: [forward workspace for this batch | input staging | output staging].
int fmx_forward_mixed_host(fmx_ctx *c, fmx_backbone_t h, const void *inputs_host, size_t inputs_bytes, const int32_t *task_ids,
                           const int32_t *lengths, int32_t n_req, float *outputs_host, void *workspace, size_t workspace_bytes,
                           void *cuda_stream) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed_host: NULL ctx");
  if (n_req < 0) return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed_host: n_req < 0");
  std::lock_guard<std::mutex> lk(c->mu);
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "forward_mixed_host: unknown backbone %d", h);
  if (n_req == 0) return FMX_OK;
  if (n_req > FMX_MAX_REQUESTS) return fmx_fail(FMX_E_CAPACITY, "forward_mixed_host: %d requests > %d", n_req, FMX_MAX_REQUESTS);
  if (!inputs_host || !task_ids || !lengths || !outputs_host || !workspace) return fmx_fail(FMX_E_INVALID_ARG, "forward_mixed_host: NULL pointer");
  std::vector<int64_t> off(n_req + 1);
  if (int e = output_layout_locked(c, task_ids, lengths, n_req, off.data())) return e;
  long long N = 0;
  for (int i = 0; i < n_req; ++i) N += std::max(lengths[i], 0);
  if (N < 1 || N > (1ll << 24)) return fmx_fail(FMX_E_BAD_LENGTH, "forward_mixed_host: %lld tokens", N);
  if (reinterpret_cast<uintptr_t>(workspace) & 1023) return fmx_fail(FMX_E_WORKSPACE, "forward_mixed_host: workspace must be 1024-byte aligned");
  const size_t fwd_bytes = align_up(carve(*bb, nullptr, n_req, N, c->n_slots).bytes, 1024);
  const size_t out_bytes = (size_t)off[n_req] * sizeof(float);
  const size_t need = fwd_bytes + align_up(inputs_bytes, 1024) + align_up(out_bytes, 1024);
  if (need > workspace_bytes)
    return fmx_fail(FMX_E_WORKSPACE, "forward_mixed_host: workspace %zu B < required %zu B (fmx_host_workspace_bytes)", workspace_bytes, need);
  CU_OK(cudaSetDevice(c->device));
  if (int e = poll_device_error(c)) return e;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  uint8_t *in_stage = static_cast<uint8_t *>(workspace) + fwd_bytes;
  float *out_stage = reinterpret_cast<float *>(in_stage + align_up(inputs_bytes, 1024));
  CU_OK(cudaMemcpyAsync(in_stage, inputs_host, inputs_bytes, cudaMemcpyHostToDevice, s));
  if (int e = forward_cached(c, bb, h, in_stage, task_ids, lengths, n_req, out_stage, workspace, fwd_bytes, s)) return e;
  CU_OK(cudaMemcpyAsync(outputs_host, out_stage, out_bytes, cudaMemcpyDeviceToHost, s));
  CU_OK(cudaStreamSynchronize(s));
  return poll_device_error(c);
}

// ---------------------------------------------------------------- token decode with a key / value cache (NEXT-3)
int fmx_register_lm_head(fmx_ctx *c, fmx_backbone_t h, const void *W, int32_t vocab) {
  if (!c || !W) return fmx_fail(FMX_E_INVALID_ARG, "register_lm_head: NULL argument");
  std::lock_guard<std::mutex> lk(c->mu);
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "register_lm_head: unknown backbone %d", h);
  if (vocab < 128 || vocab % 128) return fmx_fail(FMX_E_SHAPE, "register_lm_head: vocab %d must be a positive multiple of 128", vocab);
  if (bb->relb) return fmx_fail(FMX_E_SHAPE, "register_lm_head: backbones with a relative-position bias do not serve token decode");
  CUtensorMap m0, m1;
  if (int e = encode_2d(c, &m0, W, vocab, bb->d.d_model, bb->d.d_model, 128)) return e;
  if (int e = encode_2d(c, &m1, W, vocab, bb->d.d_model, bb->d.d_model, 64)) return e;
  bb->lm_head = (const bf16 *)W; bb->lm_vocab = vocab; bb->mLm[0] = m0; bb->mLm[1] = m1;
  ++c->config_gen;
  return FMX_OK;
}

int fmx_kv_cache_bytes(fmx_ctx *c, fmx_backbone_t h, int32_t n_slots, size_t *bytes) {
  if (!c || !bytes) return fmx_fail(FMX_E_INVALID_ARG, "kv_cache_bytes: NULL argument");
  std::lock_guard<std::mutex> lk(c->mu);
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "kv_cache_bytes: unknown backbone %d", h);
  if (n_slots < 1 || n_slots > (1 << 20)) return fmx_fail(FMX_E_CAPACITY, "kv_cache_bytes: n_slots %d", n_slots);
  *bytes = (size_t)n_slots * bb->d.n_layers * 2 * bb->d.max_seq * bb->d_kv * sizeof(bf16);
  return FMX_OK;
}

// Shared validation + launch of fmx_prefill / fmx_decode_step (c->mu held).
static int kv_forward(fmx_ctx *c, fmx_backbone_t h, const char *who, const void *inputs, const int32_t *task_ids, const int32_t *lengths,
                      const int32_t *slots, const int32_t *pos0, int32_t n_req, float *outputs, float *scores, int32_t *next_tokens,
                      void *kv_cache, int32_t n_slots, void *workspace, size_t workspace_bytes, cudaStream_t s) {
  Backbone *bb = get_bb(c, h);
  if (!bb) return fmx_fail(FMX_E_UNKNOWN_BACKBONE, "%s: unknown backbone %d", who, h);
  if (n_req == 0) return FMX_OK;
  if (n_req > FMX_MAX_REQUESTS) return fmx_fail(FMX_E_CAPACITY, "%s: %d requests > %d", who, n_req, FMX_MAX_REQUESTS);
  if (!inputs || !task_ids || !slots || !kv_cache || !workspace) return fmx_fail(FMX_E_INVALID_ARG, "%s: NULL pointer", who);
  const fmx_backbone_desc &d = bb->d;
  if (!d.causal) return fmx_fail(FMX_E_SHAPE, "%s: a key / value cache needs a causal backbone", who);
  if ((scores || next_tokens) && !bb->lm_head) return fmx_fail(FMX_E_INVALID_ARG, "%s: scores / next_tokens need fmx_register_lm_head", who);
  if (reinterpret_cast<uintptr_t>(kv_cache) & 15) return fmx_fail(FMX_E_INVALID_ARG, "%s: kv_cache must be 16-byte aligned", who);
  if (n_slots < 1) return fmx_fail(FMX_E_INVALID_ARG, "%s: n_slots < 1", who);
  std::vector<unsigned char> seen((size_t)n_slots, 0);
  std::vector<int32_t> ones;
  if (pos0) { ones.assign(n_req, 1); lengths = ones.data(); }          // a decode step: one token per request
  else if (!lengths) return fmx_fail(FMX_E_INVALID_ARG, "%s: NULL lengths", who);
  for (int i = 0; i < n_req; ++i) {
    if (slots[i] < 0 || slots[i] >= n_slots) return fmx_fail(FMX_E_INVALID_ARG, "%s: request %d: cache slot %d not in [0, %d)", who, i, slots[i], n_slots);
    if (seen[slots[i]]) return fmx_fail(FMX_E_INVALID_ARG, "%s: cache slot %d is used by two requests of the batch", who, slots[i]);
    seen[slots[i]] = 1;
    if (pos0 && (pos0[i] < 0 || pos0[i] >= d.max_seq))
      return fmx_fail(FMX_E_BAD_LENGTH, "%s: request %d: %d cached tokens, the cache holds max_seq = %d", who, i, pos0[i], d.max_seq);
  }
  CU_OK(cudaSetDevice(c->device));
  if (int e = poll_device_error(c)) return e;
  KvCall kv;
  kv.cache = (bf16 *)kv_cache; kv.n_slots = n_slots; kv.slots = slots; kv.pos0 = pos0; kv.scores = scores; kv.next_tokens = next_tokens;
  kv.decode = pos0 != nullptr;
  return forward_cached(c, bb, h, inputs, task_ids, lengths, n_req, outputs, workspace, workspace_bytes, s, &kv);
}

int fmx_prefill(fmx_ctx *c, fmx_backbone_t h, const void *inputs, const int32_t *task_ids, const int32_t *lengths, const int32_t *slots,
                int32_t n_req, float *outputs, float *scores, int32_t *next_tokens, void *kv_cache, int32_t n_slots, void *workspace,
                size_t workspace_bytes, void *cuda_stream) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "prefill: NULL ctx");
  if (n_req < 0) return fmx_fail(FMX_E_INVALID_ARG, "prefill: n_req < 0");
  std::lock_guard<std::mutex> lk(c->mu);
  return kv_forward(c, h, "prefill", inputs, task_ids, lengths, slots, nullptr, n_req, outputs, scores, next_tokens, kv_cache, n_slots,
                    workspace, workspace_bytes, (cudaStream_t)cuda_stream);
}

int fmx_decode_step(fmx_ctx *c, fmx_backbone_t h, const int32_t *tokens, const int32_t *task_ids, const int32_t *slots, const int32_t *positions,
                    int32_t n_req, float *scores, int32_t *next_tokens, void *kv_cache, int32_t n_slots, void *workspace,
                    size_t workspace_bytes, void *cuda_stream) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "decode_step: NULL ctx");
  if (n_req < 0) return fmx_fail(FMX_E_INVALID_ARG, "decode_step: n_req < 0");
  if (n_req > 0 && !positions) return fmx_fail(FMX_E_INVALID_ARG, "decode_step: NULL positions");
  std::lock_guard<std::mutex> lk(c->mu);
  Backbone *bb = get_bb(c, h);
  if (bb && bb->d.input_kind != FMX_INPUT_TOKEN_IDS) return fmx_fail(FMX_E_SHAPE, "decode_step: the backbone does not take token ids");
  if (n_req > 0 && !scores && !next_tokens) return fmx_fail(FMX_E_INVALID_ARG, "decode_step: neither scores nor next_tokens requested");
  return kv_forward(c, h, "decode_step", tokens, task_ids, nullptr, slots, positions, n_req, nullptr, scores, next_tokens, kv_cache, n_slots,
                    workspace, workspace_bytes, (cudaStream_t)cuda_stream);
}

int fmx_debug_get_segments(fmx_ctx *c, int32_t *perm, int32_t *inv_perm, int32_t *task_req_off, int32_t *cu_tok, int32_t *task_tok_off) {
  if (!c || c->last_B == 0) return fmx_fail(FMX_E_INVALID_ARG, "debug_get_segments: no forward has run");
  CU_OK(cudaStreamSynchronize(c->last_stream));
  const SegTables &t = c->last_t;
  const int B = c->last_B, T = c->last_T;
  if (perm) CU_OK(cudaMemcpy(perm, t.perm, sizeof(int) * B, cudaMemcpyDeviceToHost));
  if (inv_perm) CU_OK(cudaMemcpy(inv_perm, t.inv_perm, sizeof(int) * B, cudaMemcpyDeviceToHost));
  if (task_req_off) CU_OK(cudaMemcpy(task_req_off, t.task_req_off, sizeof(int) * (T + 1), cudaMemcpyDeviceToHost));
  if (cu_tok) CU_OK(cudaMemcpy(cu_tok, t.cu_tok, sizeof(int) * (B + 1), cudaMemcpyDeviceToHost));
  if (task_tok_off) CU_OK(cudaMemcpy(task_tok_off, t.task_tok_off, sizeof(int) * (T + 1), cudaMemcpyDeviceToHost));
  return FMX_OK;
}

int fmx_debug_get_tiles(fmx_ctx *c, int32_t *n_tiles, int32_t *n_blocks, int32_t *blocks, int32_t cap) {
  if (!c || c->last_B == 0) return fmx_fail(FMX_E_INVALID_ARG, "debug_get_tiles: no forward has run");
  CU_OK(cudaStreamSynchronize(c->last_stream));
  const SegTables &t = c->last_t;
  int nb = 0;
  CU_OK(cudaMemcpy(&nb, t.n_blk, sizeof(int), cudaMemcpyDeviceToHost));
  if (n_tiles) *n_tiles = c->last_n_tiles;
  if (n_blocks) *n_blocks = nb;
  if (blocks) {
    const int n = std::min(nb, cap);
    std::vector<int> a(n), b(n), lo(n), hi(n);
    CU_OK(cudaMemcpy(a.data(), t.blk_tile, sizeof(int) * n, cudaMemcpyDeviceToHost));
    CU_OK(cudaMemcpy(b.data(), t.blk_task, sizeof(int) * n, cudaMemcpyDeviceToHost));
    CU_OK(cudaMemcpy(lo.data(), t.blk_lo, sizeof(int) * n, cudaMemcpyDeviceToHost));
    CU_OK(cudaMemcpy(hi.data(), t.blk_hi, sizeof(int) * n, cudaMemcpyDeviceToHost));
    for (int i = 0; i < n; ++i) { blocks[4 * i] = a[i]; blocks[4 * i + 1] = b[i]; blocks[4 * i + 2] = lo[i]; blocks[4 * i + 3] = hi[i]; }
  }
  return FMX_OK;
}

int fmx_debug_read(fmx_ctx *c, int which, void *host, size_t bytes) {
  if (!c || c->last_B == 0 || which < 0 || which > 6 || !host) return fmx_fail(FMX_E_INVALID_ARG, "debug_read: bad argument or no forward has run");
  if (bytes > c->last_buf_bytes[which]) return fmx_fail(FMX_E_INVALID_ARG, "debug_read: %zu > %zu bytes", bytes, c->last_buf_bytes[which]);
  CU_OK(cudaStreamSynchronize(c->last_stream));
  CU_OK(cudaMemcpy(host, c->last_buf[which], bytes, cudaMemcpyDeviceToHost));
  return FMX_OK;
}

int fmx_profile_enable(fmx_ctx *c, int on) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "profile_enable: NULL ctx");
  std::lock_guard<std::mutex> lk(c->mu);
  CU_OK(cudaDeviceSynchronize());
  for (auto &pe : c->prof) { c->ev_pool.push_back(pe.e0); c->ev_pool.push_back(pe.e1); }
  c->prof.clear();
  c->prof_on = on != 0;
  return FMX_OK;
}

int fmx_profile_select(fmx_ctx *c, uint32_t family_mask) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "profile_select: NULL ctx");
  std::lock_guard<std::mutex> lk(c->mu);
  c->prof_mask = family_mask;
  return FMX_OK;
}

int fmx_profile_read(fmx_ctx *c, int32_t *launches, double *total_ms) {
  if (!c || !launches || !total_ms) return fmx_fail(FMX_E_INVALID_ARG, "profile_read: NULL argument");
  std::lock_guard<std::mutex> lk(c->mu);
  CU_OK(cudaDeviceSynchronize());
  for (int f = 0; f < FMX_N_FAMILIES; ++f) { launches[f] = 0; total_ms[f] = 0.0; }
  for (auto &pe : c->prof) {
    float ms = 0.0f;
    CU_OK(cudaEventElapsedTime(&ms, pe.e0, pe.e1));
    launches[pe.family]++;
    total_ms[pe.family] += ms;
  }
  return FMX_OK;
}

const char *fmx_profile_family_name(int f) { return (f >= 0 && f < FMX_N_FAMILIES) ? kFamilyNames[f] : ""; }
int fmx_last_launch_count(fmx_ctx *c) { return c ? c->last_launches : 0; }
long long fmx_graph_replays(fmx_ctx *c) { return c ? (long long)c->graph_replays : 0; }

int fmx_debug_gemm(fmx_ctx *c, const void *A, const void *W, float *C, int32_t M, int32_t N, int32_t K, void *cuda_stream) {
  if (!c || !A || !W || !C) return fmx_fail(FMX_E_INVALID_ARG, "debug_gemm: NULL argument");
  if (M < 1 || N < 128 || N % 128 || K < 8 || K % 8) return fmx_fail(FMX_E_SHAPE, "debug_gemm: need N %% 128 == 0, K %% 8 == 0");
  std::lock_guard<std::mutex> lk(c->mu);
  CU_OK(cudaSetDevice(c->device));
  PairGemmParams p{};
  int e;
  p.M = M; p.K = K; p.n_chunks = N / 128; p.n_ptiles = (M + kPairRows - 1) / kPairRows; p.mode = GM_OUT_F32;
  if ((e = encode_2d(c, &p.amap, A, M, K, K, 128))) return e;
  if ((e = encode_2d(c, &p.wmap[0], W, N, K, K, pair_wide(p) ? 128 : 64))) return e;
  if ((e = encode_2d(c, &p.wmap_h[0], W, N, K, K, 64))) return e;
  if ((e = encode_2d(c, &p.omap, C, M, N, N, 128, true))) return e;
  for (int i = 0; i < 3; ++i) { p.lora_tgt[i] = -1; p.src_end[i] = 1 << 30; }
  launch_pair_gemm(c, Strm{(cudaStream_t)cuda_stream, 0}, p);
  CU_OK(cudaGetLastError());
  return FMX_OK;
}

int fmx_debug_attention(fmx_ctx *c, const void *qkv, void *out, const int32_t *cu_tok, int32_t n_req, int32_t n_q_heads,
                        int32_t n_kv_heads, int32_t head_dim, int32_t causal, int32_t impl, void *cuda_stream) {
  if (!c || !qkv || !out || !cu_tok) return fmx_fail(FMX_E_INVALID_ARG, "debug_attention: NULL argument");
  if (n_req < 1 || n_q_heads < 1 || n_kv_heads < 1 || n_q_heads % n_kv_heads || !(head_dim == 32 || head_dim == 64 || head_dim == 128))
    return fmx_fail(FMX_E_SHAPE, "debug_attention: bad head configuration");
  std::lock_guard<std::mutex> lk(c->mu);
  CU_OK(cudaSetDevice(c->device));
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int max_len = 0;
  for (int i = 0; i < n_req; ++i) {
    if (cu_tok[i + 1] <= cu_tok[i]) return fmx_fail(FMX_E_BAD_LENGTH, "debug_attention: request %d has no tokens", i);
    max_len = std::max(max_len, cu_tok[i + 1] - cu_tok[i]);
  }
  if (n_req > FMX_MAX_REQUESTS) return fmx_fail(FMX_E_CAPACITY, "debug_attention: %d requests > %d", n_req, FMX_MAX_REQUESTS);
  CU_OK(cudaMemcpyAsync(c->d_dbg_cu, cu_tok, sizeof(int) * (n_req + 1), cudaMemcpyHostToDevice, s));
  const int N = cu_tok[n_req], d_q = n_q_heads * head_dim, d_qkv = (n_q_heads + 2 * n_kv_heads) * head_dim;
  const float scale_log2 = 1.4426950408889634f / sqrtf((float)head_dim);
  if (impl == FMX_ATTN_AUTO && attn_pair64_ok(c->o, head_dim, n_q_heads, max_len)) {
    AttnPairArgs pa2{};
    if (int e = encode_2d(c, &pa2.qkv_map, qkv, N, d_qkv, d_qkv, 64)) return e;
    pa2.out = (bf16 *)out; pa2.cu_tok = c->d_dbg_cu; pa2.ld_out = d_q; pa2.n_req = n_req; pa2.n_q_heads = n_q_heads; pa2.n_kv_heads = n_kv_heads;
    pa2.causal = causal; pa2.scale_log2 = scale_log2;
    launch_attention_pair64(Strm{s, 0}, c->sm_count, pa2);
  } else if (attn_use_tc(impl, head_dim, max_len)) {
    AttnTcArgs ta{};
    if (int e = encode_2d(c, &ta.qkv_map, qkv, N, d_qkv, d_qkv, 64)) return e;
    ta.out = (bf16 *)out; ta.cu_tok = c->d_dbg_cu; ta.ld_out = d_q; ta.n_q_heads = n_q_heads; ta.n_kv_heads = n_kv_heads;
    ta.causal = causal; ta.scale_log2 = scale_log2;
    launch_attention_tc(Strm{s, 0}, head_dim, max_len, n_q_heads, n_req, ta);
  } else {
    AttnArgs aa{};
    aa.qkv = (const bf16 *)qkv; aa.out = (bf16 *)out; aa.cu_tok = c->d_dbg_cu; aa.ld_qkv = d_qkv; aa.ld_out = d_q;
    aa.n_q_heads = n_q_heads; aa.n_kv_heads = n_kv_heads; aa.causal = causal; aa.scale_log2 = scale_log2;
    if (max_len <= 64 && c->o.attn_short) launch_attention_short(Strm{s, 0}, c->sm_count, head_dim, n_req, aa);
    else launch_attention(Strm{s, 0}, head_dim, dim3((max_len + kAttnBQ - 1) / kAttnBQ, n_q_heads, n_req), aa);
  }
  CU_OK(cudaGetLastError());
  CU_OK(cudaStreamSynchronize(s));      // cu_tok is a host array of the caller
  return FMX_OK;
}

int fmx_set_option(fmx_ctx *c, int32_t option, int32_t value) {
  if (!c) return fmx_fail(FMX_E_INVALID_ARG, "set_option: NULL ctx");
  std::lock_guard<std::mutex> lk(c->mu);
  ++c->config_gen;                      // invalidates the cached forward graph
  switch (option) {
    case FMX_OPT_ATTENTION_IMPL:
      if (value < FMX_ATTN_AUTO || value > FMX_ATTN_TCGEN05) return fmx_fail(FMX_E_INVALID_ARG, "set_option: attention impl %d", value);
      c->o.attn_impl = value;
      return FMX_OK;
    case FMX_OPT_SHRINK_STAGES:
      if (value != 4 && value != 5) return fmx_fail(FMX_E_INVALID_ARG, "set_option: shrink stages %d", value);   // 5 = as deep as the stage size allows
      c->o.shrink_stages = value;
      return FMX_OK;
    case FMX_OPT_ATTN_SHORT:
      if (value < 0 || value > 2) return fmx_fail(FMX_E_INVALID_ARG, "set_option: attn_short %d", value);
      c->o.attn_short = value;
      return FMX_OK;
    case FMX_OPT_DEEP_PIPE:
      c->o.deep_pipe = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_EXPAND_WIDE:
      c->o.expand_wide = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_REVERSE:
      c->o.reverse = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_GRAPH:
      c->o.graph = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_SHRINK_FUSED:
      if (value < 0 || value > 2) return fmx_fail(FMX_E_INVALID_ARG, "set_option: shrink_fused %d", value);
      c->o.shrink_fused = value;
      return FMX_OK;
    case FMX_OPT_HEAD_TILED:
      if (value < 0 || value > 2) return fmx_fail(FMX_E_INVALID_ARG, "set_option: head_tiled %d", value);
      c->o.head_tiled = value;
      return FMX_OK;
    case FMX_OPT_ROPE_FUSED:
      c->o.rope_fused = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_HALF_TILES:
      c->o.half_tiles = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_EMBED_SMALL:
      c->o.embed_small = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_DECODE_ROWGEMM:
      c->o.decode_rowgemm = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_DECODE_FORK:
      c->o.decode_fork = value ? 1 : 0;
      return FMX_OK;
    case FMX_OPT_PDL:
      if (value < 0 || value > 2) return fmx_fail(FMX_E_INVALID_ARG, "set_option: pdl %d", value);
      c->o.pdl = value;
      return FMX_OK;
  }
  return fmx_fail(FMX_E_INVALID_ARG, "set_option: unknown option %d", option);
}

}  // extern "C"
