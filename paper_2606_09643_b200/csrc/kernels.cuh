// Memory-bound and integer kernels of the mixed-task forward: task counting sort + segment
// tables (S1), row tables, embed/pack (S2), LayerNorm/RMSNorm (S3a), RoPE, final norm + pool
// (S4), per-task heads + output un-permute (S5/S6).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

namespace fmx {

// ============================================================================= S1
// Device pointers of the segment tables (all int32 unless noted), carved from the workspace.
struct SegTables {
  int *task_ids, *lengths;         // [B] copies of the caller's host arrays (original order)
  int *perm, *inv_perm;            // [B]
  int *task_req_off, *task_tok_off;  // [T+1]
  int *cu_tok;                     // [B+1]
  int *task_sorted;                // [B] task id at sorted position p
  long long *in_off;               // [B+1] element offset of request i in the packed input (original order)
  long long *out_off;              // [B+1] fp32 offset of request i in the output (original order)
  int *tile_blk_off;               // [n_tiles+1]
  int *blk_tile, *blk_task, *blk_lo, *blk_hi;   // [n_blk_cap]
  int *n_blk;                      // scalar
  int *row_req, *row_pos;          // [N] sorted request index / position within request, per token row
};

struct SortArgs {
  SegTables t;
  int B, T;                        // requests, task slots
  int n_tiles;                     // ceil(N / tile_rows)
  int tile_rows;                   // rows of a GEMM row tile (256: one CTA-pair tile)
  long long in_per_tok, in_per_req;  // packed-input elements per token / per request
  const int *task_head_out;        // [T]
  const int *task_head_kind;       // [T] (a dense head writes one output row per token)
  const int *task_enc_ch;          // [T] input channels of the task's encoder (<= 1: none): in_per_req is per channel
};

constexpr int kSortThreads = 1024;

// Block-wide exclusive scan of n values (global or shared), in place; returns the total.  Every thread of the block
// (kSortThreads of them) must call it.  Each thread owns a run of consecutive elements; the run sums are scanned with warp
// shuffles (one pass inside each warp, one over the 32 warp totals): two block barriers per scan, no serial loop.
// scratch: 33 values of shared memory.
template <typename V>
__device__ inline V block_exclusive_scan(V *a, int n, V *scratch) {
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, wid = tid >> 5;
  const int per = (n + nt - 1) / nt;
  const int lo = min(tid * per, n), hi = min(lo + per, n);
  V s = 0;
  for (int i = lo; i < hi; ++i) s += a[i];
  V incl = s;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const V v = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += v; }
  if (lane == 31) scratch[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const V w = lane < (nt >> 5) ? scratch[lane] : V(0);
    V wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const V v = __shfl_up_sync(0xffffffffu, wi, d); if (lane >= d) wi += v; }
    scratch[lane] = wi - w;                       // exclusive offset of warp `lane`
    if (lane == 31) scratch[32] = wi;             // grand total
  }
  __syncthreads();
  V run = scratch[wid] + incl - s;
  for (int i = lo; i < hi; ++i) { const V v = a[i]; a[i] = run; run += v; }
  const V total = scratch[32];
  __syncthreads();
  return total;
}
__device__ inline long long block_exclusive_scan_ll(long long *a, int n, long long *scratch) { return block_exclusive_scan<long long>(a, n, scratch); }
__device__ inline int block_exclusive_scan_i(int *a, int n, int *scratch) { return block_exclusive_scan<int>(a, n, scratch); }

// Exclusive scan of f(0) .. f(n - 1); emit(i, offset) receives every element's exclusive offset (f is evaluated twice per
// element, emit once, by the thread that owns the element's run); returns the total.  Every thread of the block must call it.
template <typename V, typename F, typename E>
__device__ inline V block_exclusive_scan_emit(int n, F f, E emit, V *scratch) {
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, wid = tid >> 5;
  const int per = (n + nt - 1) / nt;
  const int lo = min(tid * per, n), hi = min(lo + per, n);
  V s = 0;
  for (int i = lo; i < hi; ++i) s += f(i);
  V incl = s;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const V v = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += v; }
  if (lane == 31) scratch[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const V w = lane < (nt >> 5) ? scratch[lane] : V(0);
    V wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const V v = __shfl_up_sync(0xffffffffu, wi, d); if (lane >= d) wi += v; }
    scratch[lane] = wi - w;
    if (lane == 31) scratch[32] = wi;
  }
  __syncthreads();
  V run = scratch[wid] + incl - s;
  for (int i = lo; i < hi; ++i) { emit(i, run); run += f(i); }
  const V total = scratch[32];
  __syncthreads();
  return total;
}
// Exclusive scan over 4 consecutive values per thread (thread t owns elements 4 t .. 4 t + 3), in registers; returns the total.
template <typename V>
__device__ inline V block_exclusive_scan_reg4(V (&v)[4], V *scratch) {
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, wid = tid >> 5;
  const V s = (v[0] + v[1]) + (v[2] + v[3]);
  V incl = s;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const V x = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += x; }
  if (lane == 31) scratch[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const V w = lane < (nt >> 5) ? scratch[lane] : V(0);
    V wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const V x = __shfl_up_sync(0xffffffffu, wi, d); if (lane >= d) wi += x; }
    scratch[lane] = wi - w;
    if (lane == 31) scratch[32] = wi;
  }
  __syncthreads();
  V run = scratch[wid] + incl - s;
#pragma unroll
  for (int k = 0; k < 4; ++k) { const V x = v[k]; v[k] = run; run += x; }
  const V total = scratch[32];
  __syncthreads();
  return total;
}

// One CTA.  Stable counting sort of request indices by task id, then the prefix tables and the
// (row-tile, task) block table the segmented GEMMs walk.  Integer only; deterministic.
// Global memory is read twice, each time with every load of the block in flight at once: the ids and lengths of the thread's four
// consecutive requests, then the task tables at those ids.  Ranking, the scans of the counts and of the sorted lengths run in
// shared memory, the input / output offsets are scanned in registers, the block table is filled inside its own scan; everything
// else is a store.  (B <= 4096 = 4 x kSortThreads, T <= 1024.)
__global__ void __launch_bounds__(kSortThreads, 1) task_sort_kernel(const SortArgs a) {
  __shared__ int s_cnt[1024 + 1];          // per-task count, then task_req_off
  __shared__ int s_tok[1024 + 1];          // task_tok_off
  __shared__ int s_scratch[33];
  __shared__ long long s_scratch_ll[33];
  __shared__ unsigned short s_task[4096];  // task id of request i (T <= 1024)
  __shared__ unsigned short s_rank[4096];  // rank of request i within its task
  __shared__ int s_slen[4096 + 1];         // lengths in sorted order, then cu_tok
  const int tid = threadIdx.x, B = a.B, T = a.T;
  const SegTables &t = a.t;
  griddep_launch();
  griddep_wait();

  const int i0 = 4 * tid;                  // this thread's requests: i0 .. i0 + 3
  int id_r[4], len_r[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const bool ok = i0 + k < B;
    id_r[k] = ok ? t.task_ids[i0 + k] : 0;
    len_r[k] = ok ? t.lengths[i0 + k] : 0;
  }
  long long vin[4], vout[4];               // packed-input elements / output values of the request (0 past the end)
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const bool ok = i0 + k < B;
    const int ch = (ok && a.task_enc_ch) ? max(a.task_enc_ch[id_r[k]], 1) : 1;
    const int ho = ok ? a.task_head_out[id_r[k]] : 0, hk = ok ? a.task_head_kind[id_r[k]] : 0;
    vin[k] = ok ? (long long)len_r[k] * a.in_per_tok + a.in_per_req * ch : 0;
    vout[k] = (long long)ho * (hk == 4 ? len_r[k] : 1);
    if (ok) s_task[i0 + k] = (unsigned short)id_r[k];
  }
  for (int i = tid; i <= T; i += blockDim.x) s_cnt[i] = 0;
  __syncthreads();
  // (1) stable rank within task: warp 0 walks the requests 32 at a time, in order.
  if (tid < 32) {
    for (int base = 0; base < B; base += 32) {
      const int i = base + tid;
      const bool ok = i < B;
      const int key = ok ? (int)s_task[i] : -1 - tid;          // inactive lanes get unique keys
      const unsigned m = __match_any_sync(0xffffffffu, key);
      const int leader = __ffs(m) - 1;
      const int rank_in_chunk = __popc(m & ((1u << tid) - 1u));
      int start = 0;
      if (ok && tid == leader) { start = s_cnt[key]; s_cnt[key] = start + __popc(m); }
      start = __shfl_sync(0xffffffffu, start, leader);
      if (ok) s_rank[i] = (unsigned short)(start + rank_in_chunk);
      __syncwarp();
    }
  }
  // (5) input / output offsets in ORIGINAL request order (registers; warp 0 joins after the ranking)
  {
    const long long tin = block_exclusive_scan_reg4<long long>(vin, s_scratch_ll);
    const long long tout = block_exclusive_scan_reg4<long long>(vout, s_scratch_ll);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (i0 + k < B) { t.in_off[i0 + k] = vin[k]; t.out_off[i0 + k] = vout[k]; }
    if (tid == 0) { t.in_off[B] = tin; t.out_off[B] = tout; }
  }
  // (2) task_req_off = exclusive scan of the counts
  if (tid == 0) s_cnt[T] = 0;
  __syncthreads();
  block_exclusive_scan_i(s_cnt, T + 1, s_scratch);
  for (int i = tid; i <= T; i += blockDim.x) t.task_req_off[i] = s_cnt[i];
  // (3) perm / inv_perm / sorted lengths
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int i = i0 + k;
    if (i >= B) continue;
    const int pos = s_cnt[id_r[k]] + s_rank[i];
    t.perm[pos] = i;
    t.inv_perm[i] = pos;
    t.task_sorted[pos] = id_r[k];
    s_slen[pos] = len_r[k];
  }
  if (tid == 0) s_slen[B] = 0;
  __syncthreads();
  // (4) cu_tok = exclusive scan of the sorted lengths; task_tok_off
  block_exclusive_scan_i(s_slen, B + 1, s_scratch);
  for (int i = tid; i <= B; i += blockDim.x) t.cu_tok[i] = s_slen[i];
  for (int i = tid; i <= T; i += blockDim.x) { const int v = s_slen[s_cnt[i]]; s_tok[i] = v; t.task_tok_off[i] = v; }
  __syncthreads();
  // (6) block table: for each row tile, the non-empty task segments that intersect it; filled inside the scan of their counts.
  const int n_tok = s_tok[T];
  auto first_task_after = [&](int row) {     // smallest task with tok_off[task+1] > row
    int lo = 0, hi = T;                      // invariant: answer in [lo, hi)
    while (lo < hi) { int mid = (lo + hi) >> 1; if (s_tok[mid + 1] > row) hi = mid; else lo = mid + 1; }
    return lo;
  };
  auto tile_blocks = [&](int m) {
    if (m >= a.n_tiles) return 0;
    const int r0 = m * a.tile_rows, r1 = min(r0 + a.tile_rows, n_tok);
    int cnt = 0;
    for (int k = first_task_after(r0); k < T && s_tok[k] < r1; ++k) cnt += (s_tok[k + 1] > s_tok[k]);
    return cnt;
  };
  const int n_blk = block_exclusive_scan_emit<int>(a.n_tiles + 1, tile_blocks, [&](int m, int b) {
    t.tile_blk_off[m] = b;
    if (m >= a.n_tiles) return;
    const int r0 = m * a.tile_rows, r1 = min(r0 + a.tile_rows, n_tok);
    for (int k = first_task_after(r0); k < T && s_tok[k] < r1; ++k) {
      if (s_tok[k + 1] <= s_tok[k]) continue;
      t.blk_tile[b] = m;
      t.blk_task[b] = k;
      t.blk_lo[b] = max(s_tok[k], r0) - r0;
      t.blk_hi[b] = min(s_tok[k + 1], r1) - r0;
      ++b;
    }
  }, s_scratch);
  if (tid == 0) *t.n_blk = n_blk;
}

// row -> (sorted request index, position within the request)
__global__ void row_tables_kernel(const int *__restrict__ cu_tok, int B, int N, int *__restrict__ row_req,
                                  int *__restrict__ row_pos) {
  griddep_launch();
  griddep_wait();
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= N) return;
  int lo = 0, hi = B;                          // largest p with cu_tok[p] <= r
  while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (cu_tok[mid] <= r) lo = mid; else hi = mid; }
  row_req[r] = lo;
  row_pos[r] = r - cu_tok[lo];
}

// ============================================================================= S2
struct EmbedArgs {
  const void *inputs;              // packed, original request order
  const int *perm, *row_req, *row_pos;
  const long long *in_off;
  int N, d;
  float *X;                        // fp32 residual [N, d], task-sorted rows
  const __nv_bfloat16 *table;      // TOKEN_IDS
  const __nv_bfloat16 *pos;        // optional positional table [max_seq, d] (EMBEDDED/TOKEN_IDS)
  int vocab;                       // TOKEN_IDS: rows of the table
  unsigned *err;                   // device error word (bit 0: a token id outside [0, vocab))
};

// EMBEDDED: X[r] = x_i[pos] (+ Pos[pos]);   one warp per row, 8 bf16 per lane per step
__global__ void embed_rows_kernel(const EmbedArgs a, int token_ids) {
  griddep_launch();
  griddep_wait();
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= a.N) return;
  const int r = warp, pos = a.row_pos[r], i = a.perm[a.row_req[r]];
  const __nv_bfloat16 *src;
  if (token_ids) {
    // The ids are device data the host cannot validate: an id outside the table becomes a zero row (never an out-of-bounds
    // read) and raises the context's device error word, which the next forward call reports.
    const int id = reinterpret_cast<const int *>(a.inputs)[a.in_off[i] + pos];
    if (id < 0 || id >= a.vocab) {
      if (lane == 0) *a.err = 1u;
      float *dst0 = a.X + (size_t)r * a.d;
      for (int c = lane * 4; c < a.d; c += 128) *reinterpret_cast<float4 *>(dst0 + c) = make_float4(0.f, 0.f, 0.f, 0.f);
      return;
    }
    src = a.table + (size_t)id * a.d;
  } else {
    src = reinterpret_cast<const __nv_bfloat16 *>(a.inputs) + a.in_off[i] + (size_t)pos * a.d;
  }
  float *dst = a.X + (size_t)r * a.d;
  for (int c = lane * 8; c < a.d; c += 256) {
    const uint4 v = *reinterpret_cast<const uint4 *>(src + c);
    float f[8] = {bf16_lo(v.x), bf16_hi(v.x), bf16_lo(v.y), bf16_hi(v.y), bf16_lo(v.z), bf16_hi(v.z), bf16_lo(v.w), bf16_hi(v.w)};
    if (a.pos) {
      const uint4 q = *reinterpret_cast<const uint4 *>(a.pos + (size_t)pos * a.d + c);
      f[0] += bf16_lo(q.x); f[1] += bf16_hi(q.x); f[2] += bf16_lo(q.y); f[3] += bf16_hi(q.y);
      f[4] += bf16_lo(q.z); f[5] += bf16_hi(q.z); f[6] += bf16_lo(q.w); f[7] += bf16_hi(q.w);
    }
    *reinterpret_cast<float4 *>(dst + c) = make_float4(f[0], f[1], f[2], f[3]);
    *reinterpret_cast<float4 *>(dst + c + 4) = make_float4(f[4], f[5], f[6], f[7]);
  }
}

struct PackArgs {
  const __nv_bfloat16 *inputs;
  const int *perm, *row_req, *row_pos;
  const long long *in_off;
  int N, patch_dim, Kp, has_cls;
  int img_c, img_hw, patch_hw;     // img_c = 0: input already [n_patches, patch_dim]
  // per-task input encoder (series input only): channels, weights [C], bias [1] by task; task of each ORIGINAL request
  const int *task_ids, *task_enc_ch;
  const __nv_bfloat16 *const *task_enc_W, *const *task_enc_b;
  int series_len;                  // n_patches * patch_dim (elements of one channel)
  __nv_bfloat16 *A;                // [N, Kp] task-sorted patch rows (CLS rows and the K pad are zero)
  int tpr;                         // threads per row (a power of two <= blockDim.x): a block packs blockDim.x / tpr rows
};

// PATCH_LINEAR: gather (and patchify) into the A operand of the embed GEMM.  tpr threads per row.
__global__ void pack_patches_kernel(const PackArgs a) {
  griddep_launch();
  griddep_wait();
  const int r = blockIdx.x * (blockDim.x / a.tpr) + threadIdx.x / a.tpr;
  if (r >= a.N) return;
  const int pos = a.row_pos[r], i = a.perm[a.row_req[r]];
  const __nv_bfloat16 *src = a.inputs + a.in_off[i];
  __nv_bfloat16 *dst = a.A + (size_t)r * a.Kp;
  const int pi = pos - a.has_cls;
  const int P = a.patch_hw, g = a.img_c ? a.img_hw / P : 1;
  const int gy = pi / g, gx = pi - gy * g;
  for (int e = threadIdx.x % a.tpr; e < a.Kp; e += a.tpr) {
    __nv_bfloat16 v = __float2bfloat16(0.0f);
    if (pi >= 0 && e < a.patch_dim) {
      if (a.img_c) {
        const int c = e / (P * P), rem = e - c * P * P, py = rem / P, px = rem - py * P;
        v = src[((size_t)c * a.img_hw + gy * P + py) * a.img_hw + gx * P + px];
      } else {
        const int t = a.task_ids[i];
        const int ch = a.task_enc_ch[t];
        if (ch <= 1) {
          v = src[(size_t)pi * a.patch_dim + e];
        } else {                                            // LinearChannelCombiner: sum_c w[c] x[c, k] + b, fp32, one rounding
          const __nv_bfloat16 *wc = a.task_enc_W[t], *bc = a.task_enc_b[t];
          float acc = bc ? __bfloat162float(bc[0]) : 0.0f;
          for (int cc = 0; cc < ch; ++cc)
            acc = fmaf(__bfloat162float(wc[cc]), __bfloat162float(src[(size_t)cc * a.series_len + (size_t)pi * a.patch_dim + e]), acc);
          v = __float2bfloat16(acc);
        }
      }
    }
    dst[e] = v;
  }
}

// posb[p, :] = (p == 0 && has_cls ? cls : embed_b) + Pos[p]     (fp32; built once at registration)
__global__ void build_posb_kernel(float *posb, const __nv_bfloat16 *b, const __nv_bfloat16 *cls,
                                  const __nv_bfloat16 *pos, int n_pos, int d, int has_cls) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_pos * d) return;
  const int p = idx / d, c = idx - p * d;
  float v = 0.0f;
  if (has_cls && p == 0) v = __bfloat162float(cls[c]);
  else if (b) v = __bfloat162float(b[c]);
  if (pos) v += __bfloat162float(pos[idx]);
  posb[idx] = v;
}

// Patch embedding with a tiny patch (K_p = 8: the time-series backbones of cfg2 / cfg5): X[row, :] = A[row, :K_p] W_e^T + posb[pos(row)]
// is a stream of 4 KB fp32 rows out for 16 bytes in - through the tensor-core GEMM it costs 512 epilogues of 256 KB for one
// mostly-zero k-block each (measured 0.10 ms per step on cfg5); here a thread keeps the weights of its 4 columns in registers and
// walks kEmbRows rows.  fp32 accumulation in k order.  grid (ceil(N / kEmbRows), d / 1024 rounded up), 256 threads.
constexpr int kEmbRows = 16;
__global__ void __launch_bounds__(256) embed_small_patch_kernel(const __nv_bfloat16 *__restrict__ A, const __nv_bfloat16 *__restrict__ Wpad,
                                                                const float *__restrict__ posb, const int *__restrict__ row_pos, int N, int d,
                                                                float *__restrict__ X) {
  griddep_launch();
  griddep_wait();
  const int c = (blockIdx.y * 256 + threadIdx.x) * 4;
  if (c >= d) return;
  float w[4][8];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const uint4 v = *reinterpret_cast<const uint4 *>(Wpad + (size_t)(c + j) * 8);
    w[j][0] = bf16_lo(v.x); w[j][1] = bf16_hi(v.x); w[j][2] = bf16_lo(v.y); w[j][3] = bf16_hi(v.y);
    w[j][4] = bf16_lo(v.z); w[j][5] = bf16_hi(v.z); w[j][6] = bf16_lo(v.w); w[j][7] = bf16_hi(v.w);
  }
  const int r0 = blockIdx.x * kEmbRows, r1 = min(N, r0 + kEmbRows);
#pragma unroll 4
  for (int r = r0; r < r1; ++r) {
    const uint4 av = *reinterpret_cast<const uint4 *>(A + (size_t)r * 8);
    const float x[8] = {bf16_lo(av.x), bf16_hi(av.x), bf16_lo(av.y), bf16_hi(av.y), bf16_lo(av.z), bf16_hi(av.z), bf16_lo(av.w), bf16_hi(av.w)};
    const float4 pb = *reinterpret_cast<const float4 *>(posb + (size_t)row_pos[r] * d + c);
    float o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float acc = 0.0f;
#pragma unroll
      for (int k = 0; k < 8; ++k) acc = fmaf(x[k], w[j][k], acc);
      o[j] = acc;
    }
    *reinterpret_cast<float4 *>(X + (size_t)r * d + c) = make_float4(o[0] + pb.x, o[1] + pb.y, o[2] + pb.z, o[3] + pb.w);
  }
}

// W_e [d, patch_dim] -> [d, Kp] zero padded (row stride must be a multiple of 16 B for TMA)
__global__ void pad_rows_kernel(const __nv_bfloat16 *src, __nv_bfloat16 *dst, int rows, int k, int kp) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= rows * kp) return;
  const int r = idx / kp, c = idx - r * kp;
  dst[idx] = c < k ? src[(size_t)r * k + c] : __float2bfloat16(0.0f);
}

// ============================================================================= S3a
// One warp per row: fp32 X [N, d] -> bf16 Y [N, d].  LayerNorm (g, b) or RMSNorm (g); fp32 statistics.
template <int kVec>   // float4s per lane: d = 128 * kVec
__global__ void __launch_bounds__(256) norm_kernel(const float *__restrict__ X, __nv_bfloat16 *__restrict__ Y,
                                                   const __nv_bfloat16 *__restrict__ g,
                                                   const __nv_bfloat16 *__restrict__ b, int N, float eps, int rms, int reverse) {
  griddep_launch();
  griddep_wait();
  int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (row >= N) return;
  if (reverse) row = N - 1 - row;          // early CTAs take the rows the producing GEMM wrote last (still in L2)
  constexpr int d = 128 * kVec;
  const float4 *x = reinterpret_cast<const float4 *>(X + (size_t)row * d);
  float4 v[kVec];
  float s = 0.0f;
#pragma unroll
  for (int j = 0; j < kVec; ++j) { v[j] = x[j * 32 + lane]; s += v[j].x + v[j].y + v[j].z + v[j].w; }
  float mean = 0.0f;
  if (!rms) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    mean = s * (1.0f / d);
  }
  float q = 0.0f;
#pragma unroll
  for (int j = 0; j < kVec; ++j) {
    const float a0 = v[j].x - mean, a1 = v[j].y - mean, a2 = v[j].z - mean, a3 = v[j].w - mean;
    q += a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
  const float inv = rsqrtf(q * (1.0f / d) + eps);
  uint2 *y = reinterpret_cast<uint2 *>(Y + (size_t)row * d);
#pragma unroll
  for (int j = 0; j < kVec; ++j) {
    const int c4 = j * 32 + lane;
    const uint2 gg = reinterpret_cast<const uint2 *>(g)[c4];
    float o0 = (v[j].x - mean) * inv * bf16_lo(gg.x), o1 = (v[j].y - mean) * inv * bf16_hi(gg.x);
    float o2 = (v[j].z - mean) * inv * bf16_lo(gg.y), o3 = (v[j].w - mean) * inv * bf16_hi(gg.y);
    if (b) {
      const uint2 bb = reinterpret_cast<const uint2 *>(b)[c4];
      o0 += bf16_lo(bb.x); o1 += bf16_hi(bb.x); o2 += bf16_lo(bb.y); o3 += bf16_hi(bb.y);
    }
    y[c4] = make_uint2(pack_bf16(o0, o1), pack_bf16(o2, o3));
  }
}

// ============================================================================= RoPE (in place on the fused qkv buffer)
// rotate-half pairing (j, j + dh/2); position = row_pos[row]; cs = [max_seq, dh/2] float2 (cos, sin).
// One thread rotates 8 pairs: two 16-byte loads/stores of the row (first and second half of the head) and
// 64 bytes of the table, so a warp touches whole 128-byte lines (dh/2 must be a multiple of 8).
__global__ void __launch_bounds__(256) rope_kernel(__nv_bfloat16 *qkv, int ld, const int *__restrict__ row_pos,
                                                   const float2 *__restrict__ cs, int N, int n_heads_qk, int dh) {
  griddep_launch();
  griddep_wait();
  const int half = dh >> 1, vec_per_head = half >> 3;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;     // (row, head, vector of 8 pairs)
  const long long total = (long long)N * n_heads_qk * vec_per_head;
  if (idx >= total) return;
  const int jv = (int)(idx % vec_per_head);
  const int h = (int)((idx / vec_per_head) % n_heads_qk);
  const int row = (int)(idx / ((long long)vec_per_head * n_heads_qk));
  const float4 *c4 = reinterpret_cast<const float4 *>(cs + (size_t)row_pos[row] * half + jv * 8);
  __nv_bfloat16 *p = qkv + (size_t)row * ld + h * dh + jv * 8;
  const uint4 a = *reinterpret_cast<const uint4 *>(p), b = *reinterpret_cast<const uint4 *>(p + half);
  const uint32_t av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
  uint32_t ao[4], bo[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const float4 c = c4[q];                       // (cos, sin) of pairs 2q, 2q+1
    const float x1l = bf16_lo(av[q]), x1h = bf16_hi(av[q]), x2l = bf16_lo(bv[q]), x2h = bf16_hi(bv[q]);
    ao[q] = pack_bf16(x1l * c.x - x2l * c.y, x1h * c.z - x2h * c.w);
    bo[q] = pack_bf16(x2l * c.x + x1l * c.y, x2h * c.z + x1h * c.w);
  }
  *reinterpret_cast<uint4 *>(p) = make_uint4(ao[0], ao[1], ao[2], ao[3]);
  *reinterpret_cast<uint4 *>(p + half) = make_uint4(bo[0], bo[1], bo[2], bo[3]);
}

// transposed copy [dh/2][max_seq]: for a fixed pair index, consecutive positions are contiguous, so the threads of a warp
// (= consecutive token rows = mostly consecutive positions) read it coalesced in the GEMM epilogue
__global__ void transpose_rope_table_kernel(const float2 *cs, float2 *cs_t, int max_seq, int half) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= max_seq * half) return;
  const int p = idx / half, j = idx - p * half;
  cs_t[(size_t)j * max_seq + p] = cs[idx];
}

__global__ void build_rope_table_kernel(float2 *cs, int max_seq, int dh, double theta) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int half = dh >> 1;
  if (idx >= max_seq * half) return;
  const int p = idx / half, j = idx - p * half;
  const double ang = (double)p * pow(theta, -2.0 * (double)j / (double)dh);
  cs[idx] = make_float2((float)cos(ang), (float)sin(ang));
}

// ============================================================================= S4: final norm + pool
struct PoolArgs {
  const float *X;                  // [N, d]
  const __nv_bfloat16 *g, *b;
  const int *cu_tok, *task_sorted;
  const int *task_head_kind;       // [T]
  float *feat;                     // [B, d] fp32 pooled feature per SORTED request (mean / cls / last)
  __nv_bfloat16 *Fn;               // [N, d] bf16 normed rows (written for FLATTEN / DENSE requests only)
  int d;
  float eps;
  int rms;
};

// One block (128 threads = 4 warps) per sorted request.  Each warp normalises rows; mean-pool is
// accumulated per warp in registers (fixed row->warp assignment and fixed combine order: deterministic).
template <int kVec>
__global__ void __launch_bounds__(128) final_pool_kernel(const PoolArgs a) {
  griddep_launch();
  griddep_wait();
  constexpr int d = 128 * kVec;
  __shared__ float s_part[4][d];
  const int p = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
  const int kind = a.task_head_kind[a.task_sorted[p]];
  float4 accv[kVec];
#pragma unroll
  for (int j = 0; j < kVec; ++j) accv[j] = make_float4(0.f, 0.f, 0.f, 0.f);
  int first = 0, last = n;
  if (kind == 1) { first = 0; last = 1; }            // CLS
  else if (kind == 2) { first = n - 1; last = n; }   // LAST
  for (int i = first + warp; i < last; i += 4) {
    const float4 *x = reinterpret_cast<const float4 *>(a.X + (size_t)(r0 + i) * d);
    float4 v[kVec];
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < kVec; ++j) { v[j] = x[j * 32 + lane]; s += v[j].x + v[j].y + v[j].z + v[j].w; }
    float mean = 0.0f;
    if (!a.rms) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      mean = s * (1.0f / d);
    }
    float q = 0.0f;
#pragma unroll
    for (int j = 0; j < kVec; ++j) {
      const float a0 = v[j].x - mean, a1 = v[j].y - mean, a2 = v[j].z - mean, a3 = v[j].w - mean;
      q += a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    const float inv = rsqrtf(q * (1.0f / d) + a.eps);
#pragma unroll
    for (int j = 0; j < kVec; ++j) {
      const int c4 = j * 32 + lane;
      const uint2 gg = reinterpret_cast<const uint2 *>(a.g)[c4];
      float o0 = (v[j].x - mean) * inv * bf16_lo(gg.x), o1 = (v[j].y - mean) * inv * bf16_hi(gg.x);
      float o2 = (v[j].z - mean) * inv * bf16_lo(gg.y), o3 = (v[j].w - mean) * inv * bf16_hi(gg.y);
      if (a.b) {
        const uint2 bb = reinterpret_cast<const uint2 *>(a.b)[c4];
        o0 += bf16_lo(bb.x); o1 += bf16_hi(bb.x); o2 += bf16_lo(bb.y); o3 += bf16_hi(bb.y);
      }
      if (kind >= 3) {                                    // FLATTEN and DENSE heads read every normed row
        reinterpret_cast<uint2 *>(a.Fn + (size_t)(r0 + i) * d)[c4] = make_uint2(pack_bf16(o0, o1), pack_bf16(o2, o3));
      } else {
        accv[j].x += o0; accv[j].y += o1; accv[j].z += o2; accv[j].w += o3;
      }
    }
  }
  if (kind >= 3) return;
#pragma unroll
  for (int j = 0; j < kVec; ++j) reinterpret_cast<float4 *>(s_part[warp])[j * 32 + lane] = accv[j];
  __syncthreads();
  const float scale = kind == 0 ? 1.0f / (float)n : 1.0f;
  for (int c = threadIdx.x; c < d; c += 128) {
    float s = 0.0f;
#pragma unroll
    for (int w = 0; w < 4; ++w) s += s_part[w][c];
    a.feat[(size_t)p * d + c] = s * scale;
  }
}

// ============================================================================= S5 + S6: per-task heads
struct HeadArgs {
  const float *feat;               // [B, d] (pooled kinds)
  const __nv_bfloat16 *Fn;         // [N, d] (FLATTEN)
  const int *cu_tok, *task_sorted, *perm;
  const long long *out_off;
  const int *task_head_kind, *task_head_out;
  const __nv_bfloat16 *const *task_head_W, *const *task_head_b;
  float *out;
  int d;
  // MLP heads: first-layer width per task (= head_out for linear heads), second-layer weights (NULL = linear head), and the
  // fp32 hidden scratch [B, ld_hid] indexed by SORTED request
  const int *task_head_w1;
  const __nv_bfloat16 *const *task_head_W2, *const *task_head_b2;
  float *hid;
  int ld_hid;
  int skip_flatten;                // 1: FLATTEN heads are computed by head_flatten_kernel
};

// grid (sorted request p, output tile of 8): each warp computes one output o as a dot product over
// d_feat with 16-byte loads; result written straight to the caller's buffer in ORIGINAL order.
__global__ void __launch_bounds__(256) head_kernel(const HeadArgs a) {
  griddep_launch();
  griddep_wait();
  const int p = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = a.task_sorted[p];
  const int o = blockIdx.y * 8 + warp;
  const int n_out = a.task_head_w1[t];
  if (o >= n_out) return;
  const int kind = a.task_head_kind[t];
  if ((kind == 3 && a.skip_flatten) || kind == 4) return;       // FLATTEN on the tensor-core path; dense heads have their own kernel
  const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
  const long long K = kind == 3 ? (long long)n * a.d : a.d;
  const __nv_bfloat16 *w = a.task_head_W[t] + (size_t)o * K;
  float acc = 0.0f;
  if (kind == 3) {
    const __nv_bfloat16 *f = a.Fn + (size_t)r0 * a.d;
    for (long long c = lane * 8; c < K; c += 256) {
      const uint4 wv = *reinterpret_cast<const uint4 *>(w + c), fv = *reinterpret_cast<const uint4 *>(f + c);
      acc += bf16_lo(wv.x) * bf16_lo(fv.x) + bf16_hi(wv.x) * bf16_hi(fv.x) + bf16_lo(wv.y) * bf16_lo(fv.y) +
             bf16_hi(wv.y) * bf16_hi(fv.y) + bf16_lo(wv.z) * bf16_lo(fv.z) + bf16_hi(wv.z) * bf16_hi(fv.z) +
             bf16_lo(wv.w) * bf16_lo(fv.w) + bf16_hi(wv.w) * bf16_hi(fv.w);
    }
  } else {
    const float *f = a.feat + (size_t)p * a.d;
    for (int c = lane * 8; c < a.d; c += 256) {
      const uint4 wv = *reinterpret_cast<const uint4 *>(w + c);
      const float4 f0 = *reinterpret_cast<const float4 *>(f + c), f1 = *reinterpret_cast<const float4 *>(f + c + 4);
      acc += bf16_lo(wv.x) * f0.x + bf16_hi(wv.x) * f0.y + bf16_lo(wv.y) * f0.z + bf16_hi(wv.y) * f0.w +
             bf16_lo(wv.z) * f1.x + bf16_hi(wv.z) * f1.y + bf16_lo(wv.w) * f1.z + bf16_hi(wv.w) * f1.w;
    }
  }
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
  if (lane == 0) {
    const __nv_bfloat16 *b = a.task_head_b[t];
    const float v = acc + (b ? __bfloat162float(b[o]) : 0.0f);
    if (a.task_head_W2[t]) a.hid[(size_t)p * a.ld_hid + o] = fmaxf(v, 0.0f);      // hidden layer of an MLP head
    else a.out[a.out_off[a.perm[p]] + o] = v;
  }
}

// Dense (per-token) heads (FMX_HEAD_DENSE): y[token, :] = W_t f[token] + b_t for every token row of a dense task's request,
// f = the final-normed row (bf16, written by final_pool_kernel).  One warp per token row: the row sits in registers, the
// task's weight rows stream through (L1 / L2 hits: consecutive rows share the task), one shuffle reduction per output.
// Written at out_off[request] + position * head_out in ORIGINAL request order.
__global__ void __launch_bounds__(256) head_dense_kernel(const HeadArgs a, int N, const int *__restrict__ row_req, const int *__restrict__ row_pos) {
  griddep_launch();
  griddep_wait();
  const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (r >= N) return;
  const int p = row_req[r], t = a.task_sorted[p];
  if (a.task_head_kind[t] != 4) return;
  const int n_out = a.task_head_out[t];
  const __nv_bfloat16 *f = a.Fn + (size_t)r * a.d, *W = a.task_head_W[t], *b = a.task_head_b[t];
  float *dst = a.out + a.out_off[a.perm[p]] + (long long)row_pos[r] * n_out;
  for (int o = 0; o < n_out; ++o) {
    const __nv_bfloat16 *w = W + (size_t)o * a.d;
    float acc = 0.0f;
    for (int c = lane * 8; c < a.d; c += 256) {
      const uint4 wv = *reinterpret_cast<const uint4 *>(w + c), fv = *reinterpret_cast<const uint4 *>(f + c);
      acc += bf16_lo(wv.x) * bf16_lo(fv.x) + bf16_hi(wv.x) * bf16_hi(fv.x) + bf16_lo(wv.y) * bf16_lo(fv.y) +
             bf16_hi(wv.y) * bf16_hi(fv.y) + bf16_lo(wv.z) * bf16_lo(fv.z) + bf16_hi(wv.z) * bf16_hi(fv.z) +
             bf16_lo(wv.w) * bf16_lo(fv.w) + bf16_hi(wv.w) * bf16_hi(fv.w);
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if (lane == 0) dst[o] = acc + (b ? __bfloat162float(b[o]) : 0.0f);
  }
}

// Second layer of MLP heads: y = W2 · hid + b2, one warp per (sorted request, output), written in ORIGINAL request order.
__global__ void __launch_bounds__(256) head_mlp2_kernel(const HeadArgs a) {
  griddep_launch();
  griddep_wait();
  const int p = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = a.task_sorted[p];
  const __nv_bfloat16 *W2 = a.task_head_W2[t];
  const int o = blockIdx.y * 8 + warp;
  if (!W2 || o >= a.task_head_out[t]) return;
  const int K = a.task_head_w1[t];
  const float *h = a.hid + (size_t)p * a.ld_hid;
  const __nv_bfloat16 *w = W2 + (size_t)o * K;
  float acc = 0.0f;
  for (int c = lane; c < K; c += 32) acc = fmaf(h[c], __bfloat162float(w[c]), acc);
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
  if (lane == 0) {
    const __nv_bfloat16 *b = a.task_head_b2[t];
    a.out[a.out_off[a.perm[p]] + o] = acc + (b ? __bfloat162float(b[o]) : 0.0f);
  }
}

// FLATTEN heads (cfg2 forecasting: d_feat = 64 x 1024, 96 outputs, 12.6 MB of weights per task).  head_kernel spends ~30
// instructions per (request, output) per 8 features, almost all of them loads and bf16 unpacking, and is issue-bound.
// Here a CTA owns a 4-request x 4-output tile: every unpacked weight serves 4 requests and every unpacked feature 4
// outputs; its 8 warps split the feature axis and their partial sums are added in warp order (deterministic).
// grid (ceil(B / 4) groups of consecutive SORTED requests, ceil(max_out / 4)); requests of a group that belong to another
// task than its first FLATTEN request are handled in further passes (task boundaries only).
__global__ void __launch_bounds__(256) head_flatten_kernel(const HeadArgs a, int B) {
  __shared__ float s_part[8][16];
  griddep_launch();
  griddep_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int p0 = blockIdx.x * 4;
  const int o0 = blockIdx.y * 4;
  int task[4];
  unsigned todo = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    task[i] = p0 + i < B ? a.task_sorted[p0 + i] : -1;
    if (task[i] >= 0 && a.task_head_kind[task[i]] == 3 && o0 < a.task_head_out[task[i]]) todo |= 1u << i;
  }
  while (todo) {                                           // CTA-uniform
    const int lead = __ffs(todo) - 1;
    const int t = task[lead];
    unsigned grp = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) if (((todo >> i) & 1u) && task[i] == t) grp |= 1u << i;
    todo &= ~grp;
    const int n_out = a.task_head_out[t];
    const int r_lead = a.cu_tok[p0 + lead];
    const long long K = (long long)(a.cu_tok[p0 + lead + 1] - r_lead) * a.d;
    const __nv_bfloat16 *f[4], *w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) f[i] = a.Fn + (size_t)a.cu_tok[p0 + (((grp >> i) & 1u) ? i : lead)] * a.d;
#pragma unroll
    for (int j = 0; j < 4; ++j) w[j] = a.task_head_W[t] + (size_t)min(o0 + j, n_out - 1) * K;
    float acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j] = 0.0f;
    for (long long c = (long long)(warp * 32 + lane) * 8; c < K; c += 8 * 256) {
      float fv[4][8], wv[8];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint4 u = *reinterpret_cast<const uint4 *>(f[i] + c);
        fv[i][0] = bf16_lo(u.x); fv[i][1] = bf16_hi(u.x); fv[i][2] = bf16_lo(u.y); fv[i][3] = bf16_hi(u.y);
        fv[i][4] = bf16_lo(u.z); fv[i][5] = bf16_hi(u.z); fv[i][6] = bf16_lo(u.w); fv[i][7] = bf16_hi(u.w);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint4 u = *reinterpret_cast<const uint4 *>(w[j] + c);
        wv[0] = bf16_lo(u.x); wv[1] = bf16_hi(u.x); wv[2] = bf16_lo(u.y); wv[3] = bf16_hi(u.y);
        wv[4] = bf16_lo(u.z); wv[5] = bf16_hi(u.z); wv[6] = bf16_lo(u.w); wv[7] = bf16_hi(u.w);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int e = 0; e < 8; ++e) acc[i][j] = fmaf(fv[i][e], wv[e], acc[i][j]);
      }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        float v = acc[i][j];
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
        if (lane == 0) s_part[warp][i * 4 + j] = v;
      }
    __syncthreads();
    if (threadIdx.x < 16) {
      const int i = threadIdx.x >> 2, j = threadIdx.x & 3;
      float v = 0.0f;
#pragma unroll
      for (int wq = 0; wq < 8; ++wq) v += s_part[wq][threadIdx.x];
      const __nv_bfloat16 *b = a.task_head_b[t];
      if (((grp >> i) & 1u) && o0 + j < n_out) a.out[a.out_off[a.perm[p0 + i]] + o0 + j] = v + (b ? __bfloat162float(b[o0 + j]) : 0.0f);
    }
    __syncthreads();
  }
}

// FLATTEN heads on the tensor cores (mma.sync m16n8k16, fp32 accumulate).  The CUDA-core kernel above moves 1.5 GB through
// the L2 fabric for cfg2 (every CTA re-reads 4 feature rows and 4 weight rows of 128 KB each) and takes ~0.23 ms; here a
// warp owns a 16-request x 32-output tile over a K slice, which cuts the traffic to ~0.3 GB.
//   grid (ceil(B / 16) groups of consecutive SORTED requests, ceil(max_out / 32), n_kc K-chunks); 8 warps split the chunk.
// The dot product does not care about the order of K, so within every 32 features thread t of a quad loads features
// [8t, 8t+8) of its rows with ONE 16-byte load and feeds them to two MMAs as "k-slots"; A and B use the same assignment.
// Requests of a group that belong to different FLATTEN tasks are handled in passes (task boundaries only).  Partial sums
// of the 8 warps are added in warp order in shared memory; the n_kc chunk partials go to `part` and
// head_flatten_reduce_kernel adds them in chunk order (deterministic), adds the bias and writes in ORIGINAL request order.
__device__ __forceinline__ void mma_bf16_16816_h(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__global__ void __launch_bounds__(256) head_flatten_mma_kernel(const HeadArgs a, int B, int n_kc, float *__restrict__ part) {
  __shared__ float s_part[8][16 * 32];
  griddep_launch();
  griddep_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t4 = lane & 3;
  const int p0 = blockIdx.x * 16, o0 = blockIdx.y * 32, kc = blockIdx.z;
  // tasks of this thread's two rows (g, g + 8) and of all 16 rows (todo mask is CTA-uniform)
  unsigned todo = 0;
  for (int i = 0; i < 16; ++i) {
    const int p = p0 + i;
    if (p < B) {
      const int ti = a.task_sorted[p];
      if (a.task_head_kind[ti] == 3 && o0 < a.task_head_out[ti]) todo |= 1u << i;
    }
  }
  float fin[4][4];
#pragma unroll
  for (int nt = 0; nt < 4; ++nt) fin[nt][0] = fin[nt][1] = fin[nt][2] = fin[nt][3] = 0.0f;
  while (todo) {
    const int lead = __ffs(todo) - 1;
    const int t = a.task_sorted[p0 + lead];
    unsigned grp = 0;
    for (int i = 0; i < 16; ++i)
      if (((todo >> i) & 1u) && a.task_sorted[p0 + i] == t) grp |= 1u << i;
    todo &= ~grp;
    const int n_out = a.task_head_out[t];
    const long long K = (long long)(a.cu_tok[p0 + lead + 1] - a.cu_tok[p0 + lead]) * a.d;
    const long long k_per_warp = K / (n_kc * 8);                 // host guarantees a multiple of 32
    const long long k_lo = (long long)(kc * 8 + warp) * k_per_warp;
    const __nv_bfloat16 *f0 = a.Fn + (size_t)a.cu_tok[p0 + (((grp >> g) & 1u) ? g : lead)] * a.d + k_lo + 8 * t4;
    const __nv_bfloat16 *f1 = a.Fn + (size_t)a.cu_tok[p0 + (((grp >> (g + 8)) & 1u) ? g + 8 : lead)] * a.d + k_lo + 8 * t4;
    const __nv_bfloat16 *w[4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) w[nt] = a.task_head_W[t] + (size_t)min(o0 + nt * 8 + g, n_out - 1) * K + k_lo + 8 * t4;
    float acc[4][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.0f;
#pragma unroll 2
    for (long long k = 0; k < k_per_warp; k += 32) {
      const uint4 A0 = *reinterpret_cast<const uint4 *>(f0 + k), A1 = *reinterpret_cast<const uint4 *>(f1 + k);
      uint4 Wv[4];
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) Wv[nt] = *reinterpret_cast<const uint4 *>(w[nt] + k);
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) {
        mma_bf16_16816_h(acc[nt], A0.x, A1.x, A0.y, A1.y, Wv[nt].x, Wv[nt].y);
        mma_bf16_16816_h(acc[nt], A0.z, A1.z, A0.w, A1.w, Wv[nt].z, Wv[nt].w);
      }
    }
    // keep the rows of this pass's task (accumulator rows g and g + 8)
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      if ((grp >> g) & 1u) { fin[nt][0] = acc[nt][0]; fin[nt][1] = acc[nt][1]; }
      if ((grp >> (g + 8)) & 1u) { fin[nt][2] = acc[nt][2]; fin[nt][3] = acc[nt][3]; }
    }
  }
  // ---- add the 8 warps' partial tiles in warp order, one chunk partial per CTA ----
#pragma unroll
  for (int nt = 0; nt < 4; ++nt) {
    const int col = nt * 8 + 2 * t4;
    s_part[warp][g * 32 + col] = fin[nt][0]; s_part[warp][g * 32 + col + 1] = fin[nt][1];
    s_part[warp][(g + 8) * 32 + col] = fin[nt][2]; s_part[warp][(g + 8) * 32 + col + 1] = fin[nt][3];
  }
  __syncthreads();
  float *dst = part + ((size_t)(blockIdx.x * gridDim.y + blockIdx.y) * n_kc + kc) * 512;
  for (int e = threadIdx.x; e < 512; e += 256) {
    float v = 0.0f;
#pragma unroll
    for (int wq = 0; wq < 8; ++wq) v += s_part[wq][e];
    dst[e] = v;
  }
}

__global__ void __launch_bounds__(512) head_flatten_reduce_kernel(const HeadArgs a, int B, int n_kc, const float *__restrict__ part) {
  griddep_launch();
  griddep_wait();
  const int r = threadIdx.x >> 5, o = threadIdx.x & 31;
  const int p = blockIdx.x * 16 + r, oa = blockIdx.y * 32 + o;
  if (p >= B) return;
  const int t = a.task_sorted[p];
  if (a.task_head_kind[t] != 3 || oa >= a.task_head_out[t]) return;
  const float *src = part + (size_t)(blockIdx.x * gridDim.y + blockIdx.y) * n_kc * 512 + r * 32 + o;
  float v = 0.0f;
  for (int kc = 0; kc < n_kc; ++kc) v += src[(size_t)kc * 512];
  const __nv_bfloat16 *b = a.task_head_b[t];
  a.out[a.out_off[a.perm[p]] + oa] = v + (b ? __bfloat162float(b[oa]) : 0.0f);
}

// ============================================================================= token decode with a KV cache (NEXT-3)
// Cache layout (caller-owned device memory, fmx_kv_cache_bytes): [slot][layer][k | v][max_seq][d_kv] bf16.
struct KvArgs {
  __nv_bfloat16 *cache;
  long long slot_stride, layer_stride, kv_stride;   // elements: per slot, per layer, k -> v
  int d_kv, max_seq;
  const int *row_slot, *row_cpos;                   // [N] cache slot / cache position of every token row
};

// row -> (cache slot, cache position = RoPE position).  slots / pos0 are per ORIGINAL request; pos0 NULL = 0 (prefill).
__global__ void kv_rows_kernel(const int *__restrict__ row_req, const int *__restrict__ row_pos, const int *__restrict__ perm,
                               const int *__restrict__ slots, const int *__restrict__ pos0, int N, int *__restrict__ row_slot,
                               int *__restrict__ row_cpos) {
  griddep_launch();
  griddep_wait();
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= N) return;
  const int i = perm[row_req[r]];
  row_slot[r] = slots[i];
  row_cpos[r] = (pos0 ? pos0[i] : 0) + row_pos[r];
}

// Appends this layer's k and v rows (after RoPE) of every token row to the cache.  One warp per row, 16-byte copies.
__global__ void kv_append_kernel(const __nv_bfloat16 *__restrict__ qkv, int ld_qkv, int col_k, int col_v, int N, int layer, const KvArgs a) {
  griddep_launch();
  griddep_wait();
  const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (r >= N) return;
  __nv_bfloat16 *dst = a.cache + (long long)a.row_slot[r] * a.slot_stride + (long long)layer * a.layer_stride + (long long)a.row_cpos[r] * a.d_kv;
  const __nv_bfloat16 *src = qkv + (size_t)r * ld_qkv;
  for (int c = lane * 8; c < a.d_kv; c += 256) {
    *reinterpret_cast<uint4 *>(dst + c) = *reinterpret_cast<const uint4 *>(src + col_k + c);
    *reinterpret_cast<uint4 *>(dst + a.kv_stride + c) = *reinterpret_cast<const uint4 *>(src + col_v + c);
  }
}

// Decode attention (split over the keys): every request has ONE query token (row p of the task-sorted batch) that attends the cache
// positions 0 .. cpos (its own k / v were appended just before).  One CTA per (request, KV head, chunk of kc_keys cached
// positions); the query heads of the GQA group share the K / V rows.  Per 128 keys:
//   load     the K and V rows go to shared memory with 16-byte cp.async copies, all in flight at once (coalesced; rows padded by
//            16 bytes so that ldmatrix reads are bank-conflict free);
//   scores   S = Q K^T on mma.sync m16n8k16: the M = 16 rows are the group's query heads (padded with zeros), a warp takes 32 keys;
//   softmax  online per head over the warp's keys, in the accumulator registers (fp32, exp2 with the scale folded in);
//   P V      P (bf16) stays in registers as the A operand, V through ldmatrix.trans.
// (A first version did the two products with scalar FMAs, lane = key: 10 M instructions per launch at two warps per scheduler made
// it latency-bound at 48 us per layer for 37 MB of cache.)
// The four warps' states (m, l, o) are merged in warp order (deterministic).  A request with one chunk writes its output; with
// more, every chunk's CTA stores (o, m, l) per head and the LAST CTA to finish (a counter per (request, KV head), reset by that
// CTA) merges them in chunk order - the result depends on the request's own length only, never on the batch or on timing.
// Memory-bound: 2 * (cpos + 1) * DH * 2 bytes per (request, KV head).
constexpr int kDecGroupMax = 8;
constexpr int kDecKeys = 128;                       // keys per pass of a CTA (4 warps x 32)
template <int DH>
constexpr size_t decode_attention_smem() {
  return sizeof(__nv_bfloat16) * (2 * kDecKeys + 16) * (DH + 8) + sizeof(float) * 2 * 4 * kDecGroupMax;
}
struct DecAttnArgs {
  const __nv_bfloat16 *qkv;
  __nv_bfloat16 *out;
  int ld_qkv, ld_out, n_q_heads, n_kv_heads, layer;
  float scale_log2;
  int kc_keys;                     // cached positions per chunk (multiple of kDecKeys); gridDim.z = chunks of the longest possible sequence
  float *part;                     // [request, q head, chunk, DH + 2] (o unnormalised, m, l)
  unsigned *cnt;                   // [request, KV head], zero between launches
};
template <int DH>
__global__ void __launch_bounds__(128) decode_attention_kernel(const DecAttnArgs d, const KvArgs a) {
  constexpr int G = kDecGroupMax, KS = DH + 8;
  extern __shared__ __align__(16) unsigned char dec_smem[];
  __nv_bfloat16 *s_k = reinterpret_cast<__nv_bfloat16 *>(dec_smem);           // [128][DH + 8]
  __nv_bfloat16 *s_v = s_k + kDecKeys * KS;                                   // [128][DH + 8]
  __nv_bfloat16 *s_q = s_v + kDecKeys * KS;                                   // [16][DH + 8] queries of the group, rows >= group zero
  float *s_m = reinterpret_cast<float *>(s_q + 16 * KS), *s_l = s_m + 4 * G;  // [4][G]
  float *s_o = reinterpret_cast<float *>(s_k);                                // [4][G][DH], reuses the K rows after the last pass
  __shared__ int s_last;
  griddep_launch();
  griddep_wait();
  const int p = blockIdx.x, kvh = blockIdx.y, chunk = blockIdx.z, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int group = d.n_q_heads / d.n_kv_heads;
  const int n_keys = a.row_cpos[p] + 1;
  const int key_lo = chunk * d.kc_keys;
  if (key_lo >= n_keys) return;
  const int key_hi = min(n_keys, key_lo + d.kc_keys), n_chunks = (n_keys + d.kc_keys - 1) / d.kc_keys;
  for (int idx = threadIdx.x; idx < 16 * (DH / 8); idx += blockDim.x) {
    const int g = idx / (DH / 8), pc = idx - g * (DH / 8);
    *reinterpret_cast<uint4 *>(s_q + g * KS + pc * 8) =
        g < group ? *reinterpret_cast<const uint4 *>(d.qkv + (size_t)p * d.ld_qkv + (kvh * group + g) * DH + pc * 8) : make_uint4(0, 0, 0, 0);
  }
  const __nv_bfloat16 *K = a.cache + (long long)a.row_slot[p] * a.slot_stride + (long long)d.layer * a.layer_stride + kvh * DH;
  const __nv_bfloat16 *V = K + a.kv_stride;
  // this thread's softmax row = head hr = lane / 4 of the group (accumulator rows 8 .. 15 of the 16-row MMA tile are padding)
  float oacc[DH / 8][4], m = -INFINITY, l = 0.0f;
#pragma unroll
  for (int nt = 0; nt < DH / 8; ++nt) oacc[nt][0] = oacc[nt][1] = oacc[nt][2] = oacc[nt][3] = 0.0f;
  for (int k0 = key_lo; k0 < key_hi; k0 += kDecKeys) {
    const int nk_cta = min(kDecKeys, key_hi - k0), rows = (nk_cta + 31) & ~31;
    if (k0 > key_lo) __syncthreads();                           // the previous pass is done with the buffers
    for (int idx = threadIdx.x; idx < nk_cta * (DH / 8); idx += blockDim.x) {
      const int row = idx / (DH / 8), pc = idx - row * (DH / 8);
      cp_async_16(s_k + row * KS + pc * 8, K + (long long)(k0 + row) * a.d_kv + pc * 8, 16);
    }
    cp_async_commit();
    for (int idx = threadIdx.x; idx < rows * (DH / 8); idx += blockDim.x) {      // rows past the last key are zero (0 * stale bits could be NaN)
      const int row = idx / (DH / 8), pc = idx - row * (DH / 8);
      const bool ok = row < nk_cta;
      cp_async_16(s_v + row * KS + pc * 8, V + (long long)(k0 + (ok ? row : 0)) * a.d_kv + pc * 8, ok ? 16 : 0);
    }
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();                                            // K rows (and, first pass, the queries) are in shared memory
    const int nk = min(32, nk_cta - warp * 32);                 // this warp's keys in the pass (<= 0: none)
    uint32_t ap[2][4];
    if (nk > 0) {
      // ---- S = Q K^T: 16 (heads, padded) x 32 keys ----
      float sacc[4][4];
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) sacc[nt][0] = sacc[nt][1] = sacc[nt][2] = sacc[nt][3] = 0.0f;
#pragma unroll
      for (int ks = 0; ks < DH / 16; ++ks) {
        uint32_t aq[4];
        ldmatrix_x4(aq, s_q + (lane & 15) * KS + ks * 16 + (lane >> 4) * 8);
#pragma unroll
        for (int np = 0; np < 2; ++np) {
          uint32_t bk[4];
          ldmatrix_x4(bk, s_k + (warp * 32 + np * 16 + (lane >> 4) * 8 + (lane & 7)) * KS + ks * 16 + ((lane >> 3) & 1) * 8);
          const uint32_t b0[2] = {bk[0], bk[1]}, b1[2] = {bk[2], bk[3]};
          mma_bf16_16816(sacc[2 * np], aq, b0);
          mma_bf16_16816(sacc[2 * np + 1], aq, b1);
        }
      }
      // ---- online softmax of row hr over the warp's keys (the thread holds keys 8 nt + 2 (lane % 4) + {0, 1}) ----
      float mc = -INFINITY;
#pragma unroll
      for (int nt = 0; nt < 4; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const bool valid = nt * 8 + 2 * (lane & 3) + e < nk;
          sacc[nt][e] = valid ? sacc[nt][e] * d.scale_log2 : -INFINITY;
          mc = fmaxf(mc, sacc[nt][e]);
        }
      mc = fmaxf(mc, __shfl_xor_sync(0xffffffffu, mc, 1));
      mc = fmaxf(mc, __shfl_xor_sync(0xffffffffu, mc, 2));
      const float mn = fmaxf(m, mc);                            // finite: the warp holds at least one valid key
      const float f = fast_exp2(m - mn);
      float lc = 0.0f;
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) {
        sacc[nt][0] = fast_exp2(sacc[nt][0] - mn);
        sacc[nt][1] = fast_exp2(sacc[nt][1] - mn);
        lc += sacc[nt][0] + sacc[nt][1];
      }
      lc += __shfl_xor_sync(0xffffffffu, lc, 1);
      lc += __shfl_xor_sync(0xffffffffu, lc, 2);
      m = mn;
      l = l * f + lc;
#pragma unroll
      for (int nt = 0; nt < DH / 8; ++nt) { oacc[nt][0] *= f; oacc[nt][1] *= f; }
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {                          // P as the A operand of P V: keys 16 kk .. 16 kk + 15
        ap[kk][0] = pack_bf16(sacc[2 * kk][0], sacc[2 * kk][1]);
        ap[kk][2] = pack_bf16(sacc[2 * kk + 1][0], sacc[2 * kk + 1][1]);
        ap[kk][1] = ap[kk][3] = 0u;
      }
    }
    cp_async_wait<0>();
    __syncthreads();                                            // V rows are in shared memory
    if (nk > 0) {
      // ---- O += P V: 16 x DH ----
#pragma unroll
      for (int kk = 0; kk < 2; ++kk)
#pragma unroll
        for (int dp = 0; dp < DH / 16; ++dp) {
          uint32_t bv[4];
          ldmatrix_x4_trans(bv, s_v + (warp * 32 + kk * 16 + ((lane >> 3) & 1) * 8 + (lane & 7)) * KS + (2 * dp + (lane >> 4)) * 8);
          const uint32_t b0[2] = {bv[0], bv[1]}, b1[2] = {bv[2], bv[3]};
          mma_bf16_16816(oacc[2 * dp], ap[kk], b0);
          mma_bf16_16816(oacc[2 * dp + 1], ap[kk], b1);
        }
    }
  }
  __syncthreads();                                              // every warp is done with the K rows: s_o may overwrite them
  {
    const int hr = lane >> 2;
    if ((lane & 3) == 0) { s_m[warp * G + hr] = m; s_l[warp * G + hr] = l; }
#pragma unroll
    for (int nt = 0; nt < DH / 8; ++nt)
      *reinterpret_cast<float2 *>(&s_o[(warp * G + hr) * DH + nt * 8 + 2 * (lane & 3)]) = make_float2(oacc[nt][0], oacc[nt][1]);
  }
  __syncthreads();
  const int n_cap = gridDim.z;
  for (int idx = threadIdx.x; idx < group * DH; idx += blockDim.x) {
    const int g = idx / DH, e = idx - g * DH;
    float mx = -INFINITY;
#pragma unroll
    for (int w = 0; w < 4; ++w) mx = fmaxf(mx, s_m[w * G + g]);
    float L = 0.0f, O = 0.0f;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const float f = fast_exp2(s_m[w * G + g] - mx);        // a warp that saw no key: m = -inf -> f = 0
      L = fmaf(s_l[w * G + g], f, L);
      O = fmaf(s_o[(w * G + g) * DH + e], f, O);
    }
    if (n_chunks == 1) {
      d.out[(size_t)p * d.ld_out + (kvh * group + g) * DH + e] = __float2bfloat16(O / L);
    } else {
      float *dst = d.part + (((size_t)p * d.n_q_heads + kvh * group + g) * n_cap + chunk) * (DH + 2);
      dst[e] = O;
      if (e == 0) { dst[DH] = mx; dst[DH + 1] = L; }
    }
  }
  if (n_chunks == 1) return;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(&d.cnt[p * d.n_kv_heads + kvh], 1u) == (unsigned)(n_chunks - 1);
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x == 0) d.cnt[p * d.n_kv_heads + kvh] = 0u;      // ready for the next launch
  for (int idx = threadIdx.x; idx < group * DH; idx += blockDim.x) {
    const int g = idx / DH, e = idx - g * DH;
    const float *src = d.part + (((size_t)p * d.n_q_heads + kvh * group + g) * n_cap) * (DH + 2);
    float cm[16], cl[16], co[16];                          // every chunk's (m, l, o) in flight at once (n_cap <= 16)
#pragma unroll
    for (int c = 0; c < 16; ++c) {
      const bool ok = c < n_chunks;
      const float *q = src + (size_t)(ok ? c : 0) * (DH + 2);
      cm[c] = ok ? __ldcg(q + DH) : -INFINITY;
      cl[c] = ok ? __ldcg(q + DH + 1) : 0.0f;
      co[c] = ok ? __ldcg(q + e) : 0.0f;
    }
    float mx = -INFINITY;
#pragma unroll
    for (int c = 0; c < 16; ++c) mx = fmaxf(mx, cm[c]);
    float L = 0.0f, O = 0.0f;
#pragma unroll
    for (int c = 0; c < 16; ++c) {                         // chunk order; a chunk past the end has f = 0
      const float f = fast_exp2(cm[c] - mx);
      L = fmaf(cl[c], f, L);
      O = fmaf(co[c], f, O);
    }
    d.out[(size_t)p * d.ld_out + (kvh * group + g) * DH + e] = __float2bfloat16(O / L);
  }
}

// Final norm of every request's LAST token row -> bf16 [B, d] (sorted request order): the A operand of the LM-head GEMM.
template <int kVec>
__global__ void __launch_bounds__(256) last_row_norm_kernel(const float *__restrict__ X, const int *__restrict__ cu_tok, __nv_bfloat16 *__restrict__ Y,
                                                            const __nv_bfloat16 *__restrict__ g, const __nv_bfloat16 *__restrict__ b, int B, float eps, int rms) {
  griddep_launch();
  griddep_wait();
  const int p = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (p >= B) return;
  constexpr int d = 128 * kVec;
  const float4 *x = reinterpret_cast<const float4 *>(X + (size_t)(cu_tok[p + 1] - 1) * d);
  float4 v[kVec];
  float s = 0.0f;
#pragma unroll
  for (int j = 0; j < kVec; ++j) { v[j] = x[j * 32 + lane]; s += v[j].x + v[j].y + v[j].z + v[j].w; }
  float mean = 0.0f;
  if (!rms) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    mean = s * (1.0f / d);
  }
  float qq = 0.0f;
#pragma unroll
  for (int j = 0; j < kVec; ++j) {
    const float a0 = v[j].x - mean, a1 = v[j].y - mean, a2 = v[j].z - mean, a3 = v[j].w - mean;
    qq += a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) qq += __shfl_xor_sync(0xffffffffu, qq, o);
  const float inv = rsqrtf(qq * (1.0f / d) + eps);
  uint2 *y = reinterpret_cast<uint2 *>(Y + (size_t)p * d);
#pragma unroll
  for (int j = 0; j < kVec; ++j) {
    const int c4 = j * 32 + lane;
    const uint2 gg = reinterpret_cast<const uint2 *>(g)[c4];
    float o0 = (v[j].x - mean) * inv * bf16_lo(gg.x), o1 = (v[j].y - mean) * inv * bf16_hi(gg.x);
    float o2 = (v[j].z - mean) * inv * bf16_lo(gg.y), o3 = (v[j].w - mean) * inv * bf16_hi(gg.y);
    if (b) {
      const uint2 bb = reinterpret_cast<const uint2 *>(b)[c4];
      o0 += bf16_lo(bb.x); o1 += bf16_hi(bb.x); o2 += bf16_lo(bb.y); o3 += bf16_hi(bb.y);
    }
    y[c4] = make_uint2(pack_bf16(o0, o1), pack_bf16(o2, o3));
  }
}

// LM scores of sorted request p -> the caller's buffers in ORIGINAL request order: scores[perm[p], :] (optional) and the greedy
// next token argmax (lowest index on ties; optional).  One CTA per request.
__global__ void __launch_bounds__(256) scores_out_kernel(const float *__restrict__ sorted_scores, const int *__restrict__ perm, int vocab,
                                                         float *__restrict__ scores, int *__restrict__ next_tokens) {
  __shared__ float s_v[8];
  __shared__ int s_i[8];
  griddep_launch();
  griddep_wait();
  const int p = blockIdx.x, i = perm[p], warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const float *src = sorted_scores + (size_t)p * vocab;
  float best = -INFINITY;
  int bi = 0x7fffffff;
  for (int c = threadIdx.x; c < vocab; c += blockDim.x) {
    const float v = src[c];
    if (scores) scores[(size_t)i * vocab + c] = v;
    if (v > best) { best = v; bi = c; }                   // ascending c per thread: the first maximum is kept
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, best, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
  }
  if (lane == 0) { s_v[warp] = best; s_i[warp] = bi; }
  __syncthreads();
  if (threadIdx.x == 0 && next_tokens) {
    for (int w = 1; w < 8; ++w)
      if (s_v[w] > best || (s_v[w] == best && s_i[w] < bi)) { best = s_v[w]; bi = s_i[w]; }
    next_tokens[i] = bi;
  }
}

// ============================================================================= small-M projections (decode): split-K reduce, row-wise shrink
// Sums the fp32 partial accumulators of a split-K projection in split order (deterministic) and applies the epilogue the GEMM
// would have applied: + bias of the column's weight source, then either the fp32 residual update (X += ...) or activation and a
// bf16 store.  One thread per 4 consecutive columns of a row.
struct SplitKReduceArgs {
  const float *partial;            // [k_split, split_rows, N]
  int k_split, split_rows, M, N;
  int mode;                        // 0 bf16 out, 1 bf16 out + GeLU(erf), 2 bf16 out + ReLU, 3 fp32 residual X += ., 4 SwiGLU (N = 2 d_ffn,
                                   //   128-column chunks alternate gate / up; bf16 out [M, N / 2])
  const float *delta;              // [M, N] fp32 LoRA delta of the rows' tasks (row_expand_kernel), added before bias / activation; or NULL
  const __nv_bfloat16 *bias[3];    // per weight source (NULL = none)
  int src_end_col[3];              // first column AFTER source s (cumulative)
  __nv_bfloat16 *out_bf16;
  float *X;
  int ld_out;
};
__device__ __forceinline__ float splitk_gelu(float x) { return 0.5f * x * (1.0f + erff(x * 0.70710678118654752f)); }
__global__ void __launch_bounds__(256) splitk_reduce_kernel(const SplitKReduceArgs a) {
  griddep_launch();
  griddep_wait();
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  auto column_sum = [&](int r, int c) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 8
    for (int ks = 0; ks < a.k_split; ++ks) {
      const float4 v = *reinterpret_cast<const float4 *>(a.partial + ((size_t)ks * a.split_rows + r) * a.N + c);
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    if (a.delta) {
      const float4 v = *reinterpret_cast<const float4 *>(a.delta + (size_t)r * a.N + c);
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    return acc;
  };
  if (a.mode == 4) {                                    // SwiGLU: feature f = 128 q + j -> gate column 256 q + j, up column 256 q + 128 + j
    const int f4 = a.N / 8;
    if (idx >= (long long)a.M * f4) return;
    const int r = (int)(idx / f4), f = (int)(idx - (long long)r * f4) * 4;
    const int cg = (f >> 7) * 256 + (f & 127);
    float4 g = column_sum(r, cg), u = column_sum(r, cg + 128);
    if (const __nv_bfloat16 *b = a.bias[0]) { const uint2 bv = *reinterpret_cast<const uint2 *>(b + f); g.x += bf16_lo(bv.x); g.y += bf16_hi(bv.x); g.z += bf16_lo(bv.y); g.w += bf16_hi(bv.y); }
    if (const __nv_bfloat16 *b = a.bias[1]) { const uint2 bv = *reinterpret_cast<const uint2 *>(b + f); u.x += bf16_lo(bv.x); u.y += bf16_hi(bv.x); u.z += bf16_lo(bv.y); u.w += bf16_hi(bv.y); }
    auto silu = [](float x) { return x / (1.0f + __expf(-x)); };
    *reinterpret_cast<uint2 *>(a.out_bf16 + (size_t)r * a.ld_out + f) =
        make_uint2(pack_bf16(silu(g.x) * u.x, silu(g.y) * u.y), pack_bf16(silu(g.z) * u.z, silu(g.w) * u.w));
    return;
  }
  const int n4 = a.N / 4;
  if (idx >= (long long)a.M * n4) return;
  const int r = (int)(idx / n4), c = (int)(idx - (long long)r * n4) * 4;
  float4 acc = column_sum(r, c);
  int s = 0, begin = 0;
  if (c >= a.src_end_col[0]) { s = 1; begin = a.src_end_col[0]; }
  if (c >= a.src_end_col[1]) { s = 2; begin = a.src_end_col[1]; }
  if (const __nv_bfloat16 *b = a.bias[s]) {
    const uint2 bv = *reinterpret_cast<const uint2 *>(b + (c - begin));
    acc.x += bf16_lo(bv.x); acc.y += bf16_hi(bv.x); acc.z += bf16_lo(bv.y); acc.w += bf16_hi(bv.y);
  }
  if (a.mode == 3) {
    float4 *x = reinterpret_cast<float4 *>(a.X + (size_t)r * a.ld_out + c);
    float4 o = *x;
    o.x += acc.x; o.y += acc.y; o.z += acc.z; o.w += acc.w;
    *x = o;
    return;
  }
  if (a.mode == 1) { acc.x = splitk_gelu(acc.x); acc.y = splitk_gelu(acc.y); acc.z = splitk_gelu(acc.z); acc.w = splitk_gelu(acc.w); }
  else if (a.mode == 2) { acc.x = fmaxf(acc.x, 0.f); acc.y = fmaxf(acc.y, 0.f); acc.z = fmaxf(acc.z, 0.f); acc.w = fmaxf(acc.w, 0.f); }
  *reinterpret_cast<uint2 *>(a.out_bf16 + (size_t)r * a.ld_out + c) = make_uint2(pack_bf16(acc.x, acc.y), pack_bf16(acc.z, acc.w));
}

// The reduction of a residual projection (attention output, FFN down) fused with the norm that follows it: one CTA of 128 threads
// per row.  X[row] += sum of the partials (split order) + delta + bias, then LayerNorm / RMSNorm of the updated row -> bf16 Y (the
// same arithmetic as norm_kernel: mean, then the sum of squared deviations, fp32).  g == NULL: no norm follows (last layer).
struct ReduceNormArgs {
  const float *partial;            // [k_split, split_rows, N]
  int k_split, split_rows, N;      // N = d_model (a multiple of 4, <= 4096)
  const float *delta;              // [M, N] or NULL
  const __nv_bfloat16 *bias;       // [N] or NULL
  float *X;                        // [M, N] fp32 residual stream, updated in place
  __nv_bfloat16 *Y;                // [M, N] bf16 normalised rows
  const __nv_bfloat16 *g, *b;      // norm weight / bias (b NULL for RMSNorm)
  float eps;
  int rms;
};
__device__ __forceinline__ float block_sum_fixed(float v, float *s_red) {    // every thread gets the sum; fixed order; blockDim a multiple of 32
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();                                                            // s_red free again
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float t = 0.0f;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += s_red[w];
  return t;
}
// One CTA per row, one thread per 4 columns (blockDim = N / 4 rounded up to a warp, <= 1024): the thread's partials of every
// split, the delta and the residual are all requested before the first is used.
__global__ void __launch_bounds__(1024) reduce_resid_norm_kernel(const ReduceNormArgs a) {
  __shared__ float s_red[32];
  griddep_launch();
  griddep_wait();
  const int r = blockIdx.x, n4 = a.N >> 2, c4 = threadIdx.x;
  const bool on = c4 < n4;
  const int c = 4 * c4;
  const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
  float4 *xp = reinterpret_cast<float4 *>(a.X + (size_t)r * a.N + c);
  const float4 x0 = on ? *xp : z4;
  const float4 dl = (on && a.delta) ? *reinterpret_cast<const float4 *>(a.delta + (size_t)r * a.N + c) : z4;
  float4 acc = z4;
  if (on) {
    const float *part = a.partial + (size_t)r * a.N + c;
#pragma unroll 8
    for (int ks = 0; ks < a.k_split; ++ks) {                    // split order
      const float4 q = *reinterpret_cast<const float4 *>(part + (size_t)ks * a.split_rows * a.N);
      acc.x += q.x; acc.y += q.y; acc.z += q.z; acc.w += q.w;
    }
    acc.x += dl.x; acc.y += dl.y; acc.z += dl.z; acc.w += dl.w;
    if (a.bias) {
      const uint2 bv = *reinterpret_cast<const uint2 *>(a.bias + c);
      acc.x += bf16_lo(bv.x); acc.y += bf16_hi(bv.x); acc.z += bf16_lo(bv.y); acc.w += bf16_hi(bv.y);
    }
  }
  const float4 v = make_float4(x0.x + acc.x, x0.y + acc.y, x0.z + acc.z, x0.w + acc.w);
  if (on) *xp = v;
  if (!a.g) return;
  float mean = 0.0f;
  if (!a.rms) mean = block_sum_fixed(on ? (v.x + v.y) + (v.z + v.w) : 0.0f, s_red) * (1.0f / a.N);
  const float a0 = v.x - mean, a1 = v.y - mean, a2 = v.z - mean, a3 = v.w - mean;
  const float inv = rsqrtf(block_sum_fixed(on ? a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3 : 0.0f, s_red) * (1.0f / a.N) + a.eps);
  if (!on) return;
  const uint2 gg = reinterpret_cast<const uint2 *>(a.g)[c4];
  float o0 = a0 * inv * bf16_lo(gg.x), o1 = a1 * inv * bf16_hi(gg.x), o2 = a2 * inv * bf16_lo(gg.y), o3 = a3 * inv * bf16_hi(gg.y);
  if (a.b) {
    const uint2 bb = reinterpret_cast<const uint2 *>(a.b)[c4];
    o0 += bf16_lo(bb.x); o1 += bf16_hi(bb.x); o2 += bf16_lo(bb.y); o3 += bf16_hi(bb.y);
  }
  reinterpret_cast<uint2 *>(a.Y + (size_t)r * a.N)[c4] = make_uint2(pack_bf16(o0, o1), pack_bf16(o2, o3));
}

// The reduction of the fused q / k / v projection of a decode iteration, with what follows it: + delta + bias, RoPE at the row's
// cache position (rotate-half pairs (j, j + dh/2), applied in fp32 to the unrounded sums - one rounding, as in the prefill GEMM's
// fused epilogue), bf16 store to the qkv buffer, and the k / v heads appended to the KV cache.  One thread per (row, head, 4 pairs).
struct QkvReduceArgs {
  const float *partial;
  int k_split, split_rows, M, N;   // N = d_q + 2 d_kv
  const float *delta;              // [M, N] or NULL
  const __nv_bfloat16 *bias[3];    // q / k / v
  __nv_bfloat16 *qkv;              // [M, N]
  int n_q_heads, n_kv_heads, dh, layer;
  const float2 *rope_cs;           // [max_seq, dh / 2] (cos, sin), or NULL: no rotation
};
__global__ void __launch_bounds__(256) qkv_reduce_rope_kernel(const QkvReduceArgs a, const KvArgs kv) {
  griddep_launch();
  griddep_wait();
  const int half = a.dh >> 1, vph = half >> 2, n_heads = a.n_q_heads + 2 * a.n_kv_heads;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)a.M * n_heads * vph) return;
  const int jv = (int)(idx % vph), h = (int)((idx / vph) % n_heads), r = (int)(idx / ((long long)vph * n_heads));
  const int src = h < a.n_q_heads ? 0 : h < a.n_q_heads + a.n_kv_heads ? 1 : 2;
  const int c = h * a.dh + 4 * jv;                                  // first-half columns c .. c + 3, second half c + half ..
  const int c_src = c - (src == 0 ? 0 : src == 1 ? a.n_q_heads * a.dh : (a.n_q_heads + a.n_kv_heads) * a.dh);
  auto column_sum = [&](int col, int col_src) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 8
    for (int ks = 0; ks < a.k_split; ++ks) {
      const float4 q = *reinterpret_cast<const float4 *>(a.partial + ((size_t)ks * a.split_rows + r) * a.N + col);
      acc.x += q.x; acc.y += q.y; acc.z += q.z; acc.w += q.w;
    }
    if (a.delta) {
      const float4 q = *reinterpret_cast<const float4 *>(a.delta + (size_t)r * a.N + col);
      acc.x += q.x; acc.y += q.y; acc.z += q.z; acc.w += q.w;
    }
    if (const __nv_bfloat16 *b = a.bias[src]) {
      const uint2 bv = *reinterpret_cast<const uint2 *>(b + col_src);
      acc.x += bf16_lo(bv.x); acc.y += bf16_hi(bv.x); acc.z += bf16_lo(bv.y); acc.w += bf16_hi(bv.y);
    }
    return acc;
  };
  float4 x1 = column_sum(c, c_src), x2 = column_sum(c + half, c_src + half);
  const int pos = kv.row_cpos[r];
  if (a.rope_cs && src < 2) {
    const float4 *cs = reinterpret_cast<const float4 *>(a.rope_cs + (size_t)pos * half + 4 * jv);
    const float4 ca = cs[0], cb = cs[1];                            // (cos, sin) of pairs 4 jv, 4 jv + 1 | 4 jv + 2, 4 jv + 3
    const float4 y1 = make_float4(x1.x * ca.x - x2.x * ca.y, x1.y * ca.z - x2.y * ca.w, x1.z * cb.x - x2.z * cb.y, x1.w * cb.z - x2.w * cb.w);
    const float4 y2 = make_float4(x2.x * ca.x + x1.x * ca.y, x2.y * ca.z + x1.y * ca.w, x2.z * cb.x + x1.z * cb.y, x2.w * cb.z + x1.w * cb.w);
    x1 = y1; x2 = y2;
  }
  const uint2 o1 = make_uint2(pack_bf16(x1.x, x1.y), pack_bf16(x1.z, x1.w)), o2 = make_uint2(pack_bf16(x2.x, x2.y), pack_bf16(x2.z, x2.w));
  __nv_bfloat16 *q = a.qkv + (size_t)r * a.N + c;
  *reinterpret_cast<uint2 *>(q) = o1;
  *reinterpret_cast<uint2 *>(q + half) = o2;
  if (src > 0) {                                                    // k / v head: append to the cache
    __nv_bfloat16 *dst = kv.cache + (long long)kv.row_slot[r] * kv.slot_stride + (long long)a.layer * kv.layer_stride + (src == 2 ? kv.kv_stride : 0) +
                         (long long)pos * kv.d_kv + c_src;
    *reinterpret_cast<uint2 *>(dst) = o1;
    *reinterpret_cast<uint2 *>(dst + half) = o2;
  }
}

// Row-wise LoRA for small batches (decode iterations): delta[row, cols of target] = s_t (x_row A_t^T) B_t^T for every target of an
// input group, on CUDA cores (row_shrink_kernel, then row_expand_kernel).  With a handful of rows per task the segmented tensor-core path would
// load a 256-row U tile and a slab block per (tile, task) for a few rows of work; here a row reads its own task's slab columns
// once.  Rows whose task has no adapter on the target get zeros (the reduce kernel adds the delta unconditionally).
struct RowLoraArgs {
  const __nv_bfloat16 *x;          // [M, K] bf16 input of the projection group
  int M, K, ld_delta;
  float *delta;                    // [M, ld_delta] fp32
  int n_tg;
  int tg[3];                       // target ids
  const __nv_bfloat16 *slabA[3];   // [Rcap, K] of this layer
  const __nv_bfloat16 *slabB[3];   // RANK-MAJOR [Rcap, d_out] of this layer (Backbone::slabBt)
  int d_out[3], col0[3];           // output width of the target, its first column in delta
  int interleave2;                 // SwiGLU: target i owns the 128-column chunks 2 q + i (feature 128 q + j -> column 256 q + 128 i + j)
  int Rcap;
  const int *row_req, *task_sorted, *task_coff;
  const unsigned char *task_trpad;
  const float *task_scale;
};
// Both kernels are bound by memory latency and by the number of separate cache lines they touch, not by arithmetic, so
//  * a warp streams its share in batches of eight 16-byte loads per lane, the next batch in flight while the current one is used;
//  * adjacent lanes read adjacent 16 bytes: a shrink warp reads 512 contiguous bytes of a slab row per instruction, an expand warp
//    covers the r_pad * 2 contiguous bytes of a column of B with r_pad / 8 adjacent lanes (one cache-line lookup per column instead
//    of one per 16 bytes).
constexpr int kRowShrinkK = 1024;                   // longest input range of one shrink warp
__device__ __forceinline__ float dot8_bf16(const uint4 &p, const uint4 &q) {
  return bf16_lo(p.x) * bf16_lo(q.x) + bf16_hi(p.x) * bf16_hi(q.x) + bf16_lo(p.y) * bf16_lo(q.y) + bf16_hi(p.y) * bf16_hi(q.y) +
         bf16_lo(p.z) * bf16_lo(q.z) + bf16_hi(p.z) * bf16_hi(q.z) + bf16_lo(p.w) * bf16_lo(q.w) + bf16_hi(p.w) * bf16_hi(q.w);
}
// u_part[kc, row, i, j] = s_t <x_row[range kc], A_t[j, range kc]> for every rank j of target i (fp32, [nkc, M, 3, 64]); the expand
// kernel adds the nkc partial sums in kc order.  Warp w of the CTA (row, target, range) takes the ranks 8 w .. 8 w + 7.
__global__ void __launch_bounds__(256) row_shrink_kernel(const RowLoraArgs a, float *__restrict__ u, int k_range) {
  griddep_launch();
  griddep_wait();
  const int r = blockIdx.x, i = blockIdx.y, kc = blockIdx.z, tg = a.tg[i], warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = a.task_sorted[a.row_req[r]];
  const int rp = a.task_trpad[t * 7 + tg];               // padded rank (multiple of 16); 0 = no adapter on this target
  if (8 * warp >= rp) return;
  const float sc = a.task_scale[t * 7 + tg];
  const int k_lo = kc * k_range, k_hi = min(a.K, k_lo + k_range);
  const __nv_bfloat16 *x = a.x + (size_t)r * a.K + lane * 8;
  const __nv_bfloat16 *A = a.slabA[i] + (size_t)(a.task_coff[t] + 8 * warp) * a.K + lane * 8;
  const uint4 z4 = make_uint4(0, 0, 0, 0);
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  auto load = [&](uint4 &xv, uint4 (&v)[8], int k0) {
    const bool ok = k0 + lane * 8 < k_hi;
    xv = ok ? *reinterpret_cast<const uint4 *>(x + k0) : z4;
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = ok ? *reinterpret_cast<const uint4 *>(A + (size_t)j * a.K + k0) : z4;
  };
  auto comp = [&](const uint4 &xv, const uint4 (&v)[8]) {
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] += dot8_bf16(v[j], xv);
  };
  uint4 xa, xb, va[8], vb[8];
  load(xa, va, k_lo);
  for (int k0 = k_lo; k0 < k_hi; k0 += 512) {
    const bool more1 = k0 + 256 < k_hi, more2 = k0 + 512 < k_hi;
    if (more1) load(xb, vb, k0 + 256);
    comp(xa, va);
    if (more2) load(xa, va, k0 + 512);
    if (more1) comp(xb, vb);
  }
#pragma unroll
  for (int j = 0; j < 8; ++j)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[j] += __shfl_xor_sync(0xffffffffu, acc[j], o);
  if (lane == 0) {
    float4 *dst = reinterpret_cast<float4 *>(u + (((size_t)kc * a.M + r) * 3 + i) * 64 + 8 * warp);
    dst[0] = make_float4(acc[0] * sc, acc[1] * sc, acc[2] * sc, acc[3] * sc);
    dst[1] = make_float4(acc[4] * sc, acc[5] * sc, acc[6] * sc, acc[7] * sc);
  }
}
// delta[row, column of (target i, c)] = sum_j u[row, i, j] Bt_t[j, c] for the CTA's 512 columns.  B is read RANK-MAJOR (slabBt:
// [Rcap, d_out], a task's rank rows contiguous): the column-major copy the tensor-core path uses would make every column a separate
// 32 - 128 byte access 2 Rcap bytes apart, which DRAM serves at a fraction of its streaming rate (measured: 1.8 TB/s, 31 us for the
// gate / up pair).  Thread (g = tid / 64, cg = tid % 64) takes the ranks 16 g .. 16 g + 15 of the columns 8 cg .. 8 cg + 7 - sixteen
// 16-byte loads, all in flight at once, a warp reading 512 contiguous bytes per load - and the four rank groups are added in g order
// through shared memory.
constexpr int kRowExpandCols = 512;
__global__ void __launch_bounds__(256) row_expand_kernel(const RowLoraArgs a, const float *__restrict__ u, int nkc) {
  __shared__ float s_u[64];
  __shared__ __align__(16) float s_acc[4][kRowExpandCols];
  griddep_launch();
  griddep_wait();
  const int r = blockIdx.x, i = blockIdx.y, tg = a.tg[i], g = threadIdx.x >> 6, cg = threadIdx.x & 63;
  const int dout = a.d_out[i];
  const int c_base = blockIdx.z * kRowExpandCols;
  if (c_base >= dout) return;
  const int t = a.task_sorted[a.row_req[r]];
  const int rp = a.task_trpad[t * 7 + tg];
  float *dst = a.delta + (size_t)r * a.ld_delta;
  const int c2 = c_base + 2 * threadIdx.x;               // the two columns this thread writes at the end
  const int o2 = a.interleave2 ? ((c2 >> 7) * 256 + i * 128 + (c2 & 127)) : a.col0[i] + c2;
  if (rp == 0) {                                         // no adapter: the reduce kernel adds the delta unconditionally
    if (c2 < dout) *reinterpret_cast<float2 *>(dst + o2) = make_float2(0.f, 0.f);
    return;
  }
  const int c = c_base + 8 * cg;
  const bool live = 16 * g < rp && c < dout;
  const uint4 z4 = make_uint4(0, 0, 0, 0);
  const __nv_bfloat16 *B = a.slabB[i] + (size_t)(a.task_coff[t] + 16 * g) * dout + c;
  uint4 v[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = live ? *reinterpret_cast<const uint4 *>(B + (size_t)j * dout) : z4;
  if (threadIdx.x < 64) {
    float s = 0.0f;
    if ((int)threadIdx.x < rp)
      for (int kc = 0; kc < nkc; ++kc) s += u[(((size_t)kc * a.M + r) * 3 + i) * 64 + threadIdx.x];
    s_u[threadIdx.x] = s;
  }
  __syncthreads();
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const float uj = s_u[16 * g + j];
    acc[0] = fmaf(uj, bf16_lo(v[j].x), acc[0]); acc[1] = fmaf(uj, bf16_hi(v[j].x), acc[1]);
    acc[2] = fmaf(uj, bf16_lo(v[j].y), acc[2]); acc[3] = fmaf(uj, bf16_hi(v[j].y), acc[3]);
    acc[4] = fmaf(uj, bf16_lo(v[j].z), acc[4]); acc[5] = fmaf(uj, bf16_hi(v[j].z), acc[5]);
    acc[6] = fmaf(uj, bf16_lo(v[j].w), acc[6]); acc[7] = fmaf(uj, bf16_hi(v[j].w), acc[7]);
  }
  *reinterpret_cast<float4 *>(&s_acc[g][8 * cg]) = make_float4(acc[0], acc[1], acc[2], acc[3]);
  *reinterpret_cast<float4 *>(&s_acc[g][8 * cg + 4]) = make_float4(acc[4], acc[5], acc[6], acc[7]);
  __syncthreads();
  if (c2 < dout) {
    const int cl = 2 * threadIdx.x;
    float2 o = *reinterpret_cast<const float2 *>(&s_acc[0][cl]);
#pragma unroll
    for (int gg = 1; gg < 4; ++gg) {                     // rank groups past the task's rank hold zeros
      const float2 q = *reinterpret_cast<const float2 *>(&s_acc[gg][cl]);
      o.x += q.x; o.y += q.y;
    }
    *reinterpret_cast<float2 *>(dst + o2) = o;
  }
}

// Registration: the rank-major copy of one layer's B of an adapter, Bt[j, c] = B[c, j] for j < rank, zero for the padding ranks.
__global__ void lora_bt_fill_kernel(const __nv_bfloat16 *__restrict__ B, __nv_bfloat16 *__restrict__ Bt, int dout, int rank, int rp) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)dout * rp) return;
  const int j = (int)(idx / dout), c = (int)(idx - (size_t)j * dout);
  Bt[idx] = j < rank ? B[(size_t)c * rank + j] : __float2bfloat16(0.0f);
}

}  // namespace fmx
