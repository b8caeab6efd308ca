// CTA-pair (cta_group::2) tcgen05 / TMEM / TMA GEMM for the backbone projections, with the per-task
// LoRA expand fused in as extra K-steps and a shared-memory staged epilogue that leaves through TMA.
//
//   C[M, N] = A[M, K] · W[N, K]^T  (+ Σ_blocks  U_blk[256, r_pad] · B_task[N, r_pad]^T)      fp32 in TMEM
//
// Why a pair: one SM's 128x256 tile pulls (128+256)·64·2 B = 48 KB of operands from L2 per 512 tensor
// cycles; at 148 SMs that saturates the L2->SM fabric at ~65 % tensor utilisation (profiles/r1_01).
// Two SMs of a cluster share one 256 x kBN tile: each loads its own 128 rows of A and HALF of the W
// rows (32 KB per SM per k-block for kBN = 256), and one tcgen05.mma.cta_group::2 issued by the
// leader CTA multiplies [A0; A1] by [W0; W1]^T into both CTAs' TMEM.
//
// Rows are task-sorted token rows (S1).  The N axis is cut into 128-column CHUNKS; a chunk names its
// weight source (q | k | v, gate | up, or the single matrix), so fused QKV and SwiGLU gate/up need no
// repacked weights.  kBN = 256: the pair tile holds two chunks (CTA r loads chunk r's 128 W rows);
// kBN = 128: one chunk (CTA r loads 64 of its W rows).
//
// LoRA expand (BASELINE.json north_star item 4): after the main K loop, for every (256-row tile, task)
// BLOCK of the tile and every chunk whose source has an adapter for that task, r_pad/16 more K-steps
// (M = 256, N = 128) with A = the block's masked shrink output U (rows of other tasks are zero) and
// B = that task's B-slab columns go into the SAME TMEM accumulator, before the epilogue.  No segment
// padding: a tile may span any number of tasks.
//
// Warp roles (384 threads per CTA, persistent over tiles, 1 CTA/SM, cluster of 2):
//   warp 0   TMA producer (lane 0, both CTAs): own A rows + own W half; bytes complete on the LEADER's
//            full barrier (count 2: one arrive.expect_tx per CTA)
//   warp 1   tcgen05.mma issuer (lane 0, leader CTA only); tcgen05.commit multicast frees the smem
//            stage in both CTAs and publishes the accumulator to both CTAs' epilogues
//   warp 2   TMEM alloc / dealloc (cta_group::2, both CTAs)
//   warps 4-11  epilogue: two warpgroups x 128 threads; thread = accumulator row (TMEM lane);
//            tcgen05.ld -> bias / activation / SwiGLU -> 128B-swizzled staging tile in smem ->
//            TMA store (bf16 / fp32) or TMA reduce-add (fp32 residual stream, one add per element)
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gemm.cuh"
#include "ptx.cuh"

namespace fmx {

constexpr int kPairRows = 256;                    // rows of a pair tile (2 x 128)
// Epilogue staging: 2 warpgroups x kBufs buffers x 16 KB.  kDeep = false: two buffers per warpgroup (the bf16 / SwiGLU / RoPE
// epilogues overlap a box's TMA store with the next box's conversion); kDeep = true: ONE buffer and one more pipeline stage
// instead, which is what the fp32-residual GEMMs want (short K, mainloop-latency-bound: cfg2 O projection 1.41 -> 1.31 ms).
template <bool kDeep>
__host__ __device__ constexpr int pair_staging_bytes() { return 2 * (kDeep ? 1 : 2) * 16384; }

struct PairGemmParams {
  CUtensorMap amap;        // A [M, K] bf16, box {64, 128}
  CUtensorMap wmap[3];     // weight sources [rows_s, K] bf16, box {64, kBN/2}
  CUtensorMap wmap_h[3];   // the same sources with box {64, 64}: W rows of a HALF tile (kBN = 256 only)
  CUtensorMap umap;        // U [n_blk_cap*256, 192] bf16, box {64, 128}
  CUtensorMap lmap[3];     // B-slabs [d_out_s, Rcap] bf16, box {64, 64}
  CUtensorMap omap;        // output [M, ld]: bf16 box {64, 128}, or fp32 box {32, 128}
  int M, K;
  int n_chunks;            // N / 128
  int n_ptiles;            // ceil(M / 256)
  int expand_wide;         // 1: same-source whole tiles run their LoRA expand as one N = 256 step per block (A/B knob)
  int reverse;             // 1: row tiles are walked from the last to the first (the producer of this GEMM's input wrote
                           // ascending: its most recent rows are the ones still in L2)
  int n_full;              // kBN = 256: tiles [0, n_full) are 256 x 256; each later tile is cut into two 256 x 128 halves
                           // taken by different pairs, so a short last wave costs half a tile time (-1 = no half tiles)
  int mode;                // GemmMode (not GM_SHRINK)
  int interleave2;         // chunk c -> source c&1, row (c>>1)*128  (SwiGLU)
  int has_lora;
  int src_end[3];          // cumulative chunk count per source (non-interleaved)
  int lora_tgt[3];         // target id of source s, or -1
  int uslot[3];            // U column block (x64) of source s
  const __nv_bfloat16 *bias[3];
  const int *tile_blk_off, *blk_task;   // S1 block table over 256-row tiles
  const int *task_coff;
  const unsigned char *task_trpad;
  const float *posb;       // [max_seq, ld_pos] fp32 (embed)
  const int *row_pos;
  int ld_pos;
  // ---- fused LoRA shrink (n_sh > 0): the first *n_blk work items compute U_blk = s_t · x A_t^T for the targets that read
  // this GEMM's own input, one item per (256-row tile, task) block; the expand steps of the regular tiles wait for them
  CUtensorMap smap[3];     // A-slabs [Rcap, K] of the shrink targets, box {64, 64}
  int n_sh;                // number of shrink targets (0 = none; 3 needs kBN = 256)
  int sh_tg[3];            // their target ids
  const int *blk_tile, *blk_lo, *blk_hi, *n_blk;
  const float *task_scale; // [T*7] alpha / r
  __nv_bfloat16 *U;        // [n_blk_cap*256, 192]
  unsigned *u_flag;        // one counter: arrivals of the epilogue warps that wrote a U block (monotonic over a forward)
  unsigned *err;           // the context's device error word (bit 1: the fused-shrink wait timed out)
  unsigned u_epoch;        // 1, 2, ... over the fused launches of a forward: this launch's U is complete when the counter
                           // reaches 16 (epilogue warps of a pair) * n_blk * u_epoch
  // ---- partial-output mode / split-K (small M: a weight matrix with few N tiles would be streamed by a handful of CTA pairs).
  // k_split >= 1 (0 = off): work item
  // (tile, ks) runs k-blocks [ks * kb_per_split, ...) of a whole tile and stores its fp32 partial accumulator with a plain TMA
  // store to pmap rows [ks * split_rows + row, ...); splitk_reduce_kernel adds the partials in split order (deterministic) and
  // applies the epilogue.  The LoRA expand steps belong to split 0.
  CUtensorMap pmap;        // partials [k_split * split_rows, N] fp32, box {32, 128}
  int k_split, kb_per_split, split_rows;
  const float2 *rope_cs;   // [64, rope_ld] (cos, sin), pair-index major: fused rotate-half RoPE for head_dim 128 (chunk = head), or NULL
  int rope_ld;             // positions per pair index (= max_seq)
  int rope_src_mask;       // bit s: source s (q | k | v) is rotated
};

__device__ __forceinline__ void pair_chunk_source(const PairGemmParams &p, int c, int &s, int &r0) {
  if (p.interleave2) {
    s = c & 1;
    r0 = (c >> 1) * kChunk;
  } else {
    s = 0;
    int begin = 0;
    if (c >= p.src_end[0]) { s = 1; begin = p.src_end[0]; }
    if (c >= p.src_end[1]) { s = 2; begin = p.src_end[1]; }
    r0 = (c - begin) * kChunk;
  }
}

template <int kBN>
__host__ __device__ constexpr int pair_stage_bytes() { return kATileBytes + (kBN / 2) * kBK * 2; }
template <int kBN, bool kDeep>
__host__ __device__ constexpr int pair_stages() { return (kBN == 256 ? 5 : 6) + (kDeep ? 1 : 0); }
template <int kBN, bool kDeep>
constexpr int pair_smem_bytes() { return pair_stages<kBN, kDeep>() * pair_stage_bytes<kBN>() + pair_staging_bytes<kDeep>() + 1024; }

// 32 fp32 accumulator columns (+ bias, activation) -> 4 swizzled 16-byte chunks of bf16 in the staging row.
__device__ __forceinline__ void stage_bf16_32(const uint32_t (&v)[32], const __nv_bfloat16 *bias, int mode, uint8_t *row_base,
                                              int chunk0, int rsw) {
  float f[32];
#pragma unroll
  for (int j = 0; j < 32; ++j) f[j] = __uint_as_float(v[j]);
  if (bias) {
    const uint4 *bp = reinterpret_cast<const uint4 *>(bias);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint4 b = bp[j];
      f[8 * j + 0] += bf16_lo(b.x); f[8 * j + 1] += bf16_hi(b.x);
      f[8 * j + 2] += bf16_lo(b.y); f[8 * j + 3] += bf16_hi(b.y);
      f[8 * j + 4] += bf16_lo(b.z); f[8 * j + 5] += bf16_hi(b.z);
      f[8 * j + 6] += bf16_lo(b.w); f[8 * j + 7] += bf16_hi(b.w);
    }
  }
  if (mode == GM_OUT_BF16_GELU) {
#pragma unroll
    for (int j = 0; j < 32; ++j) f[j] = gelu_erf_f(f[j]);
  } else if (mode == GM_OUT_BF16_RELU) {
#pragma unroll
    for (int j = 0; j < 32; ++j) f[j] = fmaxf(f[j], 0.0f);
  }
#pragma unroll
  for (int j = 0; j < 4; ++j)
    *reinterpret_cast<uint4 *>(row_base + (((chunk0 + j) ^ rsw) << 4)) =
        make_uint4(pack_bf16(f[8 * j], f[8 * j + 1]), pack_bf16(f[8 * j + 2], f[8 * j + 3]), pack_bf16(f[8 * j + 4], f[8 * j + 5]),
                   pack_bf16(f[8 * j + 6], f[8 * j + 7]));
}

// Work item `item` of the persistent loop -> (row tile, first chunk, chunk count).  Items [0, n_full) are whole tiles of
// kCH chunks; item n_full + 2 i + h is half h (one chunk) of whole tile n_full + i.
template <int kCH>
__device__ __forceinline__ void pair_decode(const PairGemmParams &p, int item, int n_ntiles, int n_full, int &m_pt, int &c0, int &nch) {
  int tile = item;
  int h = -1;
  if (kCH == 2 && item >= n_full) {
    const int t2 = item - n_full;
    tile = n_full + (t2 >> 1);
    h = t2 & 1;
  }
  m_pt = tile / n_ntiles;
  const int n_tile = tile - m_pt * n_ntiles;
  if (p.reverse) m_pt = p.n_ptiles - 1 - m_pt;
  c0 = n_tile * kCH + (h > 0 ? 1 : 0);
  nch = h >= 0 ? 1 : kCH;
}

// A whole 256-wide tile whose two chunks come from the same weight source: its LoRA expand runs as ONE N = 256 step per block.
template <int kBN>
__device__ __forceinline__ bool pair_expand_wide(const PairGemmParams &p, int c0, int nch) {
  if (kBN != 256 || nch != 2 || !p.expand_wide) return false;
  int s0, r0, s1, r1;
  pair_chunk_source(p, c0, s0, r0);
  pair_chunk_source(p, c0 + 1, s1, r1);
  return s0 == s1;
}

template <int kBN, bool kDeep>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kGemmThreads, 1) pair_gemm_kernel(const __grid_constant__ PairGemmParams p) {
  constexpr int kCH = kBN / kChunk;
  constexpr int kStages = pair_stages<kBN, kDeep>();
  constexpr int kBufs = kDeep ? 1 : 2;                    // staging buffers per epilogue warpgroup
  constexpr int kStageBytes = pair_stage_bytes<kBN>();
  constexpr int kBHalf = kBN / 2;                          // W rows per CTA per stage
  constexpr int kExpandBytes = kATileBytes + 64 * kBK * 2; // U half tile + 64 slab rows
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *staging = smem + kStages * kStageBytes;
  __shared__ __align__(8) uint64_t full_bar[kStages], empty_bar[kStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint32_t tmem_base_slot;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int nK = (p.K + kBK - 1) / kBK;
  const int n_ntiles = p.n_chunks / kCH;
  const int whole_tiles = p.n_ptiles * n_ntiles;
  const int n_full = (kCH == 2 && p.n_full >= 0) ? p.n_full : whole_tiles;
  const int u_n = p.n_sh == 3 ? 256 : 128;                   // accumulator columns of a shrink item (64 per target)
  const int tile0 = (int)cluster_id_x(), tile_step = (int)cluster_nctaid_x();

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(&full_bar[s], 2); mbar_init(&empty_bar[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull_bar[a], 1); mbar_init(&tempty_bar[a], 16); }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc_2sm(&tmem_base_slot, 512);
    tmem_relinquish_2sm();
  }
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_slot;
  griddep_launch();
  griddep_wait();
  const int n_u = p.n_sh > 0 ? *p.n_blk : 0;                // fused-shrink items come first in the work list
  const bool part = p.k_split > 0;                           // partial-output mode (k_split >= 1): item = tile * ksp + ks, whole tiles only, no shrink items
  const int ksp = part ? p.k_split : 1;
  const int total_tiles = part ? whole_tiles * ksp : n_u + n_full + 2 * (whole_tiles - n_full);

  if (warp == 0) {
    // ================================ TMA producer (both CTAs) ================================
    if (lane == 0) {
      tma_prefetch_desc(&p.amap);
      tma_prefetch_desc(&p.wmap[0]);
      int stage = 0; uint32_t phase = 0;
      bool u_ready = p.n_sh == 0;
      for (int tile = tile0; tile < total_tiles; tile += tile_step) {
        if (!part && tile < n_u) {
          // ---- fused-shrink item: block `tile` of the S1 table; B = the task's A-slab rows of each shrink target.
          // u_n = 256: CTA 0 loads targets 0, 1 and CTA 1 target 2; u_n = 128: CTA r loads target r.
          const int m0 = p.blk_tile[tile] * kPairRows + (int)rank * kBM;
          const int coff = p.task_coff[p.blk_task[tile]];
          const int tg_lo = u_n == 256 ? (int)rank * 2 : (int)rank;
          const int tg_hi = min(p.n_sh, u_n == 256 ? tg_lo + 2 : tg_lo + 1);
          const uint32_t tx = kATileBytes + (uint32_t)max(tg_hi - tg_lo, 0) * 64 * kBK * 2;
          for (int kb = 0; kb < nK; ++kb) {
            mbar_wait(&empty_bar[stage], phase ^ 1);
            uint8_t *sa = smem + stage * kStageBytes, *sb = sa + kATileBytes;
            const uint32_t fb = mapa_shared(smem_u32(&full_bar[stage]), 0);
            mbar_arrive_expect_tx_cluster(fb, tx);
            tma_load_2d_2sm(sa, &p.amap, fb, kb * kBK, m0);
            for (int g = tg_lo; g < tg_hi; ++g) tma_load_2d_2sm(sb + (g - tg_lo) * 64 * kBK * 2, &p.smap[g], fb, kb * kBK, coff);
            if (++stage == kStages) { stage = 0; phase ^= 1; }
          }
          continue;
        }
        int m_pt, c0, nch;
        const int ks = part ? tile % ksp : 0;
        pair_decode<kCH>(p, part ? tile / ksp : tile - n_u, n_ntiles, n_full, m_pt, c0, nch);
        const int kb0 = ks * p.kb_per_split, kb1 = part ? min(nK, kb0 + p.kb_per_split) : nK;
        const int m0 = m_pt * kPairRows + (int)rank * kBM;
        int bsrc, brow;
        const CUtensorMap *wm;
        uint32_t stage_tx = kStageBytes;
        if (kBN == 256 && nch == 2) {                 // whole tile: CTA r loads chunk r's 128 W rows
          pair_chunk_source(p, c0 + (int)rank, bsrc, brow);
          wm = &p.wmap[bsrc];
        } else {                                      // one chunk: CTA r loads 64 of its W rows
          pair_chunk_source(p, c0, bsrc, brow);
          brow += (int)rank * 64;
          wm = kBN == 256 ? &p.wmap_h[bsrc] : &p.wmap[bsrc];
          stage_tx = kATileBytes + 64 * kBK * 2;
        }
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t *sa = smem + stage * kStageBytes, *sb = sa + kATileBytes;
          const uint32_t fb = mapa_shared(smem_u32(&full_bar[stage]), 0);
          mbar_arrive_expect_tx_cluster(fb, stage_tx);
          tma_load_2d_2sm(sa, &p.amap, fb, kb * kBK, m0);
          tma_load_2d_2sm(sb, wm, fb, kb * kBK, brow);
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        if (p.has_lora && ks == 0) {
          const int b0 = p.tile_blk_off[m_pt], b1 = p.tile_blk_off[m_pt + 1];
          // Both chunks of a whole tile from the same source (q | k | v, o, up, down; not SwiGLU's gate / up pairs) read the
          // SAME U columns: one expand step then covers the tile (U loaded once, each CTA its chunk's 128 slab rows, N = 256).
          const bool wide = pair_expand_wide<kBN>(p, c0, nch);
          int rr_wide = 0;
          if (wide) { int sr; pair_chunk_source(p, c0 + (int)rank, sr, rr_wide); }
          for (int c = 0; c < (wide ? 1 : nch); ++c) {
            int s, r0;
            pair_chunk_source(p, c0 + c, s, r0);
            const int tg = p.lora_tgt[s];
            if (tg < 0) continue;
            for (int b = b0; b < b1; ++b) {
              const int t = p.blk_task[b];
              if (p.task_trpad[t * 7 + tg] == 0) continue;
              if (!u_ready) {                               // U is written by the fused-shrink items of all pairs: wait once
                const unsigned target = 16u * (unsigned)n_u * p.u_epoch;
                const long long t_wait0 = clock64();
                while (ld_acquire_gpu(p.u_flag) < target) {
                  // the shrink items are the FIRST items of every resident pair, so this wait is short; a bound of ~2 s
                  // of SM clocks turns a scheduling assumption that does not hold into an error instead of a hang
                  if (clock64() - t_wait0 > (1ll << 32)) { *p.err = 2u; break; }   // reported by the next call; no trap
                }
                fence_proxy_async_global();
                u_ready = true;
              }
              mbar_wait(&empty_bar[stage], phase ^ 1);
              uint8_t *sa = smem + stage * kStageBytes, *sb = sa + kATileBytes;
              const uint32_t fb = mapa_shared(smem_u32(&full_bar[stage]), 0);
              mbar_arrive_expect_tx_cluster(fb, wide ? kExpandBytes + 64 * kBK * 2 : kExpandBytes);
              tma_load_2d_2sm(sa, &p.umap, fb, p.uslot[s] * 64, b * kPairRows + (int)rank * kBM);
              if (wide) {
                tma_load_2d_2sm(sb, &p.lmap[s], fb, p.task_coff[t], rr_wide);
                tma_load_2d_2sm(sb + 64 * kBK * 2, &p.lmap[s], fb, p.task_coff[t], rr_wide + 64);
              } else {
                tma_load_2d_2sm(sb, &p.lmap[s], fb, p.task_coff[t], r0 + (int)rank * 64);
              }
              if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ================================ MMA issuer (leader CTA only) ================================
    if (rank == 0 && lane == 0) {
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t accphase = 0;
      constexpr uint32_t idesc_whole = make_idesc_bf16(kPairRows, kBN);
      constexpr uint32_t idesc_lora = make_idesc_bf16(kPairRows, kChunk);
      for (int tile = tile0; tile < total_tiles; tile += tile_step) {
        int m_pt = 0, c0 = 0, nch = 0;
        const bool u_item = !part && tile < n_u;
        const int ks = part ? tile % ksp : 0;
        if (!u_item) pair_decode<kCH>(p, part ? tile / ksp : tile - n_u, n_ntiles, n_full, m_pt, c0, nch);
        const int kb0 = ks * p.kb_per_split, kb1 = part ? min(nK, kb0 + p.kb_per_split) : nK;
        const uint32_t idesc_main = u_item ? (u_n == 256 ? make_idesc_bf16(kPairRows, 256) : idesc_lora) : (nch == kCH ? idesc_whole : idesc_lora);
        mbar_wait_cluster(&tempty_bar[acc], accphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * kAccStride;
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait_cluster(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * kStageBytes);
          const uint64_t adesc = make_smem_desc_sw128(sa), bdesc = make_smem_desc_sw128(sa + kATileBytes);
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k)
            umma_bf16_2sm(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc_main, ((kb - kb0) | k) != 0);
          umma_commit_2sm(&empty_bar[stage], 3);
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        if (p.has_lora && !u_item && ks == 0) {
          const int b0 = p.tile_blk_off[m_pt], b1 = p.tile_blk_off[m_pt + 1];
          const bool wide = pair_expand_wide<kBN>(p, c0, nch);
          for (int c = 0; c < (wide ? 1 : nch); ++c) {
            int s, r0;
            pair_chunk_source(p, c0 + c, s, r0);
            const int tg = p.lora_tgt[s];
            if (tg < 0) continue;
            for (int b = b0; b < b1; ++b) {
              const int ksteps = p.task_trpad[p.blk_task[b] * 7 + tg] >> 4;
              if (ksteps == 0) continue;
              mbar_wait_cluster(&full_bar[stage], phase);
              tc_fence_after();
              const uint32_t sa = smem_u32(smem + stage * kStageBytes);
              const uint64_t adesc = make_smem_desc_sw128(sa), bdesc = make_smem_desc_sw128(sa + kATileBytes);
              for (int k = 0; k < ksteps; ++k)
                umma_bf16_2sm(d_tmem + c * kChunk, adesc + 2 * k, bdesc + 2 * k, wide ? idesc_whole : idesc_lora, 1);
              umma_commit_2sm(&empty_bar[stage], 3);
              if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
          }
        }
        umma_commit_2sm(&tfull_bar[acc], 3);
        if (++acc == 2) { acc = 0; accphase ^= 1; }
      }
    }
  } else if (warp >= 4) {
    // ================================ epilogue (both CTAs) ================================
    const int wg = (warp - 4) >> 2, quad = warp & 3;
    const int r_in_tile = quad * 32 + lane;
    const int rsw = r_in_tile & 7;
    const bool issuer = (threadIdx.x == 128 + wg * 128);
    const uint32_t bar_id = 1 + wg;
    uint8_t *stg = staging + wg * (kBufs * 16384);
    int box_seq = 0;
    int acc = 0; uint32_t accphase = 0;
    const int mode = part ? (int)GM_OUT_F32 : p.mode;          // partial mode: every item stores its raw fp32 partial
    for (int tile = tile0; tile < total_tiles; tile += tile_step) {
      if (!part && tile < n_u) {
        // ---- fused-shrink item: U_blk[row, slot*64 + j] = bf16(s_t · acc), rows outside the block's task zeroed ----
        const int b = tile, t = p.blk_task[b];
        const int rp = (int)rank * kBM + r_in_tile;             // row within the 256-row tile
        const bool in_seg = rp >= p.blk_lo[b] && rp < p.blk_hi[b];
        __nv_bfloat16 *Urow = p.U + (size_t)(b * kPairRows + rp) * 192;
        mbar_wait(&tfull_bar[acc], accphase);
        tc_fence_after();
        const uint32_t t_row = tmem_base + (uint32_t(quad * 32) << 16) + acc * kAccStride;
        uint32_t v[32];
        const int n_grp = p.n_sh * 2;                           // 32-column groups, split over the two warpgroups
        for (int g = wg; g < n_grp; g += 2) {
          __syncwarp();
          tmem_ld_32x32(t_row + g * 32, v);
          tmem_ld_wait();
          const float sc = in_seg ? p.task_scale[t * 7 + p.sh_tg[g >> 1]] : 0.0f;
          uint4 *dst = reinterpret_cast<uint4 *>(Urow + g * 32);
#pragma unroll
          for (int j = 0; j < 4; ++j)
            dst[j] = make_uint4(pack_bf16(sc * __uint_as_float(v[8 * j + 0]), sc * __uint_as_float(v[8 * j + 1])),
                                pack_bf16(sc * __uint_as_float(v[8 * j + 2]), sc * __uint_as_float(v[8 * j + 3])),
                                pack_bf16(sc * __uint_as_float(v[8 * j + 4]), sc * __uint_as_float(v[8 * j + 5])),
                                pack_bf16(sc * __uint_as_float(v[8 * j + 6]), sc * __uint_as_float(v[8 * j + 7])));
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive_cluster(mapa_shared(smem_u32(&tempty_bar[acc]), 0));
          red_release_gpu_add(p.u_flag, 1u);                    // 16 arrivals (8 epilogue warps x 2 CTAs) per block
        }
        if (++acc == 2) { acc = 0; accphase ^= 1; }
        continue;
      }
      int m_pt, c0, nch;
      const int ks = part ? tile % ksp : 0;
      pair_decode<kCH>(p, part ? tile / ksp : tile - n_u, n_ntiles, n_full, m_pt, c0, nch);
      const int bn = nch * kChunk;                              // columns of this work item (a half tile has 128)
      const int row0_cta = m_pt * kPairRows + (int)rank * kBM;
      const int row = row0_cta + r_in_tile;
      mbar_wait(&tfull_bar[acc], accphase);
      tc_fence_after();
      const uint32_t t_row = tmem_base + (uint32_t(quad * 32) << 16) + acc * kAccStride;
      const uint32_t tempty_remote = mapa_shared(smem_u32(&tempty_bar[acc]), 0);
      uint32_t v[32], u[32];

      if (mode == GM_OUT_BF16_SWIGLU) {
        // tile = [gate chunk | up chunk] of the same 128 output features; this warpgroup: 64 of them
        const int r0 = (c0 >> 1) * kChunk;                      // feature offset of the tile (never a half tile)
        const int fcol = wg * 64;
        uint8_t *buf = stg + (box_seq & (kBufs - 1)) * 16384;
        if (issuer) bulk_wait_read<kBufs - 1>();
        named_bar_sync(bar_id, 128);
        uint8_t *row_base = buf + r_in_tile * 128;
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
          tmem_ld_32x32(t_row + fcol + h * 32, v);
          tmem_ld_32x32(t_row + kChunk + fcol + h * 32, u);
          tmem_ld_wait();
          if (h == 1) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tempty_remote);
          }
          const __nv_bfloat16 *bg = p.bias[0], *bu = p.bias[1];
          const int nb = r0 + fcol + h * 32;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            float r[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
              float gt = __uint_as_float(v[8 * j + e]), up = __uint_as_float(u[8 * j + e]);
              if (bg) gt += __bfloat162float(bg[nb + 8 * j + e]);
              if (bu) up += __bfloat162float(bu[nb + 8 * j + e]);
              r[e] = silu_f(gt) * up;
            }
            *reinterpret_cast<uint4 *>(row_base + (((h * 4 + j) ^ rsw) << 4)) =
                make_uint4(pack_bf16(r[0], r[1]), pack_bf16(r[2], r[3]), pack_bf16(r[4], r[5]), pack_bf16(r[6], r[7]));
          }
        }
        fence_proxy_async();
        named_bar_sync(bar_id, 128);
        if (issuer) { tma_store_2d(&p.omap, buf, r0 + fcol, row0_cta); bulk_commit(); }
        ++box_seq;
      } else if (mode == GM_OUT_BF16 || mode == GM_OUT_BF16_GELU || mode == GM_OUT_BF16_RELU) {
        const int kBoxes = bn / 128;                            // 64-column boxes per warpgroup
        int s_wg, r0_wg;
        pair_chunk_source(p, c0 + (bn == 256 ? wg : 0), s_wg, r0_wg);
        if (!kDeep && p.rope_cs && bn == 256 && ((p.rope_src_mask >> s_wg) & 1)) {   // needs both staging buffers
          // Fused RoPE (rotate-half): this warpgroup's 128 columns are one head; dims j and j + 64 of the thread's row
          // are rotated in fp32 straight from the accumulator (one rounding) and leave as two 64-column boxes.
          const int n_out = (c0 + wg) * kChunk;
          uint8_t *rowA = stg + r_in_tile * 128, *rowB = rowA + 16384;
          if (issuer) bulk_wait_read<0>();
          named_bar_sync(bar_id, 128);
          const float2 *cs = p.rope_cs + (row < p.M ? p.row_pos[row] : 0);          // + j * rope_ld for pair index j
          const __nv_bfloat16 *bias = p.bias[s_wg];
#pragma unroll 1
          for (int h = 0; h < 2; ++h) {
            tmem_ld_32x32(t_row + wg * kChunk + h * 32, v);
            tmem_ld_32x32(t_row + wg * kChunk + 64 + h * 32, u);
            tmem_ld_wait();
            if (h == 1) {
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(tempty_remote);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              float x1[8], x2[8];
#pragma unroll
              for (int e = 0; e < 8; ++e) {
                x1[e] = __uint_as_float(v[8 * q + e]);
                x2[e] = __uint_as_float(u[8 * q + e]);
                if (bias) {
                  x1[e] += __bfloat162float(bias[r0_wg + h * 32 + 8 * q + e]);
                  x2[e] += __bfloat162float(bias[r0_wg + 64 + h * 32 + 8 * q + e]);
                }
              }
              uint32_t oa[4], ob[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                // (cos, sin) of dims 2e, 2e+1 of this group: consecutive rows read consecutive addresses
                const float2 ca = __ldg(cs + (size_t)(h * 32 + q * 8 + 2 * e) * p.rope_ld);
                const float2 cb = __ldg(cs + (size_t)(h * 32 + q * 8 + 2 * e + 1) * p.rope_ld);
                oa[e] = pack_bf16(x1[2 * e] * ca.x - x2[2 * e] * ca.y, x1[2 * e + 1] * cb.x - x2[2 * e + 1] * cb.y);
                ob[e] = pack_bf16(x2[2 * e] * ca.x + x1[2 * e] * ca.y, x2[2 * e + 1] * cb.x + x1[2 * e + 1] * cb.y);
              }
              *reinterpret_cast<uint4 *>(rowA + (((h * 4 + q) ^ rsw) << 4)) = make_uint4(oa[0], oa[1], oa[2], oa[3]);
              *reinterpret_cast<uint4 *>(rowB + (((h * 4 + q) ^ rsw) << 4)) = make_uint4(ob[0], ob[1], ob[2], ob[3]);
            }
          }
          fence_proxy_async();
          named_bar_sync(bar_id, 128);
          if (issuer) {
            tma_store_2d(&p.omap, stg, n_out, row0_cta); bulk_commit();
            tma_store_2d(&p.omap, stg + 16384, n_out + 64, row0_cta); bulk_commit();
          }
          box_seq = 0;                                          // the next box reuses the first buffer, after group 1
        } else
#pragma unroll 1
        for (int j = 0; j < kBoxes; ++j) {
          const int col = wg * (bn / 2) + j * 64;               // column within the tile
          int s, r0;
          pair_chunk_source(p, c0 + col / kChunk, s, r0);
          const int n_src = r0 + (col % kChunk);
          const int n_out = c0 * kChunk + col;
          uint8_t *buf = stg + (box_seq & (kBufs - 1)) * 16384;
          if (issuer) bulk_wait_read<kBufs - 1>();
          named_bar_sync(bar_id, 128);
          tmem_ld_32x32(t_row + col, v);
          tmem_ld_32x32(t_row + col + 32, u);
          tmem_ld_wait();
          if (j == kBoxes - 1) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tempty_remote);
          }
          uint8_t *row_base = buf + r_in_tile * 128;
          const __nv_bfloat16 *bias = p.bias[s];
          stage_bf16_32(v, bias ? bias + n_src : nullptr, mode, row_base, 0, rsw);
          stage_bf16_32(u, bias ? bias + n_src + 32 : nullptr, mode, row_base, 4, rsw);
          fence_proxy_async();
          named_bar_sync(bar_id, 128);
          if (issuer) { tma_store_2d(&p.omap, buf, n_out, row0_cta); bulk_commit(); }
          ++box_seq;
        }
      } else {
        // fp32 outputs: residual reduce-add, embed (+ positional table), plain store
        const int kBoxes = bn / 64;                             // 32-column boxes per warpgroup
        const float *posrow = nullptr;
        if (mode == GM_EMBED_F32 && row < p.M) posrow = p.posb + (size_t)p.row_pos[row] * p.ld_pos;
#pragma unroll 1
        for (int j = 0; j < kBoxes; ++j) {
          const int col = wg * (bn / 2) + j * 32;
          int s, r0;
          pair_chunk_source(p, c0 + col / kChunk, s, r0);
          const int n_src = r0 + (col % kChunk);
          const int n_out = c0 * kChunk + col;
          uint8_t *buf = stg + (box_seq & (kBufs - 1)) * 16384;
          if (issuer) bulk_wait_read<kBufs - 1>();
          named_bar_sync(bar_id, 128);
          tmem_ld_32x32(t_row + col, v);
          tmem_ld_wait();
          if (j == kBoxes - 1) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tempty_remote);
          }
          float f[32];
#pragma unroll
          for (int e = 0; e < 32; ++e) f[e] = __uint_as_float(v[e]);
          const __nv_bfloat16 *bias = part ? nullptr : p.bias[s];        // partial mode: the reduce kernel adds the bias once
          if (bias) {
            const uint4 *bp = reinterpret_cast<const uint4 *>(bias + n_src);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const uint4 b = bp[q];
              f[8 * q + 0] += bf16_lo(b.x); f[8 * q + 1] += bf16_hi(b.x);
              f[8 * q + 2] += bf16_lo(b.y); f[8 * q + 3] += bf16_hi(b.y);
              f[8 * q + 4] += bf16_lo(b.z); f[8 * q + 5] += bf16_hi(b.z);
              f[8 * q + 6] += bf16_lo(b.w); f[8 * q + 7] += bf16_hi(b.w);
            }
          }
          if (posrow) {
            const float4 *P = reinterpret_cast<const float4 *>(posrow + n_out);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              const float4 w = P[q];
              f[4 * q] += w.x; f[4 * q + 1] += w.y; f[4 * q + 2] += w.z; f[4 * q + 3] += w.w;
            }
          }
          uint8_t *row_base = buf + r_in_tile * 128;
#pragma unroll
          for (int q = 0; q < 8; ++q)
            *reinterpret_cast<float4 *>(row_base + ((q ^ rsw) << 4)) = make_float4(f[4 * q], f[4 * q + 1], f[4 * q + 2], f[4 * q + 3]);
          fence_proxy_async();
          named_bar_sync(bar_id, 128);
          if (issuer) {
            if (part) tma_store_2d(&p.pmap, buf, n_out, ks * p.split_rows + row0_cta);
            else if (mode == GM_RESID_F32) tma_reduce_add_2d(&p.omap, buf, n_out, row0_cta);
            else tma_store_2d(&p.omap, buf, n_out, row0_cta);
            bulk_commit();
          }
          ++box_seq;
        }
      }
      if (++acc == 2) { acc = 0; accphase ^= 1; }
    }
    if (issuer) bulk_wait<0>();
  }

  tc_fence_before();
  cluster_sync_all();
  if (warp == 2) tmem_dealloc_2sm(tmem_base, 512);
}

}  // namespace fmx
