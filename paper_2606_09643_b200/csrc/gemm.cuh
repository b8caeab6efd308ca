// tcgen05 / TMEM / TMA GEMM for the backbone projections with the per-task LoRA expand fused
// in as extra K-steps, plus the segmented LoRA shrink as a variant of the same pipeline.
//
//   C[M, N] = A[M, K] · W[N, K]^T  (+ Σ_blocks  U_blk[128, r_pad] · B_task[N, r_pad]^T)   fp32 in TMEM
//
// Rows are task-sorted token rows (S1).  The N axis is cut into 128-column CHUNKS; a chunk
// names its weight source (q | k | v, gate | up, or the single matrix), so fused QKV and
// SwiGLU gate/up need no repacked weights.  One CTA tile is 128 rows x kBN columns
// (kBN = 128 or 256 = 1 or 2 chunks); BLOCK_K = 64 bf16 = one 128-byte swizzle row.
//
// LoRA expand (S3c/e/f/g; BASELINE.json north_star item 4): after the main K loop the MMA
// warp issues, for every (row-tile, task) BLOCK of the tile, r_pad/16 more K-steps with
// A = the block's masked shrink output U (rows of other tasks are zero) and B = that task's
// B-slab columns, into the SAME TMEM accumulator — the delta lands before the epilogue, which
// is the only correct place for pre-activation targets (gate/up).  No segment padding: a tile
// may span any number of tasks.
//
// Warp roles (384 threads, persistent over tiles, 1 CTA/SM):
//   warp 0   TMA producer        (lane 0)        smem ring: full/empty mbarriers
//   warp 1   tcgen05.mma issuer  (lane 0)        TMEM accumulators double-buffered
//   warp 2   TMEM alloc/dealloc
//   warp 3   idle
//   warps 4-11  epilogue: two warpgroups, each thread owns one accumulator row (TMEM lane);
//               tcgen05.ld 32 columns at a time -> bias / activation / SwiGLU / residual / store
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

namespace fmx {

enum GemmMode : int {
  GM_OUT_BF16 = 0,     // out_bf16 = acc + bias
  GM_OUT_BF16_GELU,    // out_bf16 = gelu_erf(acc + bias)
  GM_OUT_BF16_RELU,    // out_bf16 = relu(acc + bias)
  GM_OUT_BF16_SWIGLU,  // out_bf16[:, j] = silu(acc_gate + b_g) * (acc_up + b_u); chunks interleaved gate/up
  GM_RESID_F32,        // X_f32 += acc + bias   (in place, fp32 residual stream)
  GM_EMBED_F32,        // X_f32 = acc + posb[row_pos[row]]   (patch embed)
  GM_OUT_F32,          // C_f32 = acc            (debug / tests)
  GM_SHRINK            // U_blk = bf16(scale_task * acc), rows outside the block's task zeroed
};

constexpr int kBM = 128;
constexpr int kBK = 64;
constexpr int kChunk = 128;
constexpr int kGemmThreads = 384;
constexpr int kATileBytes = kBM * kBK * 2;        // 16 KB
constexpr int kChunkBytes = kChunk * kBK * 2;     // 16 KB
constexpr int kAccStride = 256;                   // TMEM columns per accumulator stage

struct GemmParams {
  CUtensorMap amap;        // A [M, K] bf16, box {64, 128}
  CUtensorMap wmap[3];     // weight sources [rows_s, K] bf16, box {64, 128}; shrink: A-slabs [Rcap, K], box {64, 64}
  CUtensorMap umap;        // U_exp [n_blk_cap*128, n_slots*64] bf16, box {64, 128}
  CUtensorMap lmap[3];     // B-slabs [d_out_s, Rcap] bf16, box {64, 128}
  int M, K;
  int n_chunks;            // N / 128 (shrink: unused)
  int n_mtiles;            // ceil(M / 128)
  int mode;
  int interleave2;         // chunk c -> source c&1, row (c>>1)*128  (SwiGLU)
  int has_lora;            // any lora_tgt >= 0
  int src_end[3];          // cumulative chunk count per source (non-interleaved)
  int lora_tgt[3];         // target id of source s, or -1 = no LoRA on it
  int uslot[3];            // U column block (x64) of source s
  const __nv_bfloat16 *bias[3];
  void *out;
  int ld_out;              // elements
  // S1 tables
  const int *tile_blk_off, *blk_task, *blk_lo, *blk_hi, *blk_tile, *n_blk;
  const int *task_coff;            // [T] first slab column of the task
  const unsigned char *task_trpad; // [T*7] padded rank of (task, target), 0 = no adapter
  const float *task_scale;         // [T*7] alpha/r
  // embed
  const float *posb;               // [max_seq, d] fp32: bias/cls + positional term
  const int *row_pos;              // [M] position of the row within its request
  // shrink
  int n_tg;                        // targets in the input group (1..3)
  int tg_ids[3];
};

__device__ __forceinline__ void chunk_source(const GemmParams &p, int c, int &s, int &r0) {
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

__device__ __forceinline__ float gelu_erf_f(float x) { return 0.5f * x * (1.0f + erff(x * 0.70710678118654752440f)); }
__device__ __forceinline__ float silu_f(float x) { return x / (1.0f + __expf(-x)); }

template <int kBN, int kStages, bool kShrink>
__global__ void __launch_bounds__(kGemmThreads, 1) gemm_kernel(const __grid_constant__ GemmParams p) {
  constexpr int kCH = kBN / kChunk;                       // chunks per tile (GEMM modes)
  constexpr int kBStageBytes = kShrink ? 3 * 64 * kBK * 2 : kBN * kBK * 2;
  constexpr int kStageBytes = kATileBytes + kBStageBytes;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ __align__(8) uint64_t full_bar[kStages], empty_bar[kStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint32_t tmem_base_slot;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nK = (p.K + kBK - 1) / kBK;
  int total_tiles, n_ntiles = 1;
  if constexpr (kShrink) {
    total_tiles = *p.n_blk;
  } else {
    n_ntiles = p.n_chunks / kCH;
    total_tiles = p.n_mtiles * n_ntiles;
  }

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull_bar[a], 1); mbar_init(&tempty_bar[a], 256); }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(&tmem_base_slot, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_slot;

  if (warp == 0) {
    // ================================ TMA producer ================================
    if (lane == 0) {
      tma_prefetch_desc(&p.amap);
      tma_prefetch_desc(&p.wmap[0]);
      int stage = 0; uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        int m_tile, n_tile = 0, coff = 0;
        if constexpr (kShrink) { m_tile = p.blk_tile[tile]; coff = p.task_coff[p.blk_task[tile]]; }
        else { m_tile = tile / n_ntiles; n_tile = tile - m_tile * n_ntiles; }
        const int m0 = m_tile * kBM;
        int src[kCH], row0[kCH];
        if constexpr (!kShrink) {
#pragma unroll
          for (int c = 0; c < kCH; ++c) chunk_source(p, n_tile * kCH + c, src[c], row0[c]);
        }
        for (int kb = 0; kb < nK; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t *sa = smem + stage * kStageBytes, *sb = sa + kATileBytes;
          if constexpr (kShrink) {
            mbar_arrive_expect_tx(&full_bar[stage], kATileBytes + p.n_tg * 64 * kBK * 2);
            tma_load_2d(sa, &p.amap, &full_bar[stage], kb * kBK, m0);
            for (int j = 0; j < p.n_tg; ++j)
              tma_load_2d(sb + j * 64 * kBK * 2, &p.wmap[j], &full_bar[stage], kb * kBK, coff);
          } else {
            mbar_arrive_expect_tx(&full_bar[stage], kStageBytes);
            tma_load_2d(sa, &p.amap, &full_bar[stage], kb * kBK, m0);
#pragma unroll
            for (int c = 0; c < kCH; ++c)
              tma_load_2d(sb + c * kChunkBytes, &p.wmap[src[c]], &full_bar[stage], kb * kBK, row0[c]);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        if (!kShrink && p.has_lora) {
          // ---- LoRA expand stages: one per (chunk, block) that has an adapter ----
          const int b0 = p.tile_blk_off[m_tile], b1 = p.tile_blk_off[m_tile + 1];
#pragma unroll
          for (int c = 0; c < kCH; ++c) {
            const int tg = p.lora_tgt[src[c]];
            if (tg < 0) continue;
            for (int b = b0; b < b1; ++b) {
              const int t = p.blk_task[b];
              if (p.task_trpad[t * 7 + tg] == 0) continue;
              mbar_wait(&empty_bar[stage], phase ^ 1);
              uint8_t *sa = smem + stage * kStageBytes, *sb = sa + kATileBytes;
              mbar_arrive_expect_tx(&full_bar[stage], kATileBytes + kChunkBytes);
              tma_load_2d(sa, &p.umap, &full_bar[stage], p.uslot[src[c]] * 64, b * kBM);
              tma_load_2d(sb, &p.lmap[src[c]], &full_bar[stage], p.task_coff[t], row0[c]);
              if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ================================ MMA issuer ================================
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t accphase = 0;
      const uint32_t idesc_main = kShrink ? make_idesc_bf16(kBM, (uint32_t)p.n_tg * 64) : make_idesc_bf16(kBM, kBN);
      const uint32_t idesc_lora = make_idesc_bf16(kBM, kChunk);
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        int m_tile, n_tile = 0;
        if constexpr (kShrink) m_tile = p.blk_tile[tile];
        else { m_tile = tile / n_ntiles; n_tile = tile - m_tile * n_ntiles; }
        mbar_wait(&tempty_bar[acc], accphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * kAccStride;
        for (int kb = 0; kb < nK; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * kStageBytes);
          const uint64_t adesc = make_smem_desc_sw128(sa), bdesc = make_smem_desc_sw128(sa + kATileBytes);
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k)
            umma_bf16(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc_main, (kb | k) != 0);
          umma_commit(&empty_bar[stage]);
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        if (!kShrink && p.has_lora) {
          const int b0 = p.tile_blk_off[m_tile], b1 = p.tile_blk_off[m_tile + 1];
#pragma unroll
          for (int c = 0; c < kCH; ++c) {
            int s, r0;
            chunk_source(p, n_tile * kCH + c, s, r0);
            const int tg = p.lora_tgt[s];
            if (tg < 0) continue;
            for (int b = b0; b < b1; ++b) {
              const int ksteps = p.task_trpad[p.blk_task[b] * 7 + tg] >> 4;
              if (ksteps == 0) continue;
              mbar_wait(&full_bar[stage], phase);
              tc_fence_after();
              const uint32_t sa = smem_u32(smem + stage * kStageBytes);
              const uint64_t adesc = make_smem_desc_sw128(sa), bdesc = make_smem_desc_sw128(sa + kATileBytes);
              for (int k = 0; k < ksteps; ++k)
                umma_bf16(d_tmem + c * kChunk, adesc + 2 * k, bdesc + 2 * k, idesc_lora, 1);
              umma_commit(&empty_bar[stage]);
              if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
          }
        }
        umma_commit(&tfull_bar[acc]);
        if (++acc == 2) { acc = 0; accphase ^= 1; }
      }
    }
  } else if (warp >= 4) {
    // ================================ epilogue ================================
    const int wg = (warp - 4) >> 2, quad = warp & 3;
    const int r_in_tile = quad * 32 + lane;
    int acc = 0; uint32_t accphase = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      int m_tile, n_tile = 0;
      if constexpr (kShrink) m_tile = p.blk_tile[tile];
      else { m_tile = tile / n_ntiles; n_tile = tile - m_tile * n_ntiles; }
      const int row = m_tile * kBM + r_in_tile;
      const bool row_ok = row < p.M;
      mbar_wait(&tfull_bar[acc], accphase);
      tc_fence_after();
      const uint32_t t_row = tmem_base + (uint32_t(quad * 32) << 16) + acc * kAccStride;
      uint32_t v[32];

      if constexpr (kShrink) {
        const int t = p.blk_task[tile];
        const bool in_seg = r_in_tile >= p.blk_lo[tile] && r_in_tile < p.blk_hi[tile];
        __nv_bfloat16 *U = reinterpret_cast<__nv_bfloat16 *>(p.out) + (size_t)(tile * kBM + r_in_tile) * p.ld_out;
        for (int g = wg; g < p.n_tg * 2; g += 2) {           // 32-column groups, split over the 2 warpgroups
          __syncwarp();
          tmem_ld_32x32(t_row + g * 32, v);
          tmem_ld_wait();
          const float sc = in_seg ? p.task_scale[t * 7 + p.tg_ids[g >> 1]] : 0.0f;
          uint4 *dst = reinterpret_cast<uint4 *>(U + g * 32);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 o;
            o.x = pack_bf16(sc * __uint_as_float(v[8 * j + 0]), sc * __uint_as_float(v[8 * j + 1]));
            o.y = pack_bf16(sc * __uint_as_float(v[8 * j + 2]), sc * __uint_as_float(v[8 * j + 3]));
            o.z = pack_bf16(sc * __uint_as_float(v[8 * j + 4]), sc * __uint_as_float(v[8 * j + 5]));
            o.w = pack_bf16(sc * __uint_as_float(v[8 * j + 6]), sc * __uint_as_float(v[8 * j + 7]));
            dst[j] = o;
          }
        }
      } else if (p.mode == GM_OUT_BF16_SWIGLU) {
        // tile = [gate chunk | up chunk] of the same 128 output features
        int s, r0;
        chunk_source(p, n_tile * 2, s, r0);
        const __nv_bfloat16 *bg = p.bias[0], *bu = p.bias[1];
        __nv_bfloat16 *O = reinterpret_cast<__nv_bfloat16 *>(p.out) + (size_t)row * p.ld_out + r0;
        uint32_t u[32];
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
          const int col = wg * 64 + g * 32;
          __syncwarp();
          tmem_ld_32x32(t_row + col, v);
          tmem_ld_32x32(t_row + kChunk + col, u);
          tmem_ld_wait();
          if (row_ok) {
            uint4 *dst = reinterpret_cast<uint4 *>(O + col);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              float r[8];
#pragma unroll
              for (int e = 0; e < 8; ++e) {
                float gt = __uint_as_float(v[8 * j + e]), up = __uint_as_float(u[8 * j + e]);
                if (bg) gt += __bfloat162float(bg[r0 + col + 8 * j + e]);
                if (bu) up += __bfloat162float(bu[r0 + col + 8 * j + e]);
                r[e] = silu_f(gt) * up;
              }
              dst[j] = make_uint4(pack_bf16(r[0], r[1]), pack_bf16(r[2], r[3]), pack_bf16(r[4], r[5]), pack_bf16(r[6], r[7]));
            }
          }
        }
      } else {
        constexpr int kColsPerWg = kBN / 2;
#pragma unroll 1
        for (int g = 0; g < kColsPerWg / 32; ++g) {
          const int col = wg * kColsPerWg + g * 32;          // column within the tile
          __syncwarp();
          tmem_ld_32x32(t_row + col, v);
          tmem_ld_wait();
          if (row_ok) {
          int s, r0;
          chunk_source(p, n_tile * kCH + col / kChunk, s, r0);
          const int n_src = r0 + (col % kChunk);             // column within the source matrix
          const int n_out = (n_tile * kCH) * kChunk + col;   // column within the output
          float f[32];
          const __nv_bfloat16 *bias = p.bias[s];
#pragma unroll
          for (int j = 0; j < 32; ++j) f[j] = __uint_as_float(v[j]);
          if (bias) {
            const uint4 *bp = reinterpret_cast<const uint4 *>(bias + n_src);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const uint4 b = bp[j];
              f[8 * j + 0] += bf16_lo(b.x); f[8 * j + 1] += bf16_hi(b.x);
              f[8 * j + 2] += bf16_lo(b.y); f[8 * j + 3] += bf16_hi(b.y);
              f[8 * j + 4] += bf16_lo(b.z); f[8 * j + 5] += bf16_hi(b.z);
              f[8 * j + 6] += bf16_lo(b.w); f[8 * j + 7] += bf16_hi(b.w);
            }
          }
          if (p.mode == GM_RESID_F32 || p.mode == GM_EMBED_F32 || p.mode == GM_OUT_F32) {
            float4 *X = reinterpret_cast<float4 *>(reinterpret_cast<float *>(p.out) + (size_t)row * p.ld_out + n_out);
            if (p.mode == GM_RESID_F32) {
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                float4 x = X[j];
                x.x += f[4 * j]; x.y += f[4 * j + 1]; x.z += f[4 * j + 2]; x.w += f[4 * j + 3];
                X[j] = x;
              }
            } else if (p.mode == GM_EMBED_F32) {
              const float4 *P = reinterpret_cast<const float4 *>(p.posb + (size_t)p.row_pos[row] * p.ld_out + n_out);
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                const float4 q = P[j];
                X[j] = make_float4(f[4 * j] + q.x, f[4 * j + 1] + q.y, f[4 * j + 2] + q.z, f[4 * j + 3] + q.w);
              }
            } else {
#pragma unroll
              for (int j = 0; j < 8; ++j) X[j] = make_float4(f[4 * j], f[4 * j + 1], f[4 * j + 2], f[4 * j + 3]);
            }
          } else {
            if (p.mode == GM_OUT_BF16_GELU) {
#pragma unroll
              for (int j = 0; j < 32; ++j) f[j] = gelu_erf_f(f[j]);
            } else if (p.mode == GM_OUT_BF16_RELU) {
#pragma unroll
              for (int j = 0; j < 32; ++j) f[j] = fmaxf(f[j], 0.0f);
            }
            uint4 *dst = reinterpret_cast<uint4 *>(reinterpret_cast<__nv_bfloat16 *>(p.out) + (size_t)row * p.ld_out + n_out);
#pragma unroll
            for (int j = 0; j < 4; ++j)
              dst[j] = make_uint4(pack_bf16(f[8 * j], f[8 * j + 1]), pack_bf16(f[8 * j + 2], f[8 * j + 3]),
                                  pack_bf16(f[8 * j + 4], f[8 * j + 5]), pack_bf16(f[8 * j + 6], f[8 * j + 7]));
          }
          }  // row_ok
        }
      }
      __syncwarp();
      tc_fence_before();
      mbar_arrive(&tempty_bar[acc]);
      if (++acc == 2) { acc = 0; accphase ^= 1; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}

template <int kBN, bool kShrink>
constexpr int gemm_stages() { return kShrink ? 4 : (kBN == 256 ? 4 : 6); }
template <int kBN, bool kShrink>
constexpr int gemm_smem_bytes() {
  return gemm_stages<kBN, kShrink>() * (kATileBytes + (kShrink ? 3 * 64 * kBK * 2 : kBN * kBK * 2)) + 1024;
}

}  // namespace fmx
