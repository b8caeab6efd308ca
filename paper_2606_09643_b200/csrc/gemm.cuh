// Common definitions of the tcgen05 GEMM family (modes, tile constants, activations) and the
// single-CTA segmented LoRA shrink kernel (S3b).  The backbone projections live in pair_gemm.cuh.
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
  int reverse;                     // 1: units are walked from the last block to the first
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

// GeLU(x) = x * Phi(x), Phi(x) = 0.5 erfc(-x / sqrt 2), with erfc(z) = 2^(-z Q(z)) for z >= 0, Q a quartic fitted (minimax
// on |erf error|, fp32 evaluation) to -log2(erfc z) / z on [0, 4.2]: |error| <= 6.7e-7 in erf, |error| <= 1.4e-6 in GeLU over
// [-12, 12], far below the bf16 rounding of the output; beyond the fit range the quartic keeps growing, so erfc -> 0.  The
// 1/sqrt(2) is folded into the coefficients (in |x|).  One MUFU op (ex2) and 4 FMAs per element: the GeLU epilogue of the FFN-in GEMM was issue-bound with
// erff (~30 instructions) and still the slower side with the Abramowitz-Stegun 7.1.26 form (rcp + ex2 + 10 FMA-pipe ops).
__device__ __forceinline__ float gelu_erf_f(float x) {
  const float ax = fabsf(x);
  float p = fmaf(-0.00052327975f, ax, 0.0074127913f);
  p = fmaf(p, ax, -0.0525887412f);
  p = fmaf(p, ax, -0.459236082f);
  p = fmaf(p, ax, -1.15109488f);
  float e;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(p * ax));
  // x Phi(x) = x (1 - E / 2) for x >= 0 and x E / 2 for x < 0, i.e. max(x, 0) - |x| E / 2 on both sides: three operations instead of
  // the five of scale / subtract / compare / select / multiply (the FFN-in epilogue of the GeLU backbones is issue-bound)
  return fmaf(ax * e, -0.5f, fmaxf(x, 0.0f));
}
// silu(x) = x / (1 + e^-x) with ex2.approx and rcp.approx (2 MUFU ops, 3 FMA-pipe ops; an IEEE division is ~10 more).
// Very negative finite x: e^-x overflows to +inf, rcp gives 0, the product is -0 (the limit); relative error ~2^-22, far below
// the bf16 rounding of the output.
__device__ __forceinline__ float silu_f(float x) {
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(x * -1.4426950408889634f));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + e));
  return x * r;
}

// ---------------------------------------------------------------------------------------------
// Segmented LoRA shrink (S3b):  U_blk[row, slot*64 + j] = bf16(s_t · Σ_k x[row, k] · A_{t,P}[j, k])
// One unit = one 128-row HALF of a (256-row tile, task) block of the S1 table; rows of the half that
// belong to other tasks are written as zeros (the expand MMA then adds nothing for them).  Up to three
// targets that read the same input share one pass (N = 64 columns per target).  Single-CTA tcgen05:
// M = 128, N = n_tg * 64, TMEM accumulator double-buffered; halves with no row of the task skip the
// loads and MMAs and only write zeros.
// kTgCap: targets the stage has room for (1..3); the shared-memory ring is as deep as ~200 KB allow for that stage size,
// because the kernel is bound by bytes in flight per SM: 8 / 6 / 5 stages for 1 / 2 / 3 targets.
template <int kStages, int kTgCap>
__global__ void __launch_bounds__(kGemmThreads, 1) shrink_kernel(const __grid_constant__ GemmParams p) {
  constexpr int kBStageBytes = kTgCap * 64 * kBK * 2;
  constexpr int kStageBytes = kATileBytes + kBStageBytes;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ __align__(8) uint64_t full_bar[kStages], empty_bar[kStages], tfull_bar[2], tempty_bar[2];
  __shared__ uint32_t tmem_base_slot;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nK = (p.K + kBK - 1) / kBK;

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
  griddep_launch();
  griddep_wait();
  const int total_units = 2 * (*p.n_blk);
  // unit -> (block, half); live = the half holds at least one row of the block's task
  auto unit_live = [&](int unit, int &blk, int &half) {
    if (p.reverse) unit = total_units - 1 - unit;
    blk = unit >> 1; half = unit & 1;
    return max(p.blk_lo[blk], half * kBM) < min(p.blk_hi[blk], half * kBM + kBM);
  };

  if (warp == 0) {
    if (lane == 0) {
      tma_prefetch_desc(&p.amap);
      tma_prefetch_desc(&p.wmap[0]);
      int stage = 0; uint32_t phase = 0;
      for (int unit = blockIdx.x; unit < total_units; unit += gridDim.x) {
        int blk, half;
        if (!unit_live(unit, blk, half)) continue;
        const int m0 = p.blk_tile[blk] * 256 + half * kBM;
        const int coff = p.task_coff[p.blk_task[blk]];
        // All 64 slab rows of each target are fetched whatever the task's rank: fetching only the padded rank with a
        // 16-row box measured SLOWER on B200 (cfg4: 11.6 vs 10.2 ms per step) although it moves fewer bytes.
        for (int kb = 0; kb < nK; ++kb) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t *sa = smem + stage * kStageBytes, *sb = sa + kATileBytes;
          mbar_arrive_expect_tx(&full_bar[stage], kATileBytes + p.n_tg * 64 * kBK * 2);
          tma_load_2d(sa, &p.amap, &full_bar[stage], kb * kBK, m0);
          for (int j = 0; j < p.n_tg; ++j)
            tma_load_2d(sb + j * 64 * kBK * 2, &p.wmap[j], &full_bar[stage], kb * kBK, coff);
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t accphase = 0;
      const uint32_t idesc = make_idesc_bf16(kBM, (uint32_t)p.n_tg * 64);
      for (int unit = blockIdx.x; unit < total_units; unit += gridDim.x) {
        int blk, half;
        if (!unit_live(unit, blk, half)) continue;
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
            umma_bf16(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc, (kb | k) != 0);
          umma_commit(&empty_bar[stage]);
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        umma_commit(&tfull_bar[acc]);
        if (++acc == 2) { acc = 0; accphase ^= 1; }
      }
    }
  } else if (warp >= 4) {
    const int wg = (warp - 4) >> 2, quad = warp & 3;
    const int r_in_tile = quad * 32 + lane;
    int acc = 0; uint32_t accphase = 0;
    for (int unit = blockIdx.x; unit < total_units; unit += gridDim.x) {
      int blk, half;
      const bool live = unit_live(unit, blk, half);
      __nv_bfloat16 *U = reinterpret_cast<__nv_bfloat16 *>(p.out) + (size_t)(blk * 256 + half * kBM + r_in_tile) * p.ld_out;
      if (!live) {
        for (int g = wg; g < p.n_tg * 2; g += 2) {
          uint4 *dst = reinterpret_cast<uint4 *>(U + g * 32);
#pragma unroll
          for (int j = 0; j < 4; ++j) dst[j] = make_uint4(0u, 0u, 0u, 0u);
        }
        continue;
      }
      const int t = p.blk_task[blk];
      const int rp = half * kBM + r_in_tile;
      const bool in_seg = rp >= p.blk_lo[blk] && rp < p.blk_hi[blk];
      mbar_wait(&tfull_bar[acc], accphase);
      tc_fence_after();
      const uint32_t t_row = tmem_base + (uint32_t(quad * 32) << 16) + acc * kAccStride;
      uint32_t v[32];
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

template <int kStages, int kTgCap>
constexpr int shrink_smem_bytes() { return kStages * (kATileBytes + kTgCap * 64 * kBK * 2) + 1024; }

}  // namespace fmx
