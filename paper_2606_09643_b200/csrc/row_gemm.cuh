// Small-M projection for decode iterations (NEXT-3): partial[ks, row, n] = sum over the k-slice ks of x[row, k] W[n, k].
//
// A decode batch has one row per request (M <= 128 here), so the projection is a stream over the weight matrix with almost no
// arithmetic per byte: the prefill kernel (pair_gemm.cuh: 256-row tcgen05 tiles on CTA pairs, TMEM, a persistent grid with
// ~200 KB of shared memory per CTA) does 4x the useful MMA work at M = 64, pays its fixed costs (TMEM allocation, cluster
// barriers, an 8-box epilogue of 256 rows) on two k-blocks of real work, and keeps every SM's shared memory to itself while the
// row-wise LoRA kernels want to run beside it.  This kernel is the lean form of the same product:
//   grid (N / 128, k_split): a CTA takes 128 output columns (one weight source; gate / up chunks alternate for SwiGLU, as in the
//        prefill kernel's output layout) and one slice of K, so that ~2 CTAs per SM stream the matrix;
//   cp.async 16-byte copies of x [M, 64] and W [128, 64] chunks into a 4-stage shared-memory ring (rows padded by 16 bytes:
//        conflict-free ldmatrix);
//   mma.sync m16n8k16 (bf16 in, fp32 accumulate): warp w owns columns 16 w .. 16 w + 15 of the slice for every 16-row tile;
//   the raw fp32 partial goes to [k_split, split_rows, N]; splitk_reduce_kernel / qkv_reduce_rope_kernel /
//        reduce_resid_norm_kernel add the slices in order, the LoRA delta and the bias, and apply what follows.
// k_split depends on the projection's shape only, never on the batch, and a row's accumulation does not depend on the other rows:
// a request decodes to the same bits alone and in any batch of <= 128 rows (larger batches take the pair GEMM: another summation order).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

namespace fmx {

constexpr int kRgCols = 128, kRgBK = 64, kRgStages = 4, kRgLd = kRgBK + 8;      // smem row stride in elements (144 bytes)

struct RowGemmArgs {
  const __nv_bfloat16 *x;          // [M, K]
  int M, K, N;                     // N = total output columns (multiple of 128)
  const __nv_bfloat16 *W[3];       // weight sources [n_s, K], K contiguous
  int src_end_col[3];              // first column AFTER source s (cumulative); ignored with interleave2
  int interleave2;                 // SwiGLU: 128-column slice q takes rows 128 (q / 2) .. of source q & 1
  int chunks_per_split;            // 64-wide k chunks per slice
  int split_rows;                  // rows of one slice's partial (>= M, multiple of 16)
  float *partial;                  // [k_split, split_rows, N]
};

template <int MT>
constexpr size_t row_gemm_smem() { return (size_t)kRgStages * (MT * 16 + kRgCols) * kRgLd * sizeof(__nv_bfloat16); }

template <int MT>                  // 16-row tiles: M <= 16 MT
__global__ void __launch_bounds__(256) row_gemm_kernel(const RowGemmArgs a) {
  extern __shared__ __align__(16) unsigned char rg_smem[];
  constexpr int kRowsX = MT * 16, kStageElems = (kRowsX + kRgCols) * kRgLd;
  __nv_bfloat16 *smem = reinterpret_cast<__nv_bfloat16 *>(rg_smem);
  griddep_launch();
  griddep_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int c0 = blockIdx.x * kRgCols, ks = blockIdx.y;
  // the slice's weight rows
  const __nv_bfloat16 *Wp;
  if (a.interleave2) {
    Wp = a.W[blockIdx.x & 1] + (size_t)(blockIdx.x >> 1) * kRgCols * a.K;
  } else {
    int s = 0, begin = 0;
    if (c0 >= a.src_end_col[0]) { s = 1; begin = a.src_end_col[0]; }
    if (c0 >= a.src_end_col[1]) { s = 2; begin = a.src_end_col[1]; }
    Wp = a.W[s] + (size_t)(c0 - begin) * a.K;
  }
  const int nK = (a.K + kRgBK - 1) / kRgBK;
  const int kb0 = ks * a.chunks_per_split, kb1 = min(nK, kb0 + a.chunks_per_split);
  // the thread's copies of a chunk are the same (row, 16-byte piece) pairs every time: their source pointers and shared-memory
  // offsets are computed once, a chunk then costs one add and one cp.async per copy
  constexpr int kCopies = ((kRowsX + kRgCols) * 8 + 255) / 256;
  const __nv_bfloat16 *src[kCopies];
  int sdst[kCopies], pc8[kCopies];                              // pc8 < 0: no copy / zero row
#pragma unroll
  for (int c = 0; c < kCopies; ++c) {
    const int idx = threadIdx.x + c * 256, row = idx >> 3, pc = idx & 7;
    sdst[c] = row * kRgLd + pc * 8;
    pc8[c] = pc * 8;
    if (idx >= (kRowsX + kRgCols) * 8) { pc8[c] = -1; src[c] = a.x; sdst[c] = 0; }
    else if (row < kRowsX) { src[c] = a.x + (size_t)(row < a.M ? row : 0) * a.K + pc * 8; if (row >= a.M) pc8[c] = -2; }
    else src[c] = Wp + (size_t)(row - kRowsX) * a.K + pc * 8;
  }
  auto load_stage = [&](int kb, int stage) {
    __nv_bfloat16 *sbase = smem + (size_t)stage * kStageElems;
    const int k0 = kb * kRgBK;
#pragma unroll
    for (int c = 0; c < kCopies; ++c) {
      if (pc8[c] == -1) continue;
      const bool ok = pc8[c] >= 0 && k0 + pc8[c] < a.K;         // (K is a multiple of 8; rows past M and the K tail are zero-filled)
      cp_async_16(sbase + sdst[c], src[c] + (ok ? k0 : 0), ok ? 16 : 0);
    }
  };
  float acc[MT][2][4];
#pragma unroll
  for (int mt = 0; mt < MT; ++mt)
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = acc[mt][nt][2] = acc[mt][nt][3] = 0.0f;
  // prologue: up to kRgStages - 1 chunks in flight
#pragma unroll
  for (int s = 0; s < kRgStages - 1; ++s) {
    if (kb0 + s < kb1) load_stage(kb0 + s, s);
    cp_async_commit();
  }
  for (int kb = kb0; kb < kb1; ++kb) {
    const int it = kb - kb0;
    cp_async_wait<kRgStages - 2>();
    __syncthreads();                                            // chunk `it` has landed; the stage refilled below is free
    if (kb + kRgStages - 1 < kb1) load_stage(kb + kRgStages - 1, (it + kRgStages - 1) % kRgStages);
    cp_async_commit();
    const __nv_bfloat16 *sx = smem + (size_t)(it % kRgStages) * kStageElems, *sw = sx + kRowsX * kRgLd;
#pragma unroll
    for (int kk = 0; kk < kRgBK / 16; ++kk) {
      uint32_t bw[4];                                           // W^T fragments of the warp's two 8-column tiles
      ldmatrix_x4(bw, sw + (warp * 16 + (lane >> 4) * 8 + (lane & 7)) * kRgLd + kk * 16 + ((lane >> 3) & 1) * 8);
      const uint32_t b0[2] = {bw[0], bw[1]}, b1[2] = {bw[2], bw[3]};
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        uint32_t ax[4];
        ldmatrix_x4(ax, sx + (mt * 16 + (lane & 15)) * kRgLd + kk * 16 + (lane >> 4) * 8);
        mma_bf16_16816(acc[mt][0], ax, b0);
        mma_bf16_16816(acc[mt][1], ax, b1);
      }
    }
  }
  cp_async_wait<0>();
  float *dst = a.partial + (size_t)ks * a.split_rows * a.N + c0 + warp * 16 + 2 * (lane & 3);
#pragma unroll
  for (int mt = 0; mt < MT; ++mt) {
    const int r0 = mt * 16 + (lane >> 2), r1 = r0 + 8;
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      if (r0 < a.M) *reinterpret_cast<float2 *>(dst + (size_t)r0 * a.N + nt * 8) = make_float2(acc[mt][nt][0], acc[mt][nt][1]);
      if (r1 < a.M) *reinterpret_cast<float2 *>(dst + (size_t)r1 * a.N + nt * 8) = make_float2(acc[mt][nt][2], acc[mt][nt][3]);
    }
  }
}

}  // namespace fmx
