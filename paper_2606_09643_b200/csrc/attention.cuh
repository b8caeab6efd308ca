// Fused variable-length attention (S3d): softmax(q k^T / sqrt(d_h) + mask) v per request and head,
// online softmax in fp32, GQA (query head g reads KV head g / (H_q/H_kv)), optional causal mask.
// Reads q, k, v from the fused bf16 qkv buffer [N, (H_q + 2 H_kv) d_h] (task-sorted packed rows,
// request p owns rows cu_tok[p] .. cu_tok[p+1]); writes bf16 [N, H_q d_h].
//
// Round-1 implementation: flash-style tiles (64 queries x 64 keys per step) on warp-level
// mma.sync.m16n8k16 with cp.async double-buffered K/V.  Attention is 1-4 % of the forward's
// FLOPs; the tcgen05 version is listed in DESIGN.md "next".
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

namespace fmx {

struct AttnArgs {
  const __nv_bfloat16 *qkv;
  __nv_bfloat16 *out;
  const int *cu_tok;
  int ld_qkv, ld_out;
  int n_q_heads, n_kv_heads;
  int causal;
  float scale_log2;      // log2(e) / sqrt(d_h)
  // optional relative-position bias (attention_kernel only): relb[head * relb_ld + (key - query) + relb_off], already times log2(e)
  const float *relb;
  int relb_ld, relb_off;
};


constexpr int kAttnBQ = 64, kAttnBKV = 64, kAttnThreads = 128;

template <int DH>
constexpr int attn_smem_bytes() { return (kAttnBQ + 4 * kAttnBKV) * (DH + 8) * 2; }

// Copies rows [row0, row0+64) x DH bf16 of a strided global matrix into smem (stride DH+8); rows >= n_valid zero.
template <int DH>
__device__ __forceinline__ void load_tile_async(__nv_bfloat16 *s, const __nv_bfloat16 *g, int ld, int row0, int n_valid) {
  constexpr int kChunks = DH / 8;                       // 16-byte chunks per row
  for (int idx = threadIdx.x; idx < 64 * kChunks; idx += kAttnThreads) {
    const int r = idx / kChunks, c = idx - r * kChunks;
    const int row = row0 + r;
    const bool ok = row < n_valid;
    cp_async_16(s + r * (DH + 8) + c * 8, g + (size_t)(ok ? row : 0) * ld + c * 8, ok ? 16 : 0);
  }
}

template <int DH>
__global__ void __launch_bounds__(kAttnThreads) attention_kernel(const AttnArgs a) {
  constexpr int LD = DH + 8;
  extern __shared__ __align__(16) uint8_t attn_smem[];
  __nv_bfloat16 *sQ = reinterpret_cast<__nv_bfloat16 *>(attn_smem);
  __nv_bfloat16 *sK = sQ + kAttnBQ * LD;                // 2 stages
  __nv_bfloat16 *sV = sK + 2 * kAttnBKV * LD;           // 2 stages
  __shared__ float s_rel[kAttnBQ + kAttnBKV];           // relative-position bias of the current (query tile, key tile): index (key - key0) - (query - q0) + 63

  const int p = blockIdx.z, head = blockIdx.y, q0 = blockIdx.x * kAttnBQ;
  griddep_launch();
  griddep_wait();
  const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
  if (q0 >= n) return;
  const int kvh = head / (a.n_q_heads / a.n_kv_heads);
  const __nv_bfloat16 *gq = a.qkv + (size_t)r0 * a.ld_qkv + head * DH;
  const __nv_bfloat16 *gk = a.qkv + (size_t)r0 * a.ld_qkv + (a.n_q_heads + kvh) * DH;
  const __nv_bfloat16 *gv = a.qkv + (size_t)r0 * a.ld_qkv + (a.n_q_heads + a.n_kv_heads + kvh) * DH;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;

  const int kv_end = a.causal ? min(n, q0 + kAttnBQ) : n;   // keys beyond are masked for every query of the tile
  const int n_kv_tiles = (kv_end + kAttnBKV - 1) / kAttnBKV;

  load_tile_async<DH>(sQ, gq, a.ld_qkv, q0, n);
  load_tile_async<DH>(sK, gk, a.ld_qkv, 0, n);
  load_tile_async<DH>(sV, gv, a.ld_qkv, 0, n);
  cp_async_commit();

  uint32_t qf[DH / 16][4];
  float o[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.0f;
  float m_run[2] = {-1e30f, -1e30f}, l_run[2] = {0.0f, 0.0f};
  const int qrow_a = q0 + warp * 16 + g, qrow_b = qrow_a + 8;   // position of this thread's two rows in the request

  for (int j = 0; j < n_kv_tiles; ++j) {
    const int st = j & 1;
    if (a.relb && threadIdx.x < kAttnBQ + kAttnBKV - 1) {      // the previous iteration ended with a block barrier: s_rel is free
      const int rel = j * kAttnBKV - q0 - (kAttnBQ - 1) + (int)threadIdx.x;
      s_rel[threadIdx.x] = __ldg(a.relb + head * a.relb_ld + min(max(rel + a.relb_off, 0), a.relb_ld - 1));   // (clamped: padding rows / keys only)
    }
    if (j + 1 < n_kv_tiles) {
      load_tile_async<DH>(sK + (st ^ 1) * kAttnBKV * LD, gk, a.ld_qkv, (j + 1) * kAttnBKV, n);
      load_tile_async<DH>(sV + (st ^ 1) * kAttnBKV * LD, gv, a.ld_qkv, (j + 1) * kAttnBKV, n);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    if (j == 0) {
#pragma unroll
      for (int ks = 0; ks < DH / 16; ++ks)
        ldmatrix_x4(qf[ks], sQ + (warp * 16 + (lane & 15)) * LD + ks * 16 + (lane >> 4) * 8);
    }
    const __nv_bfloat16 *k_s = sK + st * kAttnBKV * LD, *v_s = sV + st * kAttnBKV * LD;
    // ---- S = Q K^T (16 x 64 per warp) ----
    float s[8][4];
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.0f;
#pragma unroll
      for (int ks = 0; ks < DH / 16; ++ks) {
        uint32_t b[2];
        ldmatrix_x2(b, k_s + (nt * 8 + (lane & 7)) * LD + ks * 16 + ((lane >> 3) & 1) * 8);
        mma_bf16_16816(s[nt], qf[ks], b);
      }
    }
    // ---- scale, mask, online softmax ----
    const int key0 = j * kAttnBKV;
    float mx[2] = {-1e30f, -1e30f};
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int key = key0 + nt * 8 + t * 2 + (e & 1);
        const int qrow = (e < 2) ? qrow_a : qrow_b;
        const bool masked = key >= n || (a.causal && key > qrow);
        float v = -1e30f;
        if (!masked) {
          v = s[nt][e] * a.scale_log2;
          if (a.relb) v += s_rel[(key - key0) - (qrow - q0) + (kAttnBQ - 1)];
        }
        s[nt][e] = v;
        mx[e >> 1] = fmaxf(mx[e >> 1], v);
      }
    }
    float corr[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
      mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
      const float m_new = fmaxf(m_run[h], mx[h]);
      corr[h] = exp2f(m_run[h] - m_new);
      m_run[h] = m_new;
    }
    float rs[2] = {0.0f, 0.0f};
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float pv = exp2f(s[nt][e] - m_run[e >> 1]);
        s[nt][e] = pv;
        rs[e >> 1] += pv;
      }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) l_run[h] = l_run[h] * corr[h] + rs[h];
#pragma unroll
    for (int i = 0; i < DH / 8; ++i) { o[i][0] *= corr[0]; o[i][1] *= corr[0]; o[i][2] *= corr[1]; o[i][3] *= corr[1]; }
    // ---- O += P V ----
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      uint32_t pa[4];
      pa[0] = pack_bf16(s[2 * kk][0], s[2 * kk][1]);
      pa[1] = pack_bf16(s[2 * kk][2], s[2 * kk][3]);
      pa[2] = pack_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
      pa[3] = pack_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
      for (int dt = 0; dt < DH / 8; ++dt) {
        uint32_t b[2];
        ldmatrix_x2_trans(b, v_s + (kk * 16 + (lane & 15)) * LD + dt * 8);
        mma_bf16_16816(o[dt], pa, b);
      }
    }
    __syncthreads();      // all warps done with stage st before it is refilled
  }
  // ---- normalise and store ----
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 1);
    l_run[h] += __shfl_xor_sync(0xffffffffu, l_run[h], 2);
  }
  const float inv_a = 1.0f / l_run[0], inv_b = 1.0f / l_run[1];
  __nv_bfloat16 *out = a.out + (size_t)r0 * a.ld_out + head * DH;
#pragma unroll
  for (int dt = 0; dt < DH / 8; ++dt) {
    const int col = dt * 8 + t * 2;
    if (qrow_a < n) *reinterpret_cast<uint32_t *>(out + (size_t)qrow_a * a.ld_out + col) = pack_bf16(o[dt][0] * inv_a, o[dt][1] * inv_a);
    if (qrow_b < n) *reinterpret_cast<uint32_t *>(out + (size_t)qrow_b * a.ld_out + col) = pack_bf16(o[dt][2] * inv_b, o[dt][3] * inv_b);
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// Short sequences (every request <= 64 tokens: cfg1 / cfg2 / cfg5): one (request, head) item is a single 64 x 64 tile, so
// the flash loop above degenerates into load -> compute -> store with nothing to overlap, and the step is bound by
// per-CTA latency (ncu, cfg2: 42 us per layer for 113 MB of traffic).  Here a CTA walks a strided list of items with a
// two-stage cp.async pipeline (Q, K, V of item i+1 are in flight while item i is computed), and the output tile leaves
// through shared memory as whole 128-byte row segments.
template <int DH>
constexpr int attn_short_smem_bytes() { return 2 * 3 * 64 * (DH + 8) * 2; }

template <int DH>
__global__ void __launch_bounds__(kAttnThreads) attention_short_kernel(const AttnArgs a, int n_req) {
  constexpr int LD = DH + 8;
  constexpr int kTile = 64 * LD;                        // elements of one 64-row tile
  extern __shared__ __align__(16) uint8_t attn_smem[];
  __nv_bfloat16 *sbase = reinterpret_cast<__nv_bfloat16 *>(attn_smem);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int n_items = n_req * a.n_q_heads;
  const int group = a.n_q_heads / a.n_kv_heads;
  griddep_launch();
  griddep_wait();

  auto issue = [&](int item, int st) {
    const int p = item / a.n_q_heads, head = item - p * a.n_q_heads;
    const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
    const int kvh = head / group;
    const __nv_bfloat16 *base = a.qkv + (size_t)r0 * a.ld_qkv;
    __nv_bfloat16 *s = sbase + st * 3 * kTile;
    load_tile_async<DH>(s, base + head * DH, a.ld_qkv, 0, n);
    load_tile_async<DH>(s + kTile, base + (a.n_q_heads + kvh) * DH, a.ld_qkv, 0, n);
    load_tile_async<DH>(s + 2 * kTile, base + (a.n_q_heads + a.n_kv_heads + kvh) * DH, a.ld_qkv, 0, n);
  };

  int item = blockIdx.x;
  if (item < n_items) issue(item, 0);
  cp_async_commit();
  for (int it = 0; item < n_items; item += gridDim.x, ++it) {
    const int st = it & 1;
    const int next = item + gridDim.x;
    if (next < n_items) issue(next, st ^ 1);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();
    const int p = item / a.n_q_heads, head = item - p * a.n_q_heads;
    const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
    __nv_bfloat16 *sQ = sbase + st * 3 * kTile, *k_s = sQ + kTile, *v_s = sQ + 2 * kTile;
    const int qrow_a = warp * 16 + g, qrow_b = qrow_a + 8;
    if (warp * 16 < n) {                                  // warps whose 16 queries do not exist skip the math
      uint32_t qf[DH / 16][4];
#pragma unroll
      for (int ks = 0; ks < DH / 16; ++ks) ldmatrix_x4(qf[ks], sQ + (warp * 16 + (lane & 15)) * LD + ks * 16 + (lane >> 4) * 8);
      float s[8][4];
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.0f;
#pragma unroll
        for (int ks = 0; ks < DH / 16; ++ks) {
          uint32_t b[2];
          ldmatrix_x2(b, k_s + (nt * 8 + (lane & 7)) * LD + ks * 16 + ((lane >> 3) & 1) * 8);
          mma_bf16_16816(s[nt], qf[ks], b);
        }
      }
      // raw scores; the 1/sqrt(d_h) log2(e) scale is folded into the exponent: p = 2^(s c - max(s) c), c > 0
      if (n < 64 || a.causal) {                           // CTA-uniform: a full non-causal tile needs no mask
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int key = nt * 8 + t * 2 + (e & 1);
            const int qrow = (e < 2) ? qrow_a : qrow_b;
            if (key >= n || (a.causal && key > qrow)) s[nt][e] = -INFINITY;
          }
        }
      }
      float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        mx[0] = fmaxf(mx[0], fmaxf(s[nt][0], s[nt][1]));
        mx[1] = fmaxf(mx[1], fmaxf(s[nt][2], s[nt][3]));
      }
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
        mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
        mx[h] *= -a.scale_log2;                           // key 0 is visible to every query: the maximum is finite
      }
      float rs[2] = {0.0f, 0.0f};
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float pv = fast_exp2(fmaf(s[nt][e], a.scale_log2, mx[e >> 1]));
          s[nt][e] = pv;
          rs[e >> 1] += pv;
        }
      }
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        rs[h] += __shfl_xor_sync(0xffffffffu, rs[h], 1);
        rs[h] += __shfl_xor_sync(0xffffffffu, rs[h], 2);
      }
      float o[DH / 8][4];
#pragma unroll
      for (int i = 0; i < DH / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.0f;
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        uint32_t pa[4];
        pa[0] = pack_bf16(s[2 * kk][0], s[2 * kk][1]);
        pa[1] = pack_bf16(s[2 * kk][2], s[2 * kk][3]);
        pa[2] = pack_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
        pa[3] = pack_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
        for (int dt = 0; dt < DH / 8; ++dt) {
          uint32_t b[2];
          ldmatrix_x2_trans(b, v_s + (kk * 16 + (lane & 15)) * LD + dt * 8);
          mma_bf16_16816(o[dt], pa, b);
        }
      }
      // O / l -> bf16 into this warp's own 16 rows of the Q tile (only this warp read them), then whole rows to global
      const float inv_a = 1.0f / rs[0], inv_b = 1.0f / rs[1];
      __syncwarp();
#pragma unroll
      for (int dt = 0; dt < DH / 8; ++dt) {
        const int col = dt * 8 + t * 2;
        *reinterpret_cast<uint32_t *>(sQ + qrow_a * LD + col) = pack_bf16(o[dt][0] * inv_a, o[dt][1] * inv_a);
        *reinterpret_cast<uint32_t *>(sQ + qrow_b * LD + col) = pack_bf16(o[dt][2] * inv_b, o[dt][3] * inv_b);
      }
      __syncwarp();
      constexpr int kChunks = DH / 8;                     // 16-byte chunks per row
      __nv_bfloat16 *out = a.out + (size_t)r0 * a.ld_out + head * DH;
      for (int idx = lane; idx < 16 * kChunks; idx += 32) {
        const int r = warp * 16 + idx / kChunks, c = idx % kChunks;
        if (r < n) *reinterpret_cast<uint4 *>(out + (size_t)r * a.ld_out + c * 8) = *reinterpret_cast<const uint4 *>(sQ + r * LD + c * 8);
      }
    }
    __syncthreads();      // stage st is refilled by the next iteration's prefetch
  }
}

}  // namespace fmx
