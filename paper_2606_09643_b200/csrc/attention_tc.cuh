// Fused variable-length attention on tcgen05 / TMEM / TMA (S3d) for head_dim 64 and 128:
//   o = softmax(q k^T / sqrt(d_h) + mask) v   per request and query head, online softmax in fp32,
//   GQA (query head g reads KV head g / (H_q / H_kv)), optional causal mask.
// q, k, v live in the fused bf16 buffer [N, (H_q + 2 H_kv) d_h] (task-sorted packed rows, request p owns rows
// cu_tok[p] .. cu_tok[p+1]); output bf16 [N, H_q d_h].
//
// One CTA = (request, query head, kQT consecutive 128-query tiles).  Per 64-key tile j and q-tile q:
//   S_q  = Q_q K_j^T        tcgen05.mma  M=128 N=64  K=d_h   A = Q (smem, K-major), B = K_j (smem, K-major) -> TMEM
//   P_q  = exp2(S_q * c - m)  one softmax warpgroup per q-tile; thread = query row = TMEM lane, so the row max and
//                           the row sum need no shuffles; P goes to smem as bf16 in the 128B-swizzled K-major layout
//   O_q += P_q V_j          tcgen05.mma  M=128 N=d_h K=64    A = P (smem), B = V_j (smem, MN-major: V is [key, d_h]
//                           with d_h contiguous, exactly what TMA delivers) -> TMEM accumulator
// The running maximum is updated lazily: the reference m only moves when the tile maximum exceeds it by more than
// 2^8, and only then is O (in TMEM) rescaled by the softmax warps; O / l is exact either way because P, l and O all
// use the same reference.
//
// Warp roles (128 + 128 kQT threads): warp 0 TMA producer (Q once, K/V ring), warp 1 tcgen05.mma issuer, warp 2
// TMEM allocator, warps 4.. softmax warpgroups.  While warpgroup q works on tile j the tensor core runs S_q(j+1)
// (S is released as soon as it is in registers) and the other warpgroup's MMAs.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

namespace fmx {

constexpr int kAtBQ = 128;       // queries per q-tile (TMEM lanes)
constexpr int kAtBKV = 64;       // keys per KV tile

struct AttnTcArgs {
  CUtensorMap qkv_map;           // [N, d_qkv] bf16, box {64 columns, 64 rows}, 128B swizzle
  __nv_bfloat16 *out;
  const int *cu_tok;
  int ld_out;
  int n_q_heads, n_kv_heads;
  int causal;
  float scale_log2;              // log2(e) / sqrt(d_h)
  int reverse;                   // 1: requests are walked from the last to the first (blockIdx.z reversed)
};

// Dynamic shared memory: the operand tiles (1024-byte aligned for the 128B swizzle) plus 1 KB that holds the alignment
// slack and the mbarriers; no static shared memory, so two CTAs of the d_h = 128 variant (112 KB of tiles) fit one SM.
template <int DH, int kQT, int kAtStages>
__host__ __device__ constexpr int attn_tc_tile_bytes() { return kQT * (DH / 64) * 16384 + 2 * kAtStages * (DH / 64) * 8192 + kQT * 16384; }
template <int DH, int kQT, int kAtStages>
constexpr int attn_tc_smem_bytes() { return attn_tc_tile_bytes<DH, kQT, kAtStages>() + 1024; }
template <int kQT>
constexpr int attn_tc_threads() { return 128 + 128 * kQT; }

// MN-major, 128B-swizzled B operand: [K rows of 128 bytes][64-column blocks lbo_bytes apart]
__device__ __forceinline__ uint64_t make_smem_desc_sw128_mn(uint32_t smem_addr, uint32_t lbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
  d |= (uint64_t)(lbo_bytes >> 4) << 16;                 // next 64 MN elements
  d |= (uint64_t)(1024u >> 4) << 32;                     // next 8 K rows
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

// kAtStages: K and V ring depth; kMinBlocks: CTAs that must fit one SM (registers are capped accordingly)
template <int DH, int kQT, int kAtStages, int kMinBlocks>
__global__ void __launch_bounds__(128 + 128 * kQT, kMinBlocks) attention_tc_kernel(const __grid_constant__ AttnTcArgs a) {
  constexpr int kKB = DH / 64;                        // 64-column blocks of the head
  constexpr int kQBytes = kKB * 16384;                // one q-tile
  constexpr int kKVBytes = kKB * 8192;                // one K (or V) tile
  constexpr uint32_t kTmemCols = (kQT * (64 + DH) <= 128) ? 128 : (kQT * (64 + DH) <= 256) ? 256 : 512;
  static_assert(kQT * (64 + DH) <= 512, "TMEM budget");
  extern __shared__ uint8_t at_smem_raw[];
  const uint32_t raw_addr = smem_u32(at_smem_raw);
  const uint32_t pad = (1024u - (raw_addr & 1023u)) & 1023u;
  uint8_t *smem = at_smem_raw + pad;
  uint8_t *sQ = smem;
  uint8_t *sK = sQ + kQT * kQBytes;
  uint8_t *sV = sK + kAtStages * kKVBytes;
  uint8_t *sP = sV + kAtStages * kKVBytes;
  // barriers (256 bytes) live in the alignment slack: before the tiles when the pad is large enough, else after them
  constexpr int kTileBytes = attn_tc_tile_bytes<DH, kQT, kAtStages>();
  uint64_t *bars = reinterpret_cast<uint64_t *>(pad >= 256 ? at_smem_raw + ((pad - 256) & ~7u) : smem + kTileBytes);
  uint64_t &q_full = bars[0];
  uint64_t *k_full = bars + 1, *k_empty = k_full + kAtStages, *v_full = k_empty + kAtStages, *v_empty = v_full + kAtStages;
  uint64_t *s_full = v_empty + kAtStages, *s_free = s_full + kQT, *p_ready = s_free + kQT, *pv_done = p_ready + kQT;
  uint32_t &tmem_base_slot = *reinterpret_cast<uint32_t *>(pv_done + kQT);
  static_assert((1 + 4 * kAtStages + 4 * kQT + 1) * 8 <= 256, "barrier block");

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int p = a.reverse ? (int)gridDim.z - 1 - (int)blockIdx.z : (int)blockIdx.z, head = blockIdx.y;
  griddep_launch();
  griddep_wait();
  const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
  const int q0 = ((int)gridDim.x - 1 - (int)blockIdx.x) * (kAtBQ * kQT);      // heavy (late) causal tiles first
  if (q0 >= n) return;
  const int kvh = head / (a.n_q_heads / a.n_kv_heads);
  const int col_q = head * DH, col_k = (a.n_q_heads + kvh) * DH, col_v = (a.n_q_heads + a.n_kv_heads + kvh) * DH;
  int nkv[kQT], max_kv = 0;
#pragma unroll
  for (int q = 0; q < kQT; ++q) {
    const int row0 = q0 + q * kAtBQ;
    const int kv_end = row0 >= n ? 0 : (a.causal ? min(n, row0 + kAtBQ) : n);
    nkv[q] = (kv_end + kAtBKV - 1) / kAtBKV;
    max_kv = max(max_kv, nkv[q]);
  }

  if (threadIdx.x == 0) {
    mbar_init(&q_full, 1);
    for (int s = 0; s < kAtStages; ++s) { mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], 1); mbar_init(&v_full[s], 1); mbar_init(&v_empty[s], 1); }
    for (int q = 0; q < kQT; ++q) { mbar_init(&s_full[q], 1); mbar_init(&s_free[q], 4); mbar_init(&p_ready[q], 4); mbar_init(&pv_done[q], 1); }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(&tmem_base_slot, kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_slot;

  if (warp == 0) {
    // ================================ TMA producer ================================
    if (lane == 0) {
      tma_prefetch_desc(&a.qkv_map);
      int n_qt = 0;
#pragma unroll
      for (int q = 0; q < kQT; ++q) n_qt += nkv[q] > 0;
      mbar_arrive_expect_tx(&q_full, n_qt * kQBytes);
#pragma unroll
      for (int q = 0; q < kQT; ++q) {
        if (nkv[q] == 0) continue;
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb)
#pragma unroll
          for (int h = 0; h < 2; ++h)
            tma_load_2d(sQ + q * kQBytes + kb * 16384 + h * 8192, &a.qkv_map, &q_full, col_q + kb * 64, r0 + q0 + q * kAtBQ + h * 64);
      }
      int stage = 0; uint32_t phase = 0;
      for (int j = 0; j < max_kv; ++j) {
        const int row = r0 + j * kAtBKV;
        mbar_wait(&k_empty[stage], phase ^ 1);
        mbar_arrive_expect_tx(&k_full[stage], kKVBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) tma_load_2d(sK + stage * kKVBytes + kb * 8192, &a.qkv_map, &k_full[stage], col_k + kb * 64, row);
        mbar_wait(&v_empty[stage], phase ^ 1);
        mbar_arrive_expect_tx(&v_full[stage], kKVBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) tma_load_2d(sV + stage * kKVBytes + kb * 8192, &a.qkv_map, &v_full[stage], col_v + kb * 64, row);
        if (++stage == kAtStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ================================ MMA issuer ================================
    if (lane == 0) {
      constexpr uint32_t idesc_s = make_idesc_bf16(kAtBQ, kAtBKV);
      constexpr uint32_t idesc_o = make_idesc_bf16(kAtBQ, DH) | (1u << 16);      // B (= V) is MN-major
      auto issue_s = [&](int q, int stage) {
        const uint32_t qa = smem_u32(sQ + q * kQBytes), ka = smem_u32(sK + stage * kKVBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) {
          const uint64_t adesc = make_smem_desc_sw128(qa + kb * 16384), bdesc = make_smem_desc_sw128(ka + kb * 8192);
#pragma unroll
          for (int k = 0; k < 4; ++k) umma_bf16(tmem_base + q * 64, adesc + 2 * k, bdesc + 2 * k, idesc_s, (kb | k) != 0);
        }
        umma_commit(&s_full[q]);
      };
      mbar_wait(&q_full, 0);
      mbar_wait(&k_full[0], 0);
      tc_fence_after();
#pragma unroll
      for (int q = 0; q < kQT; ++q) if (nkv[q] > 0) issue_s(q, 0);
      umma_commit(&k_empty[0]);
      int stage = 0; uint32_t phase = 0;
      for (int j = 0; j < max_kv; ++j) {
        int nstage = stage + 1; uint32_t nphase = phase;
        if (nstage == kAtStages) { nstage = 0; nphase ^= 1; }
        if (j + 1 < max_kv) {
          mbar_wait(&k_full[nstage], nphase);
#pragma unroll
          for (int q = 0; q < kQT; ++q) {
            if (j + 1 >= nkv[q]) continue;
            mbar_wait(&s_free[q], j & 1);            // S_q(j) is in the softmax warps' registers
            tc_fence_after();
            issue_s(q, nstage);
          }
          umma_commit(&k_empty[nstage]);
        }
        mbar_wait(&v_full[stage], phase);
#pragma unroll
        for (int q = 0; q < kQT; ++q) {
          if (j >= nkv[q]) continue;
          mbar_wait(&p_ready[q], j & 1);             // P_q(j) in smem, O_q rescaled if it had to be
          tc_fence_after();
          const uint32_t pa = smem_u32(sP + q * 16384), va = smem_u32(sV + stage * kKVBytes);
#pragma unroll
          for (int k = 0; k < 4; ++k)
            umma_bf16(tmem_base + kQT * 64 + q * DH, make_smem_desc_sw128(pa) + 2 * k, make_smem_desc_sw128_mn(va + k * 2048, 8192),
                      idesc_o, (j | k) != 0);
          umma_commit(&pv_done[q]);
        }
        umma_commit(&v_empty[stage]);
        stage = nstage; phase = nphase;
      }
    }
  } else if (warp >= 4) {
    // ================================ softmax warpgroups ================================
    const int q = (warp - 4) >> 2, quad = warp & 3;
    const int n_tiles = nkv[q];
    if (n_tiles > 0) {
      const int r_in_tile = quad * 32 + lane;
      const int qrow = q0 + q * kAtBQ + r_in_tile;                 // position within the request
      const int warp_row_lo = q0 + q * kAtBQ + quad * 32;
      const uint32_t t_s = tmem_base + (uint32_t(quad * 32) << 16) + q * 64;
      const uint32_t t_o = tmem_base + (uint32_t(quad * 32) << 16) + kQT * 64 + q * DH;
      uint8_t *p_row = sP + q * 16384 + r_in_tile * 128;
      const int rsw = r_in_tile & 7;
      float m_ref = 0.0f, l_run = 0.0f;
      uint32_t v[64];
      if (warp_row_lo >= n) {
        // No query of this warp exists (cfg3: the third q-tile of a 257-token request holds ONE row): keep the barrier
        // protocol going and leave the exp2 / issue slots to the warps (and the co-resident CTA) that have rows.
        for (int j = 0; j < n_tiles; ++j) {
          mbar_wait(&s_full[q], j & 1);
          __syncwarp();
          if (lane == 0) mbar_arrive(&s_free[q]);
          if (j > 0) mbar_wait(&pv_done[q], (j - 1) & 1);            // p_ready phase j-1 is complete: no arrival can land in it
          __syncwarp();
          if (lane == 0) mbar_arrive(&p_ready[q]);
        }
      } else {
      for (int j = 0; j < n_tiles; ++j) {
        mbar_wait(&s_full[q], j & 1);
        tc_fence_after();
        tmem_ld_32x32(t_s, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tmem_ld_32x32(t_s + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_free[q]);
        const int key0 = j * kAtBKV;
        float mx = -INFINITY;
        if (key0 + kAtBKV > n || (a.causal && key0 + kAtBKV - 1 > warp_row_lo)) {
          const int lim = a.causal ? min(n, qrow + 1) : n;         // keys [0, lim) are visible to this row
#pragma unroll
          for (int c = 0; c < 64; ++c) {
            const float s = (key0 + c < lim) ? __uint_as_float(v[c]) : -INFINITY;
            v[c] = __float_as_uint(s);
            mx = fmaxf(mx, s);
          }
        } else {
#pragma unroll
          for (int c = 0; c < 64; ++c) mx = fmaxf(mx, __uint_as_float(v[c]));
        }
        mx *= a.scale_log2;                                         // scale > 0; -inf stays -inf
        float factor = 1.0f;
        bool rescale = false;
        if (j == 0) {
          m_ref = (mx == -INFINITY) ? 0.0f : mx;
        } else if (mx > m_ref + 8.0f) {
          factor = fast_exp2(m_ref - mx);
          m_ref = mx;
          rescale = true;
        }
        float rs = 0.0f;
        uint32_t pk[32];
#pragma unroll
        for (int c = 0; c < 64; c += 2) {
          const float p0 = fast_exp2(fmaf(__uint_as_float(v[c]), a.scale_log2, -m_ref));
          const float p1 = fast_exp2(fmaf(__uint_as_float(v[c + 1]), a.scale_log2, -m_ref));
          rs += p0 + p1;
          pk[c >> 1] = pack_bf16(p0, p1);
        }
        l_run = l_run * factor + rs;
        if (j > 0) {
          mbar_wait(&pv_done[q], (j - 1) & 1);                      // P buffer free, O_q quiescent
          if (__any_sync(0xffffffffu, rescale)) {
            tc_fence_after();
#pragma unroll 1
            for (int c = 0; c < DH; c += 32) {
              uint32_t o[32];
              tmem_ld_32x32(t_o + c, o);
              tmem_ld_wait();
#pragma unroll
              for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * factor);
              tmem_st_32x32(t_o + c, o);
            }
            tmem_st_wait();
            tc_fence_before();
          }
        }
#pragma unroll
        for (int c = 0; c < 8; ++c)
          *reinterpret_cast<uint4 *>(p_row + ((c ^ rsw) << 4)) = make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive(&p_ready[q]);
      }
      // ---- O / l -> bf16 -> global ----
      mbar_wait(&pv_done[q], (n_tiles - 1) & 1);
      tc_fence_after();
      const float inv = 1.0f / l_run;
      __nv_bfloat16 *dst = a.out + (size_t)(r0 + qrow) * a.ld_out + head * DH;
#pragma unroll 1
      for (int c = 0; c < DH; c += 32) {
        uint32_t o[32];
        tmem_ld_32x32(t_o + c, o);
        tmem_ld_wait();
        if (qrow < n) {
#pragma unroll
          for (int e = 0; e < 4; ++e)
            reinterpret_cast<uint4 *>(dst + c)[e] =
                make_uint4(pack_bf16(__uint_as_float(o[8 * e]) * inv, __uint_as_float(o[8 * e + 1]) * inv),
                           pack_bf16(__uint_as_float(o[8 * e + 2]) * inv, __uint_as_float(o[8 * e + 3]) * inv),
                           pack_bf16(__uint_as_float(o[8 * e + 4]) * inv, __uint_as_float(o[8 * e + 5]) * inv),
                           pack_bf16(__uint_as_float(o[8 * e + 6]) * inv, __uint_as_float(o[8 * e + 7]) * inv));
        }
      }
      }   // warp with rows
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace fmx
