// Fused attention for batches of SHORT requests (every request <= 64 tokens, head_dim 64: cfg2 / cfg5) on tcgen05 / TMEM /
// TMA (S3d).  A (request, head) problem is one 64 x 64 tile, half of the 128-row tcgen05 MMA; so TWO heads of a request
// share one MMA as a block-diagonal problem:
//     A = [Q_h ; Q_h+1]  (128 x 64)      B = [K_h ; K_h+1]  (128 keys x 64)      S = A B^T  (128 x 128, M128 N128 K64)
// rows 0-63 use S columns 0-63, rows 64-127 use columns 64-127 (the off-diagonal blocks are never read).  Softmax: thread
// = row = TMEM lane, no shuffles; one KV tile per item, so no running maximum.  P goes back to TMEM as bf16 pairs over
// K = 128 (the other head's 64 keys are written as zeros) and O = P [V_h ; V_h+1] is one M128 N64 K128 tcgen05.mma with a
// TMEM A operand; V is MN-major exactly as TMA delivers it.
//
// Persistent CTA, kP64Lanes independent lanes, each with its own producer thread, MMA-issuer thread, softmax warpgroup,
// 256 TMEM columns [S 128 | P 64 | O 64] and a two-stage shared-memory ring of (Q, K, V) item tiles, so the loads of the
// next two items are always in flight.  Per lane the issuer runs PV_i as soon as P_i is ready and S_(i+1) right behind it
// (its operands are already resident), which overlaps S_(i+1) with the output epilogue of item i; the other lane fills the
// remaining bubbles.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "attention_fa.cuh"
#include "ptx.cuh"

namespace fmx {

struct AttnPairArgs {
  CUtensorMap qkv_map;           // [N, d_qkv] bf16, box {64 columns, 64 rows}, 128B swizzle
  __nv_bfloat16 *out;
  const int *cu_tok;
  int ld_out;
  int n_req, n_q_heads, n_kv_heads;
  int causal;
  float scale_log2;              // log2(e) / sqrt(d_h)
  int reverse;                   // 1: items are walked from the last request to the first
};

constexpr int kP64Lanes = 2;
constexpr int kP64StageBytes = 3 * 16384;                     // Q | K | V tiles of one item (two heads each)
constexpr int kP64LaneBytes = 2 * kP64StageBytes;
constexpr int kP64Threads = 256 + 128 * kP64Lanes;
constexpr int attn_pair64_smem_bytes() { return kP64Lanes * kP64LaneBytes + 1024 + 256; }

__global__ void __launch_bounds__(kP64Threads, 1) attention_pair64_kernel(const __grid_constant__ AttnPairArgs a) {
  constexpr int DH = 64;
  extern __shared__ uint8_t ap_smem_raw[];
  const uint32_t pad = (1024u - (smem_u32(ap_smem_raw) & 1023u)) & 1023u;
  uint8_t *tiles = ap_smem_raw + pad;
  uint64_t *bars = reinterpret_cast<uint64_t *>(tiles + kP64Lanes * kP64LaneBytes);    // 7 per lane
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 7 * kP64Lanes);

  const int warp = threadIdx.x >> 5, lane_id = threadIdx.x & 31;
  const int wg = warp >> 2;                                   // 0 producers, 1 MMA issuers, 2.. softmax (one per lane)
  if (threadIdx.x == 0) {
    for (int l = 0; l < kP64Lanes; ++l) {
      uint64_t *b = bars + 7 * l;
      for (int i = 0; i < 5; ++i) mbar_init(&b[i], 1);        // full[2] empty[2] s_full
      mbar_init(&b[5], 4);                                    // p_ready (one arrive per softmax warp)
      mbar_init(&b[6], 1);                                    // o_full  (tcgen05.commit)
    }
    fence_barrier_init();
  }
  if (warp == 4) {
    tmem_alloc(tmem_slot, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  griddep_launch();
  griddep_wait();

  const int lane = wg == 0 ? warp : (wg == 1 ? warp - 4 : wg - 2);
  const bool active = lane < kP64Lanes;
  uint8_t *sIt = tiles + (active ? lane : 0) * kP64LaneBytes;
  uint64_t *lb = bars + 7 * (active ? lane : 0);
  uint64_t *full = lb, *empty = lb + 2;
  uint64_t &s_full = lb[4], &p_ready = lb[5], &o_full = lb[6];
  const uint32_t t_lane = tmem_base + lane * 256;

  const int n_hp = a.n_q_heads >> 1;                          // head pairs per request
  const int total_items = a.n_req * n_hp;
  const int item0 = blockIdx.x * kP64Lanes + lane, item_step = gridDim.x * kP64Lanes;
  const int group = a.n_q_heads / a.n_kv_heads;

  if (wg == 0) {
    // ================================ TMA producers (one thread per lane) ================================
    if (active && lane_id == 0) {
      tma_prefetch_desc(&a.qkv_map);
      int stage = 0; uint32_t phase = 0;
      for (int idx = item0; idx < total_items; idx += item_step) {
        const int p = a.reverse ? a.n_req - 1 - idx / n_hp : idx / n_hp, h0 = (idx % n_hp) * 2;
        const int r0 = a.cu_tok[p];
        const int kv0 = h0 / group, kv1 = (h0 + 1) / group;
        uint8_t *sQ = sIt + stage * kP64StageBytes, *sK = sQ + 16384, *sV = sK + 16384;
        mbar_wait(&empty[stage], phase ^ 1);
        mbar_arrive_expect_tx(&full[stage], kP64StageBytes);
        tma_load_2d(sQ, &a.qkv_map, &full[stage], h0 * DH, r0);
        tma_load_2d(sQ + 8192, &a.qkv_map, &full[stage], (h0 + 1) * DH, r0);
        tma_load_2d(sK, &a.qkv_map, &full[stage], (a.n_q_heads + kv0) * DH, r0);
        tma_load_2d(sK + 8192, &a.qkv_map, &full[stage], (a.n_q_heads + kv1) * DH, r0);
        tma_load_2d(sV, &a.qkv_map, &full[stage], (a.n_q_heads + a.n_kv_heads + kv0) * DH, r0);
        tma_load_2d(sV + 8192, &a.qkv_map, &full[stage], (a.n_q_heads + a.n_kv_heads + kv1) * DH, r0);
        if (++stage == 2) { stage = 0; phase ^= 1; }
      }
    }
  } else if (wg == 1) {
    // ================================ MMA issuers (one thread per lane) ================================
    if (active && lane_id == 0) {
      constexpr uint32_t idesc_s = make_idesc_bf16(128, 128);
      constexpr uint32_t idesc_o = make_idesc_bf16(128, DH) | (1u << 16);        // B (= V) is MN-major
      const uint32_t t_s = t_lane, t_p = t_lane + 128, t_o = t_lane + 192;
      int stage = 0; uint32_t phase = 0, it = 0;
      auto issue_s = [&](int st) {
        const uint32_t base = smem_u32(sIt + st * kP64StageBytes);
        const uint64_t adesc = make_smem_desc_sw128(base), bdesc = make_smem_desc_sw128(base + 16384);
#pragma unroll
        for (int k = 0; k < 4; ++k) umma_bf16(t_s, adesc + 2 * k, bdesc + 2 * k, idesc_s, k != 0);
        umma_commit(&s_full);
      };
      if (item0 < total_items) {
        mbar_wait(&full[0], 0);
        tc_fence_after();
        issue_s(0);
      }
      for (int idx = item0; idx < total_items; idx += item_step, ++it) {
        const int nstage = stage ^ 1; const uint32_t nphase = stage == 1 ? phase ^ 1 : phase;
        mbar_wait(&p_ready, it & 1);                         // P_it sits in TMEM (so S_it has been read); O_(it-1) has been read out
        tc_fence_after();
        const uint32_t va = smem_u32(sIt + stage * kP64StageBytes + 32768);
#pragma unroll
        for (int k = 0; k < 8; ++k) umma_bf16_ts(t_o, t_p + 8 * k, make_smem_desc_sw128_mn(va + k * 2048, 8192), idesc_o, k != 0);
        umma_commit(&empty[stage]);
        umma_commit(&o_full);
        if (idx + item_step < total_items) {
          mbar_wait(&full[nstage], nphase);
          tc_fence_after();
          issue_s(nstage);
        }
        stage = nstage; phase = nphase;
      }
    }
  } else if (active) {
    // ================================ softmax warpgroups (one per lane) ================================
    const int quad = warp & 3;
    const int r_in_tile = quad * 32 + lane_id;
    const int hb = quad >> 1;                                 // which head of the pair this warp's rows belong to
    const int qpos = r_in_tile & 63;                          // position within the request
    const int warp_pos_lo = (quad & 1) * 32;
    const uint32_t t_row = t_lane + (uint32_t(quad * 32) << 16);
    const uint32_t t_s = t_row + hb * 64, t_p = t_row + 128, t_o = t_row + 192;
    uint32_t it = 0;
    for (int idx = item0; idx < total_items; idx += item_step, ++it) {
      const int p = a.reverse ? a.n_req - 1 - idx / n_hp : idx / n_hp, h0 = (idx % n_hp) * 2;
      const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
      const bool warp_valid = warp_pos_lo < n;                // else no query of this warp exists: barriers only
      uint32_t v[64];
      mbar_wait(&s_full, it & 1);
      tc_fence_after();
      if (warp_valid) {
        tmem_ld_32x32(t_s, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tmem_ld_32x32(t_s + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tmem_ld_wait();
      }
      float l_sum = 1.0f;
      if (warp_valid) {
        if (n < 64 || a.causal) {
          const int lim = a.causal ? min(n, qpos + 1) : n;    // keys [0, lim) are visible to this row (lim >= 1)
#pragma unroll
          for (int c = 0; c < 64; ++c)
            if (c >= lim) v[c] = 0xff800000u;                  // -inf
        }
        float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
        for (int c = 0; c < 64; ++c) mx4[c & 3] = fmaxf(mx4[c & 3], __uint_as_float(v[c]));
        const float m = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * -a.scale_log2;   // key 0 is always visible: finite
        float rs4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        uint32_t pk[32], zero[32];
#pragma unroll
        for (int c = 0; c < 64; c += 2) {
          const float p0 = fast_exp2(fmaf(__uint_as_float(v[c]), a.scale_log2, m));
          const float p1 = fast_exp2(fmaf(__uint_as_float(v[c + 1]), a.scale_log2, m));
          rs4[(c >> 1) & 3] += p0 + p1;
          pk[c >> 1] = pack_bf16(p0, p1);
        }
        l_sum = (rs4[0] + rs4[1]) + (rs4[2] + rs4[3]);
#pragma unroll
        for (int c = 0; c < 32; ++c) zero[c] = 0u;
        tmem_st_32x32(t_p + hb * 32, pk);                     // this head's 64 keys
        tmem_st_32x32(t_p + (hb ^ 1) * 32, zero);             // the other head's keys contribute nothing
        tmem_st_wait();
      }
      tc_fence_before();
      __syncwarp();
      if (lane_id == 0) mbar_arrive(&p_ready);
      // ---- O / l -> bf16 -> global ----
      mbar_wait(&o_full, it & 1);
      tc_fence_after();
      if (warp_valid) {
        const float inv = 1.0f / l_sum;
        __nv_bfloat16 *dst = a.out + (size_t)(r0 + qpos) * a.ld_out + (h0 + hb) * DH;
#pragma unroll 1
        for (int c = 0; c < DH; c += 32) {
          uint32_t o[32];
          tmem_ld_32x32(t_o + c, o);
          tmem_ld_wait();
          if (qpos < n) {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              reinterpret_cast<uint4 *>(dst + c)[e] =
                  make_uint4(pack_bf16(__uint_as_float(o[8 * e]) * inv, __uint_as_float(o[8 * e + 1]) * inv),
                             pack_bf16(__uint_as_float(o[8 * e + 2]) * inv, __uint_as_float(o[8 * e + 3]) * inv),
                             pack_bf16(__uint_as_float(o[8 * e + 4]) * inv, __uint_as_float(o[8 * e + 5]) * inv),
                             pack_bf16(__uint_as_float(o[8 * e + 6]) * inv, __uint_as_float(o[8 * e + 7]) * inv));
          }
        }
      }
      tc_fence_before();
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc(tmem_base, 512);
}

}  // namespace fmx
