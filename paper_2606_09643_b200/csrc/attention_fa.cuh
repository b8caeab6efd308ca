// Fused variable-length attention on tcgen05 / TMEM / TMA (S3d) for sequences longer than one KV tile, head_dim 64 / 128:
//   o = softmax(q k^T / sqrt(d_h) + mask) v   per request and query head, online softmax in fp32,
//   GQA (query head g reads KV head g / (H_q / H_kv)), optional causal mask.
// q, k, v live in the fused bf16 buffer [N, (H_q + 2 H_kv) d_h] (task-sorted packed rows, request p owns rows
// cu_tok[p] .. cu_tok[p+1]); output bf16 [N, H_q d_h].
//
// What bounds this step (ncu, profiles/r2_*): not the tensor pipe and not DRAM but the softmax - 64 ex2 per row and KV tile
// on the 16-lane MUFU, plus the latency of every S -> softmax -> PV hand-off.  The design therefore (a) packs as many
// independent q-tiles onto an SM as its TMEM, shared memory and registers allow (head_dim 64: FOUR 192-thread CTAs per SM),
// (b) keeps a CTA light so that this holds - P goes back to TMEM over S's own columns (no P tile in shared memory, no
// proxy fence), the softmax walks S in 32-column chunks (few live registers), no idle warps - and (c) computes nothing that
// is not there: a last KV tile of <= 16 keys runs as an N = 16 MMA and a 16-column softmax, warps whose 32 query rows do
// not exist only keep the barrier protocol going.
//
// One CTA = (request, query head, 128-query tile).  Per 64-key tile j:
//   S  = Q K_j^T          tcgen05.mma M=128 N=64|16 K=d_h, A = Q, B = K_j (smem, K-major) -> TMEM
//   P  = exp2(S c - m)    softmax warpgroup, thread = query row = TMEM lane (no shuffles); bf16 pairs written back over S's
//                         own TMEM columns with tcgen05.st
//   O += P V_j            tcgen05.mma M=128 N=d_h K=64|16, A = P (TMEM), B = V_j (smem, MN-major as TMA delivers it)
// kSBuf = 2 (head_dim 128: TMEM holds 2 x 64 + 128 = 256 columns) double-buffers S so that S_(j+1) runs under softmax_j;
// kSBuf = 1 (head_dim 64: 64 + 64 = 128 columns, four CTAs per SM) issues S_(j+1) in pipe order behind PV_j and lets the
// co-resident CTAs fill the gap.  The reference maximum m moves lazily (only when a tile maximum exceeds it by > 2^8); only
// then is O rescaled in TMEM.
//
// Warp roles (192 threads): warp 0 TMA producer, warp 1 TMEM allocator + tcgen05.mma issuer, warps 2..5 softmax (warp w
// owns TMEM lanes 32 (w & 3) ..).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

namespace fmx {

constexpr int kAtBQ = 128;       // queries per q-tile (TMEM lanes)
constexpr int kAtBKV = 64;       // keys per KV tile
constexpr int kFaThreads = 192;
constexpr int kFaStages = 2;     // K / V ring depth

struct AttnTcArgs {
  CUtensorMap qkv_map;           // [N, d_qkv] bf16, box {64 columns, 64 rows}, 128B swizzle
  __nv_bfloat16 *out;
  const int *cu_tok;
  int ld_out;
  int n_q_heads, n_kv_heads;
  int causal;
  float scale_log2;              // log2(e) / sqrt(d_h)
  int reverse;                   // 1: requests are walked from the last to the first (blockIdx.z reversed)
  // kBias instantiations only: relative-position bias by distance, relb[head * relb_ld + (key - query) + relb_off], times log2(e);
  // the table is padded so that the padding rows / keys of a tile index inside it
  const float *relb;
  int relb_ld, relb_off;
};

template <int DH>
__host__ __device__ constexpr int attn_fa_tile_bytes() { return (DH / 64) * (16384 + 2 * kFaStages * 8192); }
template <int DH>
constexpr int attn_fa_smem_bytes() { return attn_fa_tile_bytes<DH>() + 1024; }

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
// D[tmem] (+)= A[tmem] * B[smem]^T : A = bf16 pairs in TMEM (lane = row, 32-bit column c = elements 2c, 2c+1)
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_st_32x8(uint32_t taddr, const uint32_t (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};\n" ::"r"(taddr), "r"(v[0]),
               "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
               : "memory");
}
__device__ __forceinline__ void tmem_st_32x16(uint32_t taddr, const uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};\n" ::"r"(taddr),
      "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]),
      "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
      : "memory");
}
// 32 (or 16) score columns of the calling thread's row -> their maximum, four independent chains.
template <int NC>
__device__ __forceinline__ float fa_chunk_max(uint32_t (&v)[NC], int key0, int lim, bool need_mask) {
  if (need_mask) {
#pragma unroll
    for (int c = 0; c < NC; ++c)
      if (key0 + c >= lim) v[c] = 0xff800000u;                     // -inf
  }
  float m4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
  for (int c = 0; c < NC; ++c) m4[c & 3] = fmaxf(m4[c & 3], __uint_as_float(v[c]));
  return fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
}
// kBias: raw scores -> scores in the log2 domain with the relative-position bias of the row added (rel = the row's table entry for
// the chunk's first key); the maximum / exponent steps then run with a scale of 1.
template <int NC>
__device__ __forceinline__ void fa_chunk_bias(uint32_t (&v)[NC], float scale_log2, const float *__restrict__ rel) {
#pragma unroll
  for (int c = 0; c < NC; ++c) v[c] = __float_as_uint(fmaf(__uint_as_float(v[c]), scale_log2, __ldg(rel + c)));
}
// ... -> P = exp2(S c - m_ref) as NC / 2 packed bf16 pairs; returns the row sum of the chunk.
template <int NC>
__device__ __forceinline__ float fa_chunk_exp(const uint32_t (&v)[NC], uint32_t (&pk)[NC / 2], float scale_log2, float m_ref) {
  float r4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
  for (int c = 0; c < NC; c += 2) {
    const float p0 = fast_exp2(fmaf(__uint_as_float(v[c]), scale_log2, -m_ref));
    const float p1 = fast_exp2(fmaf(__uint_as_float(v[c + 1]), scale_log2, -m_ref));
    r4[(c >> 1) & 3] += p0 + p1;
    pk[c >> 1] = pack_bf16(p0, p1);
  }
  return (r4[0] + r4[1]) + (r4[2] + r4[3]);
}

template <int DH, int kSBuf, int kMinBlocks, bool kOnePass, bool kBias = false>
__global__ void __launch_bounds__(kFaThreads, kMinBlocks) attention_fa_kernel(const __grid_constant__ AttnTcArgs a) {
  constexpr int kKB = DH / 64;                        // 64-column blocks of the head
  constexpr int kQBytes = kKB * 16384;                // the q-tile
  constexpr int kKVBytes = kKB * 8192;                // one K (or V) tile
  constexpr uint32_t kTmemUsed = kSBuf * 64 + DH;     // [S / P : 64] x kSBuf, [O : DH]
  constexpr uint32_t kTmemCols = kTmemUsed <= 128 ? 128 : 256;      // the allocation is a power of two
  static_assert(kTmemUsed <= 256, "TMEM budget");
  extern __shared__ uint8_t fa_smem_raw[];
  const uint32_t raw_addr = smem_u32(fa_smem_raw);
  const uint32_t pad = (1024u - (raw_addr & 1023u)) & 1023u;
  uint8_t *smem = fa_smem_raw + pad;
  uint8_t *sQ = smem;
  uint8_t *sK = sQ + kQBytes;
  uint8_t *sV = sK + kFaStages * kKVBytes;
  // barriers (<= 128 bytes) live in the alignment slack: before the tiles when the pad is large enough, else after them
  constexpr int kTileBytes = attn_fa_tile_bytes<DH>();
  uint64_t *bars = reinterpret_cast<uint64_t *>(pad >= 128 ? fa_smem_raw + ((pad - 128) & ~7u) : smem + kTileBytes);
  uint64_t &q_full = bars[0];
  uint64_t *k_full = bars + 1, *k_empty = k_full + kFaStages, *v_full = k_empty + kFaStages, *v_empty = v_full + kFaStages;
  uint64_t *s_full = v_empty + kFaStages;             // [kSBuf]
  // one p_ready barrier per S buffer: with a single one a softmax warp that runs ahead into tile j + 1 (its S is already there
  // when S is double-buffered) would complete phase j with its second arrival
  uint64_t *p_ready = s_full + kSBuf;                 // [kSBuf]
  // pv_done: one phase per PV (the rare O rescale of tile j waits for PV_(j-1): at that point at most one phase is pending);
  // o_full: completes once, after the LAST PV - the epilogue cannot use pv_done, a fast tail tile may be two phases ahead
  uint64_t &pv_done = s_full[2 * kSBuf], &o_full = s_full[2 * kSBuf + 1];
  uint32_t &tmem_base_slot = *reinterpret_cast<uint32_t *>(&s_full[2 * kSBuf + 2]);
  static_assert((1 + 4 * kFaStages + 2 * kSBuf + 2) * 8 + 4 <= 128, "barrier block");

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int p = a.reverse ? (int)gridDim.z - 1 - (int)blockIdx.z : (int)blockIdx.z, head = blockIdx.y;
  griddep_launch();
  griddep_wait();
  const int r0 = a.cu_tok[p], n = a.cu_tok[p + 1] - r0;
  const int q0 = ((int)gridDim.x - 1 - (int)blockIdx.x) * kAtBQ;       // heavy (late) causal tiles first
  if (q0 >= n) return;
  const int kvh = head / (a.n_q_heads / a.n_kv_heads);
  const int col_q = head * DH, col_k = (a.n_q_heads + kvh) * DH, col_v = (a.n_q_heads + a.n_kv_heads + kvh) * DH;
  const int kv_end = a.causal ? min(n, q0 + kAtBQ) : n;               // keys [0, kv_end) are visible to some row of the tile
  const int nkv = (kv_end + kAtBKV - 1) / kAtBKV;
  const int tail_cols = (kv_end - (nkv - 1) * kAtBKV <= 16) ? 16 : 64;  // columns of the LAST KV tile that take part

  if (threadIdx.x == 0) {
    mbar_init(&q_full, 1);
    for (int s = 0; s < kFaStages; ++s) { mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], 1); mbar_init(&v_full[s], 1); mbar_init(&v_empty[s], 1); }
    for (int s = 0; s < kSBuf; ++s) { mbar_init(&s_full[s], 1); mbar_init(&p_ready[s], 4); }
    mbar_init(&pv_done, 1);
    mbar_init(&o_full, 1);
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(&tmem_base_slot, kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_slot;
  const uint32_t tm_o = tmem_base + kSBuf * 64;

  if (warp == 0) {
    // ================================ TMA producer ================================
    if (lane == 0) {
      tma_prefetch_desc(&a.qkv_map);
      mbar_arrive_expect_tx(&q_full, kQBytes);
#pragma unroll
      for (int kb = 0; kb < kKB; ++kb)
#pragma unroll
        for (int h = 0; h < 2; ++h)
          tma_load_2d(sQ + kb * 16384 + h * 8192, &a.qkv_map, &q_full, col_q + kb * 64, r0 + q0 + h * 64);
      int stage = 0; uint32_t phase = 0;
      for (int j = 0; j < nkv; ++j) {
        const int row = r0 + j * kAtBKV;
        mbar_wait(&k_empty[stage], phase ^ 1);
        mbar_arrive_expect_tx(&k_full[stage], kKVBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) tma_load_2d(sK + stage * kKVBytes + kb * 8192, &a.qkv_map, &k_full[stage], col_k + kb * 64, row);
        mbar_wait(&v_empty[stage], phase ^ 1);
        mbar_arrive_expect_tx(&v_full[stage], kKVBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) tma_load_2d(sV + stage * kKVBytes + kb * 8192, &a.qkv_map, &v_full[stage], col_v + kb * 64, row);
        if (++stage == kFaStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ================================ MMA issuer ================================
    if (lane == 0) {
      constexpr uint32_t idesc_s64 = make_idesc_bf16(kAtBQ, 64), idesc_s16 = make_idesc_bf16(kAtBQ, 16);
      constexpr uint32_t idesc_o = make_idesc_bf16(kAtBQ, DH) | (1u << 16);      // B (= V) is MN-major
      auto cols_of = [&](int j) { return j == nkv - 1 ? tail_cols : 64; };
      auto issue_s = [&](int j, int st) {
        const uint32_t qa = smem_u32(sQ), ka = smem_u32(sK + st * kKVBytes);
        const uint32_t t_s = tmem_base + (kSBuf == 2 ? (j & 1) * 64 : 0);
        const uint32_t idesc = cols_of(j) == 64 ? idesc_s64 : idesc_s16;
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) {
          const uint64_t adesc = make_smem_desc_sw128(qa + kb * 16384), bdesc = make_smem_desc_sw128(ka + kb * 8192);
#pragma unroll
          for (int k = 0; k < 4; ++k) umma_bf16(t_s, adesc + 2 * k, bdesc + 2 * k, idesc, (kb | k) != 0);
        }
        umma_commit(&s_full[kSBuf == 2 ? (j & 1) : 0]);
        umma_commit(&k_empty[st]);
      };
      mbar_wait(&q_full, 0);
      mbar_wait(&k_full[0], 0);
      tc_fence_after();
      issue_s(0, 0);
      int stage = 0; uint32_t phase = 0;
      for (int j = 0; j < nkv; ++j) {
        int nstage = stage + 1; uint32_t nphase = phase;
        if (nstage == kFaStages) { nstage = 0; nphase ^= 1; }
        if (kSBuf == 2 && j + 1 < nkv) {               // S_(j+1) into the other buffer, under softmax_j (its P_(j-1) was read by
          mbar_wait(&k_full[nstage], nphase);          // PV_(j-1), issued before this in pipe order)
          tc_fence_after();
          issue_s(j + 1, nstage);
        }
        mbar_wait(&p_ready[kSBuf == 2 ? (j & 1) : 0], kSBuf == 2 ? ((j >> 1) & 1) : (j & 1));   // P_j sits in TMEM (over S_j), O rescaled if it had to be
        mbar_wait(&v_full[stage], phase);
        tc_fence_after();
        const uint32_t t_p = tmem_base + (kSBuf == 2 ? (j & 1) * 64 : 0);
        const uint32_t va = smem_u32(sV + stage * kKVBytes);
        const int ksteps = cols_of(j) >> 4;
        for (int k = 0; k < ksteps; ++k)
          umma_bf16_ts(tm_o, t_p + 8 * k, make_smem_desc_sw128_mn(va + k * 2048, 8192), idesc_o, (j | k) != 0);
        umma_commit(&v_empty[stage]);
        umma_commit(&pv_done);
        if (j + 1 == nkv) umma_commit(&o_full);
        if (kSBuf == 1 && j + 1 < nkv) {               // same S buffer: in pipe order after PV_j has read P_j
          mbar_wait(&k_full[nstage], nphase);
          tc_fence_after();
          issue_s(j + 1, nstage);
        }
        stage = nstage; phase = nphase;
      }
    }
  } else {
    // ================================ softmax warps ================================
    const int quad = warp & 3;
    const int r_in_tile = quad * 32 + lane;
    const int qrow = q0 + r_in_tile;                                 // position within the request
    const int warp_row_lo = q0 + quad * 32;
    const bool warp_valid = warp_row_lo < n;                         // else: no query of this warp exists
    const uint32_t lane_sel = uint32_t(quad * 32) << 16;
    const uint32_t t_o = tm_o + lane_sel;
    const int lim = a.causal ? min(n, qrow + 1) : n;                 // keys [0, lim) are visible to this row
    float m_ref = 0.0f, l_run = 0.0f;
    const float sc = kBias ? 1.0f : a.scale_log2;                    // kBias: fa_chunk_bias has already scaled the scores
    const float *relrow = kBias ? a.relb + head * a.relb_ld + a.relb_off - qrow : nullptr;    // + key = this row's bias for that key
    for (int j = 0; j < nkv; ++j) {
      const int cols = j == nkv - 1 ? tail_cols : 64;
      const int sb = kSBuf == 2 ? (j & 1) : 0;
      mbar_wait(&s_full[sb], kSBuf == 2 ? ((j >> 1) & 1) : (j & 1));
      if (warp_valid) {
        tc_fence_after();
        const uint32_t t_s = tmem_base + sb * 64 + lane_sel;
        const int key0 = j * kAtBKV;
        const bool need_mask = key0 + cols > n || (a.causal && key0 + cols - 1 > warp_row_lo);
        // the reference maximum moves lazily; when it does, O (quiescent once PV_(j-1) has completed) is rescaled in TMEM
        float factor = 1.0f;
        auto update_ref = [&](float mx) {
          mx *= sc;                                                  // scale > 0; -inf stays -inf
          bool rescale = false;
          if (j == 0) {
            m_ref = (mx == -INFINITY) ? 0.0f : mx;
          } else if (mx > m_ref + 8.0f) {
            factor = fast_exp2(m_ref - mx);
            m_ref = mx;
            rescale = true;
          }
          if (j > 0 && __any_sync(0xffffffffu, rescale)) {
            mbar_wait(&pv_done, (j - 1) & 1);
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
          }
        };
        // P = exp2(S c - m_ref) goes back over S's own columns (chunk c of P lands on columns that S chunks <= c occupied)
        float rs;
        if (cols == 64 && kOnePass) {
          // all 64 scores of the row in registers: one TMEM round trip
          uint32_t v0[32], v1[32], pk[16];
          tmem_ld_32x32(t_s, v0);
          tmem_ld_32x32(t_s + 32, v1);
          tmem_ld_wait();
          if constexpr (kBias) { fa_chunk_bias<32>(v0, a.scale_log2, relrow + key0); fa_chunk_bias<32>(v1, a.scale_log2, relrow + key0 + 32); }
          update_ref(fmaxf(fa_chunk_max<32>(v0, key0, lim, need_mask), fa_chunk_max<32>(v1, key0 + 32, lim, need_mask)));
          rs = fa_chunk_exp<32>(v0, pk, sc, m_ref);
          tmem_st_32x16(t_s, pk);
          rs += fa_chunk_exp<32>(v1, pk, sc, m_ref);
          tmem_st_32x16(t_s + 16, pk);
        } else if (cols == 64) {
          // two passes over S in 32-column chunks: half the live registers, twice the TMEM loads
          uint32_t v[32], pk[16];
          tmem_ld_32x32(t_s, v);
          tmem_ld_wait();
          if constexpr (kBias) fa_chunk_bias<32>(v, a.scale_log2, relrow + key0);
          float mx = fa_chunk_max<32>(v, key0, lim, need_mask);
          tmem_ld_32x32(t_s + 32, v);
          tmem_ld_wait();
          if constexpr (kBias) fa_chunk_bias<32>(v, a.scale_log2, relrow + key0 + 32);
          update_ref(fmaxf(mx, fa_chunk_max<32>(v, key0 + 32, lim, need_mask)));
          rs = fa_chunk_exp<32>(v, pk, sc, m_ref);                   // second chunk first: it is in registers
          tmem_ld_32x32(t_s, v);
          tmem_ld_wait();
          tmem_st_32x16(t_s + 16, pk);
          if constexpr (kBias) fa_chunk_bias<32>(v, a.scale_log2, relrow + key0);
          if (need_mask) fa_chunk_max<32>(v, key0, lim, true);
          rs += fa_chunk_exp<32>(v, pk, sc, m_ref);
          tmem_st_32x16(t_s, pk);
        } else {
          uint32_t v[16], pk[8];
          tmem_ld_32x16(t_s, v);
          tmem_ld_wait();
          if constexpr (kBias) fa_chunk_bias<16>(v, a.scale_log2, relrow + key0);
          update_ref(fa_chunk_max<16>(v, key0, lim, need_mask));
          rs = fa_chunk_exp<16>(v, pk, sc, m_ref);
          tmem_st_32x8(t_s, pk);
        }
        l_run = l_run * factor + rs;
        tmem_st_wait();
        tc_fence_before();
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&p_ready[sb]);
    }
    // ---- O / l -> bf16 -> global ----
    if (warp_valid) {
      mbar_wait(&o_full, 0);
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
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace fmx
