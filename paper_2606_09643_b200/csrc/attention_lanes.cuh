// Fused variable-length attention on tcgen05 / TMEM / TMA (S3d), persistent multi-lane version.
//   o = softmax(q k^T / sqrt(d_h) + mask) v   per request and query head, online softmax in fp32,
//   GQA (query head g reads KV head g / (H_q / H_kv)), optional causal mask.
// q, k, v live in the fused bf16 buffer [N, (H_q + 2 H_kv) d_h] (task-sorted packed rows, request p owns rows
// cu_tok[p] .. cu_tok[p+1]); output bf16 [N, H_q d_h].
//
// Why lanes.  A kernel using tcgen05 gets ONE resident CTA per SM (the driver reserves the SM's TMEM for it), and one
// softmax warp per scheduler runs at ~0.2 IPC on its dependent max / exp2 / sum chain (profiles/r1_03).  So the
// parallelism that co-resident CTAs would give is built into one persistent CTA per SM: kLanes independent pipelines,
// each with its own producer warp, MMA-issuer warp, softmax warpgroup, TMEM columns and shared-memory ring, each
// walking its own stream of work items (request, query head, 128-query tile).  The tensor core and the four warp
// schedulers interleave the lanes; launch, TMEM allocation and the first-load latency are paid once per SM, and a
// lane's producer prefetches the next item's Q / K / V under the current item's tail.
//
// Per lane, per 64-key tile j of an item:
//   S  = Q K_j^T          tcgen05.mma M=128 N=64(or 16 for a short tail) K=d_h, A = Q, B = K_j (smem, K-major) -> TMEM
//   P  = exp2(S c - m)    softmax warpgroup, thread = query row = TMEM lane (no shuffles); bf16 pairs written back
//                         over S's own TMEM columns with tcgen05.st
//   O += P V_j            tcgen05.mma M=128 N=d_h K=64, A = P (TMEM), B = V_j (smem, MN-major as TMA delivers it)
// The reference maximum m moves lazily (only when a tile maximum exceeds it by > 2^8); only then is O rescaled in TMEM.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "attention_tc.cuh"
#include "ptx.cuh"

namespace fmx {

struct AttnLaneArgs {
  CUtensorMap qkv_map;           // [N, d_qkv] bf16, box {64 columns, 64 rows}, 128B swizzle
  __nv_bfloat16 *out;
  const int *cu_tok;
  int ld_out;
  int n_req, n_q_heads, n_kv_heads;
  int n_qt_max;                  // ceil(max_len / 128)
  int causal;
  float scale_log2;              // log2(e) / sqrt(d_h)
};

constexpr int kLaneCuCap = 1024;        // requests whose cu_tok is staged in shared memory (else read from global)

template <int DH, int kLanes>
__host__ __device__ constexpr int attn_lane_bytes() { return (DH / 64) * (16384 + 4 * 8192); }   // Q + 2 K + 2 V stages
template <int DH, int kLanes>
constexpr int attn_lanes_smem_bytes() { return kLanes * attn_lane_bytes<DH, kLanes>() + 1024 + 1024 + kLaneCuCap * 4; }
template <int kLanes>
constexpr int attn_lanes_threads() { return 256 + 128 * kLanes; }

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
template <int kRegs>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(kRegs)); }
template <int kRegs>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(kRegs)); }

// One work item of a lane: (request, head, q-tile) decoded from the lane's linear item index.
struct AttnItem {
  int r0, n, q0, head, nkv;      // first row of the request, its length, first query row of the tile, KV tiles to visit
};


// One (128-query x NC-key) tile of the online softmax for the calling thread's row: S (fp32, TMEM columns [0, NC)) ->
// P = exp2(S c - m_ref) as bf16 pairs into TMEM columns [0, NC/2); updates m_ref / l_run; rescales O when m_ref moves.
template <int NC, int DH>
__device__ __forceinline__ void attn_softmax_tile(uint32_t t_s, uint32_t t_o, int key0, int lim, bool need_mask, bool first,
                                                  float scale_log2, float &m_ref, float &l_run) {
  uint32_t v[NC];
  if constexpr (NC == 64) {
    tmem_ld_32x32(t_s, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
    tmem_ld_32x32(t_s + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
  } else {
    tmem_ld_32x16(t_s, *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
  }
  tmem_ld_wait();
  if (need_mask) {
#pragma unroll
    for (int c = 0; c < NC; ++c)
      if (key0 + c >= lim) v[c] = 0xff800000u;                     // -inf
  }
  float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
  for (int c = 0; c < NC; ++c) mx4[c & 3] = fmaxf(mx4[c & 3], __uint_as_float(v[c]));
  const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * scale_log2;     // scale > 0; -inf stays -inf
  float factor = 1.0f;
  bool rescale = false;
  if (first) {
    m_ref = (mx == -INFINITY) ? 0.0f : mx;
  } else if (mx > m_ref + 8.0f) {
    factor = fast_exp2(m_ref - mx);
    m_ref = mx;
    rescale = true;
  }
  if (!first && __any_sync(0xffffffffu, rescale)) {               // O is quiescent: s_full implied PV_(j-1) done
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
  float rs4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
  uint32_t pk[NC / 2];
#pragma unroll
  for (int c = 0; c < NC; c += 2) {
    const float p0 = fast_exp2(fmaf(__uint_as_float(v[c]), scale_log2, -m_ref));
    const float p1 = fast_exp2(fmaf(__uint_as_float(v[c + 1]), scale_log2, -m_ref));
    rs4[(c >> 1) & 3] += p0 + p1;
    pk[c >> 1] = pack_bf16(p0, p1);
  }
  l_run = l_run * factor + ((rs4[0] + rs4[1]) + (rs4[2] + rs4[3]));
  if constexpr (NC == 64) tmem_st_32x32(t_s, pk);
  else tmem_st_32x8(t_s, pk);
  tmem_st_wait();
}

template <int DH, int kLanes>
__global__ void __launch_bounds__(256 + 128 * kLanes, 1) attention_lanes_kernel(const __grid_constant__ AttnLaneArgs a) {
  constexpr int kKB = DH / 64;                        // 64-column blocks of the head
  constexpr int kQBytes = kKB * 16384, kKVBytes = kKB * 8192;
  constexpr int kLaneBytes = attn_lane_bytes<DH, kLanes>();
  constexpr int kLaneCols = 64 + DH;                  // TMEM columns of a lane: [S / P : 64][O : DH]
  static_assert(kLanes * kLaneCols <= 512, "TMEM budget");
  constexpr int kBarsPerLane = 11;                    // q_full q_empty k_full[2] k_empty[2] v_full[2] v_empty[2] s_full p_ready o_full -> 13
  (void)kBarsPerLane;
  extern __shared__ uint8_t al_smem_raw[];
  const uint32_t pad = (1024u - (smem_u32(al_smem_raw) & 1023u)) & 1023u;
  uint8_t *tiles = al_smem_raw + pad;
  uint64_t *bars = reinterpret_cast<uint64_t *>(tiles + kLanes * kLaneBytes);          // 13 per lane
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 13 * kLanes);
  int *s_cu = reinterpret_cast<int *>(tiles + kLanes * kLaneBytes + 1024);

  const int warp = threadIdx.x >> 5, lane_id = threadIdx.x & 31;
  const int wg = warp >> 2;                                                            // 0 producers, 1 MMA issuers, 2.. softmax
  const bool cu_in_smem = a.n_req < kLaneCuCap;
  griddep_launch();
  griddep_wait();
  if (cu_in_smem)
    for (int i = threadIdx.x; i <= a.n_req; i += blockDim.x) s_cu[i] = a.cu_tok[i];
  const int *cu = cu_in_smem ? s_cu : a.cu_tok;

  if (threadIdx.x == 0) {
    for (int l = 0; l < kLanes; ++l) {
      uint64_t *b = bars + 13 * l;
      for (int i = 0; i < 10; ++i) mbar_init(&b[i], 1);       // q_full q_empty k_full[2] k_empty[2] v_full[2] v_empty[2]
      mbar_init(&b[10], 1);                                   // s_full  (tcgen05.commit)
      mbar_init(&b[11], 4);                                   // p_ready (one arrive per softmax warp)
      mbar_init(&b[12], 1);                                   // o_full  (tcgen05.commit)
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
  if constexpr (kLanes == 4) {                       // 768 threads: 80 registers each at launch
    if (wg < 2) setmaxnreg_dec<40>();
    else setmaxnreg_inc<96>();
  }

  // ---- the lane this warp serves and its resources ----
  const int lane = wg == 0 ? warp : (wg == 1 ? warp - 4 : wg - 2);
  const bool active = lane < kLanes;
  uint8_t *sQ = tiles + (active ? lane : 0) * kLaneBytes, *sK = sQ + kQBytes, *sV = sK + 2 * kKVBytes;
  uint64_t *lb = bars + 13 * (active ? lane : 0);
  uint64_t &q_full = lb[0], &q_empty = lb[1];
  uint64_t *k_full = lb + 2, *k_empty = lb + 4, *v_full = lb + 6, *v_empty = lb + 8;
  uint64_t &s_full = lb[10], &p_ready = lb[11], &o_full = lb[12];
  const uint32_t t_lane = tmem_base + lane * kLaneCols;

  const int per_level = a.n_req * a.n_q_heads;
  const int total_items = a.n_qt_max * per_level;
  const int item0 = blockIdx.x * kLanes + lane, item_step = gridDim.x * kLanes;
  const int group = a.n_q_heads / a.n_kv_heads;
  // item index -> (request, head, q-tile); late (for causal: heavy) q-tiles first.  false = the tile is past the request's end.
  auto decode = [&](int idx, AttnItem &it) {
    const int lvl = idx / per_level, rem = idx - lvl * per_level;
    const int p = rem / a.n_q_heads;
    it.head = rem - p * a.n_q_heads;
    it.q0 = (a.n_qt_max - 1 - lvl) * kAtBQ;
    it.r0 = cu[p];
    it.n = cu[p + 1] - it.r0;
    if (it.q0 >= it.n) return false;
    const int kv_end = a.causal ? min(it.n, it.q0 + kAtBQ) : it.n;
    it.nkv = (kv_end + kAtBKV - 1) / kAtBKV;
    return true;
  };
  // columns of KV tile j that take part: 16 when the last tile holds <= 16 keys, else 64
  auto tile_cols = [&](const AttnItem &it, int j) {
    const int kv_end = a.causal ? min(it.n, it.q0 + kAtBQ) : it.n;
    return (j == it.nkv - 1 && kv_end - j * kAtBKV <= 16) ? 16 : 64;
  };

  if (wg == 0) {
    // ================================ TMA producers (one thread per lane) ================================
    if (active && lane_id == 0) {
      tma_prefetch_desc(&a.qkv_map);
      int stage = 0; uint32_t phase = 0, qphase = 0;
      AttnItem it;
      for (int idx = item0; idx < total_items; idx += item_step) {
        if (!decode(idx, it)) continue;
        const int kvh = it.head / group;
        const int col_q = it.head * DH, col_k = (a.n_q_heads + kvh) * DH, col_v = (a.n_q_heads + a.n_kv_heads + kvh) * DH;
        mbar_wait(&q_empty, qphase ^ 1);
        mbar_arrive_expect_tx(&q_full, kQBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb)
#pragma unroll
          for (int h = 0; h < 2; ++h)
            tma_load_2d(sQ + kb * 16384 + h * 8192, &a.qkv_map, &q_full, col_q + kb * 64, it.r0 + it.q0 + h * 64);
        qphase ^= 1;
        for (int j = 0; j < it.nkv; ++j) {
          const int row = it.r0 + j * kAtBKV;
          mbar_wait(&k_empty[stage], phase ^ 1);
          mbar_arrive_expect_tx(&k_full[stage], kKVBytes);
#pragma unroll
          for (int kb = 0; kb < kKB; ++kb) tma_load_2d(sK + stage * kKVBytes + kb * 8192, &a.qkv_map, &k_full[stage], col_k + kb * 64, row);
          mbar_wait(&v_empty[stage], phase ^ 1);
          mbar_arrive_expect_tx(&v_full[stage], kKVBytes);
#pragma unroll
          for (int kb = 0; kb < kKB; ++kb) tma_load_2d(sV + stage * kKVBytes + kb * 8192, &a.qkv_map, &v_full[stage], col_v + kb * 64, row);
          if (++stage == 2) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (wg == 1) {
    // ================================ MMA issuers (one thread per lane) ================================
    if (active && lane_id == 0) {
      constexpr uint32_t idesc_s64 = make_idesc_bf16(kAtBQ, 64), idesc_s16 = make_idesc_bf16(kAtBQ, 16);
      constexpr uint32_t idesc_o = make_idesc_bf16(kAtBQ, DH) | (1u << 16);      // B (= V) is MN-major
      const uint32_t t_s = t_lane, t_o = t_lane + 64;
      int stage = 0; uint32_t phase = 0, qphase = 0, step = 0;
      auto issue_s = [&](int st, int cols) {
        const uint32_t qa = smem_u32(sQ), ka = smem_u32(sK + st * kKVBytes);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) {
          const uint64_t adesc = make_smem_desc_sw128(qa + kb * 16384), bdesc = make_smem_desc_sw128(ka + kb * 8192);
#pragma unroll
          for (int k = 0; k < 4; ++k) umma_bf16(t_s, adesc + 2 * k, bdesc + 2 * k, cols == 64 ? idesc_s64 : idesc_s16, (kb | k) != 0);
        }
        umma_commit(&s_full);
        umma_commit(&k_empty[st]);
      };
      AttnItem it;
      for (int idx = item0; idx < total_items; idx += item_step) {
        if (!decode(idx, it)) continue;
        mbar_wait(&q_full, qphase);
        qphase ^= 1;
        mbar_wait(&k_full[stage], phase);
        tc_fence_after();
        issue_s(stage, tile_cols(it, 0));
        if (it.nkv == 1) umma_commit(&q_empty);
        for (int j = 0; j < it.nkv; ++j) {
          int nstage = stage + 1; uint32_t nphase = phase;
          if (nstage == 2) { nstage = 0; nphase ^= 1; }
          mbar_wait(&p_ready, step & 1);               // P_j sits in TMEM (over S_j), O rescaled if it had to be
          ++step;
          mbar_wait(&v_full[stage], phase);
          tc_fence_after();
          const uint32_t va = smem_u32(sV + stage * kKVBytes);
          const int ksteps = tile_cols(it, j) >> 4;
          for (int k = 0; k < ksteps; ++k)
            umma_bf16_ts(t_o, t_s + 8 * k, make_smem_desc_sw128_mn(va + k * 2048, 8192), idesc_o, (j | k) != 0);
          umma_commit(&v_empty[stage]);
          if (j + 1 < it.nkv) {
            mbar_wait(&k_full[nstage], nphase);
            tc_fence_after();
            issue_s(nstage, tile_cols(it, j + 1));       // in pipe order after PV_j has read P_j
            if (j + 2 == it.nkv) umma_commit(&q_empty);
          } else {
            umma_commit(&o_full);
          }
          stage = nstage; phase = nphase;
        }
      }
    }
  } else if (active) {
    // ================================ softmax warpgroups (one per lane) ================================
    const int quad = warp & 3;
    const int r_in_tile = quad * 32 + lane_id;
    const uint32_t t_s = t_lane + (uint32_t(quad * 32) << 16), t_o = t_s + 64;
    uint32_t step = 0, iphase = 0;
    AttnItem it;
    for (int idx = item0; idx < total_items; idx += item_step) {
      if (!decode(idx, it)) continue;
      const int qrow = it.q0 + r_in_tile;                          // position within the request
      const int warp_row_lo = it.q0 + quad * 32;
      const bool warp_valid = warp_row_lo < it.n;                  // else: no query of this warp exists
      const int lim = a.causal ? min(it.n, qrow + 1) : it.n;       // keys [0, lim) are visible to this row
      float m_ref = 0.0f, l_run = 0.0f;
      for (int j = 0; j < it.nkv; ++j) {
        const int cols = tile_cols(it, j);
        mbar_wait(&s_full, step & 1);                              // also: PV_(j-1) has completed
        ++step;
        if (warp_valid) {
          tc_fence_after();
          const int key0 = j * kAtBKV;
          const bool need_mask = key0 + cols > it.n || (a.causal && key0 + cols - 1 > warp_row_lo);
          if (cols == 64) attn_softmax_tile<64, DH>(t_s, t_o, key0, lim, need_mask, j == 0, a.scale_log2, m_ref, l_run);
          else attn_softmax_tile<16, DH>(t_s, t_o, key0, lim, need_mask, j == 0, a.scale_log2, m_ref, l_run);
          tc_fence_before();
        }
        __syncwarp();
        if (lane_id == 0) mbar_arrive(&p_ready);
      }
      // ---- O / l -> bf16 -> global ----
      if (warp_valid) {
        mbar_wait(&o_full, iphase);
        tc_fence_after();
        const float inv = 1.0f / l_run;
        __nv_bfloat16 *dst = a.out + (size_t)(it.r0 + qrow) * a.ld_out + it.head * DH;
#pragma unroll 1
        for (int c = 0; c < DH; c += 32) {
          uint32_t o[32];
          tmem_ld_32x32(t_o + c, o);
          tmem_ld_wait();
          if (qrow < it.n) {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              reinterpret_cast<uint4 *>(dst + c)[e] =
                  make_uint4(pack_bf16(__uint_as_float(o[8 * e]) * inv, __uint_as_float(o[8 * e + 1]) * inv),
                             pack_bf16(__uint_as_float(o[8 * e + 2]) * inv, __uint_as_float(o[8 * e + 3]) * inv),
                             pack_bf16(__uint_as_float(o[8 * e + 4]) * inv, __uint_as_float(o[8 * e + 5]) * inv),
                             pack_bf16(__uint_as_float(o[8 * e + 6]) * inv, __uint_as_float(o[8 * e + 7]) * inv));
          }
        }
        tc_fence_before();
      }
      iphase ^= 1;
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc(tmem_base, 512);
}
}  // namespace fmx
