// SRA forward kernel for sm_100a.
//
// One CTA = one work item (a 256-row query slab of G or of one R block) x one (batch, head).
// The slab is two 128-row Q tiles that ping-pong on the tensor core:
//
//   warps 0-3   softmax warpgroup of Q tile 0   (thread = one query row, TMEM lane = row)
//   warps 4-7   softmax warpgroup of Q tile 1
//   warp  8     MMA issuer (one thread): S_i = Q_i K_j^T (SS), O_i += P_i V_j (A = P from TMEM)
//   warp  9     TMA loader (one thread): Q once, then the K/V tile ring
//   warps 10-11 idle (they only pad the third warpgroup for setmaxnreg)
//
// TMEM (512 columns x 128 lanes x fp32): S0 @0, S1 @128, O0 @256, O1 @256+D; P_i (bf16, 64
// columns) aliases the first 64 columns of S_i once the softmax thread holds S_i in registers.
// Masked tiles are never visited: the key-tile loop walks only the item's visible segments;
// only the last tile of a segment pays for a column mask (n_valid < 128).
#include "ptx.cuh"
#include "sra_common.h"

namespace sra {

template <int D>
struct FwdCfg {
  static constexpr int kTileBytes = kTile * D * 2;          // one Q/K/V tile in smem
  static constexpr int kBoxes = D / 64;                      // 64-column (128 B) TMA boxes per tile
  static constexpr int kBoxBytes = kTile * 128;              // 16 KB
  static constexpr int kStages = (D == 128) ? 5 : 10;        // K/V ring depth (tiles)
  static constexpr int kNumBars = 1 + 2 * kStages + 6;
  static constexpr int kSmemBytes = 1024 /*align slack*/ + (2 + kStages) * kTileBytes + kNumBars * 8 + 16;
  static constexpr int kTmemCols = 512;
  static constexpr int kThreads = 384;
};

template <int D>
__device__ __forceinline__ void load_tile(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int row, int h, int b,
                                          bool head_major) {
#pragma unroll
  for (int x = 0; x < FwdCfg<D>::kBoxes; ++x) {
    if (head_major)
      tma_load_4d(dst + x * FwdCfg<D>::kBoxBytes, tm, bar, x * 64, row, h, b);
    else
      tma_load_4d(dst + x * FwdCfg<D>::kBoxBytes, tm, bar, x * 64, h, row, b);
  }
}

template <int D>
__global__ void __launch_bounds__(FwdCfg<D>::kThreads, 1)
    sra_fwd_kernel(const __grid_constant__ CUtensorMap tm_q_gen, const __grid_constant__ CUtensorMap tm_k_gen,
                   const __grid_constant__ CUtensorMap tm_v_gen, const __grid_constant__ CUtensorMap tm_q_ref,
                   const __grid_constant__ CUtensorMap tm_k_ref, const __grid_constant__ CUtensorMap tm_v_ref,
                   const FwdParams p) {
  using C = FwdCfg<D>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base;                         // 2 tiles
  const uint32_t sKV = smem_base + 2 * C::kTileBytes;    // kStages tiles
  const uint32_t sBar = sKV + C::kStages * C::kTileBytes;
  const uint32_t bar_q_full = sBar;
  const uint32_t bar_kv_full = sBar + 8;
  const uint32_t bar_kv_empty = bar_kv_full + 8 * C::kStages;
  const uint32_t bar_s_full = bar_kv_empty + 8 * C::kStages;
  const uint32_t bar_p_full = bar_s_full + 16;
  const uint32_t bar_o_full = bar_p_full + 16;
  const uint32_t s_tmem_ptr = bar_o_full + 16;
  uint32_t* tmem_ptr_generic = reinterpret_cast<uint32_t*>(smem_raw + (s_tmem_ptr - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  const FwdItem item = p.items[blockIdx.x];
  const int h = blockIdx.y;
  const int b = blockIdx.z;
  const int n0 = (item.seg0_len + kTile - 1) / kTile;
  const int n1 = (item.seg1_len + kTile - 1) / kTile;
  const int n_kv = n0 + n1;
  const int n_qt = item.q_rows > kTile ? 2 : 1;  // Q tiles that hold at least one valid row

  if (threadIdx.x == 0) {
    mbar_init(bar_q_full, 1);
    for (int s = 0; s < C::kStages; ++s) {
      mbar_init(bar_kv_full + 8 * s, 1);
      mbar_init(bar_kv_empty + 8 * s, 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_s_full + 8 * i, 1);
      mbar_init(bar_p_full + 8 * i, 128);
      mbar_init(bar_o_full + 8 * i, 1);
    }
    fence_mbar_init();
  }
  if (warp == 9 && lane == 0) {
    tma_prefetch_desc(item.q_is_ref ? &tm_q_ref : &tm_q_gen);
    tma_prefetch_desc(item.seg0_is_ref ? &tm_k_ref : &tm_k_gen);
    tma_prefetch_desc(item.seg0_is_ref ? &tm_v_ref : &tm_v_gen);
  }
  if (warp == 8) tmem_alloc(s_tmem_ptr, C::kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr_generic;
  const uint32_t tS0 = tmem, tO0 = tmem + 256;

  if (warp < 8) {
    // ======================================================= softmax warpgroups
    reg_inc<224>();
    const int i = warp >> 2;  // Q tile of this warpgroup
    if (i < n_qt) {
      const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
      const uint32_t tS = tS0 + i * 128 + lane_off;
      const uint32_t tO = tO0 + i * D + lane_off;
      const float sl2 = p.scale_log2;
      float m_ref = -INFINITY;  // reference max of the raw scores (lazily updated)
      float l = 0.f;            // running sum of exp2((s - m_ref) * sl2)
      for (int j = 0; j < n_kv; ++j) {
        const int n_valid = (j < n0) ? min(kTile, item.seg0_len - j * kTile) : min(kTile, item.seg1_len - (j - n0) * kTile);
        mbar_wait(bar_s_full + 8 * i, j & 1);
        tc_fence_after();
        uint32_t s[4][32];
#pragma unroll
        for (int c = 0; c < 4; ++c) tmem_ld32(tS + c * 32, s[c]);
        tmem_wait_ld();
        if (n_valid < kTile) {
#pragma unroll
          for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int k = 0; k < 32; ++k)
              if (c * 32 + k >= n_valid) s[c][k] = 0xff800000u;  // -inf
        }
        float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          mx0 = fmaxf(mx0, __uint_as_float(s[0][k]));
          mx1 = fmaxf(mx1, __uint_as_float(s[1][k]));
          mx2 = fmaxf(mx2, __uint_as_float(s[2][k]));
          mx3 = fmaxf(mx3, __uint_as_float(s[3][k]));
        }
        const float m_tile = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
        if (j == 0) {
          m_ref = m_tile;
        } else {
          // Lazy rescale: keep the stale reference max while the new max exceeds it by < 2^8.
          const bool need = (m_tile - m_ref) * sl2 > 8.0f;
          if (__any_sync(0xffffffffu, need)) {
            const float m_new = fmaxf(m_ref, m_tile);
            const float alpha = ex2((m_ref - m_new) * sl2);
            m_ref = m_new;
            l *= alpha;
            // s_full(j) completed => every earlier MMA, including O_i += P_i V_{j-1}, is complete.
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
              uint32_t o[32];
              tmem_ld32(tO + c * 32, o);
              tmem_wait_ld();
#pragma unroll
              for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
              tmem_st32(tO + c * 32, o);
            }
          }
        }
        const float neg_m = -m_ref * sl2;
        float l0 = 0.f, l1 = 0.f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            const float p0 = ex2(fmaf(__uint_as_float(s[c][2 * k]), sl2, neg_m));
            const float p1 = ex2(fmaf(__uint_as_float(s[c][2 * k + 1]), sl2, neg_m));
            l0 += p0;
            l1 += p1;
            pk[k] = pack_bf16(p0, p1);
          }
          tmem_st16(tS + c * 16, pk);  // P_i: bf16 pairs, columns [16c, 16c+16) of S_i
        }
        l += l0 + l1;
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bar_p_full + 8 * i);
      }
      // ---------------------------------------------------- epilogue (a5): O / l -> bf16, LSE
      mbar_wait(bar_o_full + 8 * i, 0);
      tc_fence_after();
      const int row = i * kTile + (warp & 3) * 32 + lane;
      const bool valid = row < item.q_rows;
      const int n_tok = item.q_is_ref ? p.n_ref : p.n_gen;
      const int grow = item.q_row0 + row;
      __nv_bfloat16* obase = item.q_is_ref ? p.o_ref : p.o_gen;
      uint4* orow = reinterpret_cast<uint4*>(obase + ((size_t(b) * n_tok + grow) * p.heads + h) * D);
      const float inv_l = 1.0f / l;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(tO + c * 32, o);
        tmem_wait_ld();
        if (valid) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint4 v;
            v.x = pack_bf16(__uint_as_float(o[8 * q + 0]) * inv_l, __uint_as_float(o[8 * q + 1]) * inv_l);
            v.y = pack_bf16(__uint_as_float(o[8 * q + 2]) * inv_l, __uint_as_float(o[8 * q + 3]) * inv_l);
            v.z = pack_bf16(__uint_as_float(o[8 * q + 4]) * inv_l, __uint_as_float(o[8 * q + 5]) * inv_l);
            v.w = pack_bf16(__uint_as_float(o[8 * q + 6]) * inv_l, __uint_as_float(o[8 * q + 7]) * inv_l);
            orow[c * 4 + q] = v;
          }
        }
      }
      float* lse = item.q_is_ref ? p.lse_ref : p.lse_gen;
      if (lse != nullptr && valid) lse[(size_t(b) * p.heads + h) * n_tok + grow] = m_ref * p.scale + __logf(l);
      tc_fence_before();
    }
  } else {
    reg_dec<56>();
    if (warp == 9 && lane == 0) {
      // ===================================================== TMA loader
      const CUtensorMap* tq = item.q_is_ref ? &tm_q_ref : &tm_q_gen;
      mbar_arrive_expect_tx(bar_q_full, n_qt * C::kTileBytes);
      for (int i = 0; i < n_qt; ++i) load_tile<D>(sQ + i * C::kTileBytes, tq, bar_q_full, item.q_row0 + i * kTile, h, b, false);
      int it = 0;
      for (int j = 0; j < n_kv; ++j) {
        const bool first = j < n0;
        const bool is_ref = first ? (item.seg0_is_ref != 0) : true;
        const int row = first ? item.seg0_start + j * kTile : item.seg1_start + (j - n0) * kTile;
        const bool hm = is_ref && p.ref_kv_head_major;
#pragma unroll
        for (int kv = 0; kv < 2; ++kv, ++it) {
          const int s = it % C::kStages;
          const uint32_t ph = (it / C::kStages) & 1;
          const CUtensorMap* tm = kv == 0 ? (is_ref ? &tm_k_ref : &tm_k_gen) : (is_ref ? &tm_v_ref : &tm_v_gen);
          mbar_wait(bar_kv_empty + 8 * s, ph ^ 1);
          mbar_arrive_expect_tx(bar_kv_full + 8 * s, C::kTileBytes);
          load_tile<D>(sKV + s * C::kTileBytes, tm, bar_kv_full + 8 * s, row, h, b, hm);
        }
      }
    } else if (warp == 8 && lane == 0) {
      // ===================================================== MMA issuer
      constexpr uint32_t idesc_qk = make_idesc_bf16(kTile, kTile, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc_bf16(kTile, D, 0, 1);
      auto issue_qk = [&](int i, int stage) {
        const uint32_t q = sQ + i * C::kTileBytes, k = sKV + stage * C::kTileBytes;
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t off = (kk / 4) * C::kBoxBytes + (kk % 4) * 32;
          umma_ss(tS0 + i * 128, make_smem_desc_sw128(q + off, 16, 1024), make_smem_desc_sw128(k + off, 16, 1024),
                  idesc_qk, kk > 0);
        }
      };
      auto issue_pv = [&](int i, int stage, bool acc) {
        const uint32_t v = sKV + stage * C::kTileBytes;
#pragma unroll
        for (int kk = 0; kk < kTile / 16; ++kk)
          umma_ts(tO0 + i * D, tS0 + i * 128 + kk * 8, make_smem_desc_sw128(v + kk * 2048, C::kBoxBytes, 1024), idesc_pv,
                  (acc || kk > 0) ? 1u : 0u);
      };
      auto stage_of = [&](int it) { return it % C::kStages; };
      auto phase_of = [&](int it) { return uint32_t((it / C::kStages) & 1); };

      mbar_wait(bar_q_full, 0);
      int it = 0;
      mbar_wait(bar_kv_full + 8 * stage_of(it), phase_of(it));
      tc_fence_after();
      for (int i = 0; i < n_qt; ++i) {
        issue_qk(i, stage_of(it));
        umma_commit(bar_s_full + 8 * i);
      }
      umma_commit(bar_kv_empty + 8 * stage_of(it));
      ++it;
      for (int j = 0; j < n_kv; ++j) {
        const int sv = stage_of(it);
        mbar_wait(bar_kv_full + 8 * sv, phase_of(it));
        ++it;
        const bool more = j + 1 < n_kv;
        const int sk = stage_of(it);
        for (int i = 0; i < n_qt; ++i) {
          mbar_wait(bar_p_full + 8 * i, j & 1);
          tc_fence_after();
          issue_pv(i, sv, j > 0);
          if (!more) umma_commit(bar_o_full + 8 * i);
          if (i == n_qt - 1) umma_commit(bar_kv_empty + 8 * sv);
          if (more) {
            if (i == 0) {
              mbar_wait(bar_kv_full + 8 * sk, phase_of(it));
              tc_fence_after();
            }
            issue_qk(i, sk);
            umma_commit(bar_s_full + 8 * i);
            if (i == n_qt - 1) umma_commit(bar_kv_empty + 8 * sk);
          }
        }
        if (more) ++it;
      }
    }
  }
  __syncthreads();
  if (warp == 8) {
    tc_fence_after();
    tmem_dealloc(tmem, C::kTmemCols);
  }
}

template <int D>
cudaError_t launch_fwd(const CUtensorMap* maps, const FwdParams& p, cudaStream_t stream) {
  using C = FwdCfg<D>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(sra_fwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid(p.n_items, p.heads, p.batch);
  sra_fwd_kernel<D><<<grid, C::kThreads, C::kSmemBytes, stream>>>(maps[0], maps[1], maps[2], maps[3], maps[4], maps[5], p);
  return cudaGetLastError();
}

template cudaError_t launch_fwd<64>(const CUtensorMap*, const FwdParams&, cudaStream_t);
template cudaError_t launch_fwd<128>(const CUtensorMap*, const FwdParams&, cudaStream_t);

}  // namespace sra
