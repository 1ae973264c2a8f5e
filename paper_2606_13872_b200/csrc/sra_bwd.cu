// SRA backward for sm_100a (PAPER.md:173 - SFT trains through SRA).
//
//   a6  sra_bwd_preprocess_kernel   D_i = sum_c dO_ic O_ic and LSE_i * log2(e), rows [G ; R] concatenated
//   a7  sra_bwd_kernel<D>           one CTA = one 128-key tile x one (batch, head); it loops over the 64-row
//                                   query tiles that may see the tile (all G queries; for a reference key tile
//                                   also the R queries of its own block - the transposed SRA mask), 5 MMAs each:
//         S^T  = K   Q_i^T      [keys x queries]   SS, -> TMEM S[i&1]
//         dP^T = V   dO_i^T     [keys x queries]   SS, -> TMEM dP
//         dV  += P^T dO_i       [keys x d]         A = P^T (bf16) from TMEM, aliasing S[i&1]
//         dK  += dS^T Q_i       [keys x d]         A = dS^T (bf16) from shared memory
//         dQ_i^T = K^T dS^T     [d x queries]      A = K (MN-major), B = dS^T (MN-major), -> TMEM dQ
//       with P^T = exp2(S^T * scale*log2e - LSE*log2e) formed by one warpgroup and dS^T = P^T o (dP^T - D) by a
//       second one (thread = key = TMEM lane; the two are pipeline stages of consecutive tiles).  dQ_i^T is
//       drained by a third warpgroup (thread = d = TMEM lane) straight from registers into the fp32 workspace
//       [B*H][n_pad][d] with coalesced red.global.add.f32 (many key tiles add into the same query rows; the
//       summation order is not deterministic - SURVEY.md 8c A13).  What bounds the kernel is the tensor pipe
//       itself: the N = 64 SS MMAs (S^T, dP^T, dQ^T) run at 2/3 rate (operand reads), see DESIGN.md 6.2.
//   a8  sra_bwd_dq_finalize_kernel  workspace * scale -> bf16 dQ [B, N, H, d]
//
// TMEM columns (D = 128): S0 @0 (64), S1 @64 (64), dP0 @128 (64), dP1 @192 (64), dV @256 (128), dK @384 (128);
// dQ^T(it) overwrites dP^T(it) in dP[it & 1].
#include "ptx.cuh"
#include "sra_common.h"
#include "sra_ctx.h"

namespace sra {

template <int D>
struct BwdCfg {
  static constexpr int kQT = kBwdQTile;
  static constexpr int kKBytes = kTile * D * 2;         // K or V tile
  static constexpr int kKBoxBytes = kTile * 128;        // one 64-column box of K/V
  static constexpr int kQBytes = kQT * D * 2;           // Q_i or dO_i tile
  static constexpr int kQBoxBytes = kQT * 128;
  static constexpr int kBoxes = D / 64;
  static constexpr int kStages = 4;
  static constexpr int kStageBytes = 2 * kQBytes;       // Q_i + dO_i
  static constexpr int kDsBytes = kTile * kQT * 2;      // dS^T tile [128 keys][64 queries] bf16, x2 buffers
  static constexpr int kVecBytes = kStages * 2 * kQT * 4;  // lse2[64] + delta[64] per stage
  static constexpr int kNumBars = 1 + 2 * kStages + 2 + 2 + 2 + 2 + 2 + 2 + 2 + 1;
  static constexpr int kSmemBytes = 2 * kKBytes + kStages * kStageBytes + 2 * kDsBytes + kVecBytes + kNumBars * 8 + 16;
  static constexpr int kThreads = 512;  // P, dS and dQ warpgroups, MMA + TMA warps (+2 idle)
  // TMEM columns: S0 | S1 | dP0 | dP1 (64 each) | dV | dK.  dQ^T(it) is written over dP^T(it) in dP[it & 1] once the dS
  // warpgroup has read it, so dP^T(it+1) has a buffer of its own and does not wait for tile it's dS / dQ chain.
  static constexpr int kColS = 0, kColDP = 128, kColDV = 256, kColDK = 256 + D;
};

template <int D>
__device__ __forceinline__ void bwd_load_tile(uint32_t dst, int box_bytes, const CUtensorMap* tm, uint32_t bar, int row,
                                              int h, int b, bool head_major) {
#pragma unroll
  for (int x = 0; x < D / 64; ++x) {
    if (head_major)
      tma_load_4d(dst + x * box_bytes, tm, bar, x * 64, row, h, b);
    else
      tma_load_4d(dst + x * box_bytes, tm, bar, x * 64, h, row, b);
  }
}

struct QTile {
  int is_ref, row0, valid, cat0;
};

__device__ __forceinline__ QTile q_tile_of(int it, int n0, const BwdItem& item, int n_gen) {
  QTile t;
  if (it < n0) {
    t.is_ref = 0;
    t.row0 = item.g_start + it * kBwdQTile;
    t.valid = min(kBwdQTile, item.g_start + item.g_len - t.row0);
    t.cat0 = t.row0;
  } else {
    t.is_ref = 1;
    t.row0 = item.seg1_start + (it - n0) * kBwdQTile;
    t.valid = min(kBwdQTile, item.seg1_start + item.seg1_len - t.row0);
    t.cat0 = n_gen + t.row0;
  }
  return t;
}

template <int D>
__global__ void __launch_bounds__(BwdCfg<D>::kThreads, 1)
    sra_bwd_kernel(const __grid_constant__ CUtensorMap tm_q_gen, const __grid_constant__ CUtensorMap tm_do_gen,
                   const __grid_constant__ CUtensorMap tm_q_ref, const __grid_constant__ CUtensorMap tm_do_ref,
                   const __grid_constant__ CUtensorMap tm_k_gen, const __grid_constant__ CUtensorMap tm_v_gen,
                   const __grid_constant__ CUtensorMap tm_k_ref, const __grid_constant__ CUtensorMap tm_v_ref,
                   const BwdParams p) {
  using C = BwdCfg<D>;
  constexpr int QT = C::kQT;
  constexpr int ST = C::kStages;
  extern __shared__ __align__(1024) uint8_t smem_raw[];  // 128-byte-swizzled tiles need 1024-byte alignment
  const uint32_t smem_base = smem_u32(smem_raw);
  if ((smem_base & 1023u) != 0) __trap();
  const uint32_t sK = smem_base;
  const uint32_t sV = sK + C::kKBytes;
  const uint32_t sStage = sV + C::kKBytes;                      // [ST] x {Q_i, dO_i}
  const uint32_t sDs = sStage + ST * C::kStageBytes;            // [2] dS^T
  const uint32_t sVec = sDs + 2 * C::kDsBytes;                  // [ST] x {lse2[64], delta[64]}
  const uint32_t sBar = sVec + C::kVecBytes;
  const uint32_t bar_kv_full = sBar;
  const uint32_t bar_q_full = sBar + 8;                         // [ST]
  const uint32_t bar_q_empty = bar_q_full + 8 * ST;             // [ST]
  const uint32_t bar_s_full = bar_q_empty + 8 * ST;             // [2]
  const uint32_t bar_dp_full = bar_s_full + 16;                 // [2]
  const uint32_t bar_p_full = bar_dp_full + 16;                 // [2]
  const uint32_t bar_ds_full = bar_p_full + 16;                 // [2]
  const uint32_t bar_ds_empty = bar_ds_full + 16;               // [2]
  const uint32_t bar_dq_full = bar_ds_empty + 16;               // [2]
  const uint32_t bar_dq_empty = bar_dq_full + 16;               // [1]
  const uint32_t bar_acc_full = bar_dq_empty + 8;               // [1]
  const uint32_t s_tmem_ptr = bar_acc_full + 8;
  uint32_t* tmem_ptr_generic = reinterpret_cast<uint32_t*>(smem_raw + (s_tmem_ptr - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const BwdItem item = p.items[blockIdx.x];
  const int h = blockIdx.y;
  const int b = blockIdx.z;
  const int bh = b * p.heads + h;
  const int n0 = (item.g_len + QT - 1) / QT;  // generation query tiles that see this key tile
  const int n1 = (item.seg1_len + QT - 1) / QT;
  const int n_it = n0 + n1;

  if (threadIdx.x == 0) {
    mbar_init(bar_kv_full, 1);
    for (int s = 0; s < ST; ++s) {
      mbar_init(bar_q_full + 8 * s, 1);
      mbar_init(bar_q_empty + 8 * s, 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_s_full + 8 * i, 1);
      mbar_init(bar_p_full + 8 * i, 128);
      mbar_init(bar_ds_full + 8 * i, 128);
      mbar_init(bar_ds_empty + 8 * i, 1);
      mbar_init(bar_dp_full + 8 * i, 1);
      mbar_init(bar_dq_full + 8 * i, 1);
    }
    mbar_init(bar_dq_empty, 128);
    mbar_init(bar_acc_full, 1);
    fence_mbar_init();
  }
  if (warp == 13 && lane == 0) {
    tma_prefetch_desc(&tm_q_gen);
    tma_prefetch_desc(&tm_do_gen);
    tma_prefetch_desc(item.k_is_ref ? &tm_k_ref : &tm_k_gen);
    tma_prefetch_desc(item.k_is_ref ? &tm_v_ref : &tm_v_gen);
  }
  if (warp == 12) tmem_alloc(s_tmem_ptr, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr_generic;

  if (warp < 4) {
    // ================================================= P warpgroup: P^T = exp2(S^T * sl2 - LSE * log2e) (thread = key)
    // The elementwise work of a tile is split into two pipeline stages on two warpgroups (this one and the
    // dS warpgroup below), so each SM sub-partition always has warps in different phases (MUFU-bound exp2
    // here, FMA/LSU-bound dS there, tcgen05.ld round trips in both) and a tile's P^T is ready for dV while
    // the previous tile's dS^T is still being formed.
    const int key = warp * 32 + lane;
    const bool key_valid = key < item.k_rows;
    const uint32_t lane_off = uint32_t(warp * 32) << 16;
    const float sl2 = p.scale_log2;
    for (int it = 0; it < n_it; ++it) {
      const int bf = it & 1, s = it % ST;
      const uint32_t tS = tmem + lane_off + C::kColS + bf * QT;
      const uint32_t vec = sVec + s * (2 * QT * 4);
      mbar_wait(bar_q_full + 8 * s, (it / ST) & 1);  // acquire the loader's lse2 writes
      mbar_wait(bar_s_full + 8 * bf, (it >> 1) & 1);
      tc_fence_after();
      uint32_t sv[2][32];
      tmem_ld32(tS, sv[0]);
      tmem_ld32(tS + 32, sv[1]);
      tmem_wait_ld();
      uint32_t pk[32];
#pragma unroll
      for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int q4 = 0; q4 < 8; ++q4) {
          const float4 l = ld_shared_f4(vec + (c * 32 + q4 * 4) * 4);
          const float p0 = ex2(fmaf(__uint_as_float(sv[c][q4 * 4 + 0]), sl2, -l.x));
          const float p1 = ex2(fmaf(__uint_as_float(sv[c][q4 * 4 + 1]), sl2, -l.y));
          const float p2 = ex2(fmaf(__uint_as_float(sv[c][q4 * 4 + 2]), sl2, -l.z));
          const float p3 = ex2(fmaf(__uint_as_float(sv[c][q4 * 4 + 3]), sl2, -l.w));
          pk[c * 16 + q4 * 2 + 0] = pack_bf16(p0, p1);
          pk[c * 16 + q4 * 2 + 1] = pack_bf16(p2, p3);
        }
      tmem_st32(tS, pk);  // P^T: bf16 pairs in the first 32 columns of S[bf]
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(bar_p_full + 8 * bf);
    }
    // ---------------------------------------------------- epilogue: dV (lanes = keys)
    mbar_wait(bar_acc_full, 0);
    tc_fence_after();
    {
      const int n_tok = item.k_is_ref ? p.n_ref : p.n_gen;
      const int grow = item.k_row0 + key;
      __nv_bfloat16* base = item.k_is_ref ? p.dv_ref : p.dv_gen;
      uint4* orow = reinterpret_cast<uint4*>(base + ((size_t(b) * n_tok + grow) * p.heads + h) * D);
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(tmem + lane_off + C::kColDV + c * 32, o);
        tmem_wait_ld();
        if (key_valid) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint4 v;
            v.x = pack_bf16(__uint_as_float(o[8 * q + 0]), __uint_as_float(o[8 * q + 1]));
            v.y = pack_bf16(__uint_as_float(o[8 * q + 2]), __uint_as_float(o[8 * q + 3]));
            v.z = pack_bf16(__uint_as_float(o[8 * q + 4]), __uint_as_float(o[8 * q + 5]));
            v.w = pack_bf16(__uint_as_float(o[8 * q + 6]), __uint_as_float(o[8 * q + 7]));
            orow[c * 4 + q] = v;
          }
        }
      }
    }
    tc_fence_before();
  } else if (warp < 8) {
    // ================================================= dS warpgroup: dS^T = P^T o (dP^T - D) (thread = key)
    // P^T is read back from TMEM as the bf16 the dV MMA consumes (S[bf] is not overwritten before the
    // MMA issuer has seen ds_full of this tile).
    const int wk = warp - 4;
    const int key = wk * 32 + lane;
    const bool key_valid = key < item.k_rows;
    const uint32_t lane_off = uint32_t(wk * 32) << 16;
    for (int it = 0; it < n_it; ++it) {
      const int bf = it & 1, s = it % ST;
      const uint32_t tP = tmem + lane_off + C::kColS + bf * QT;
      const uint32_t tDP = tmem + lane_off + C::kColDP + bf * QT;
      const uint32_t vec = sVec + s * (2 * QT * 4) + QT * 4;  // delta[64]
      mbar_wait(bar_q_full + 8 * s, (it / ST) & 1);  // acquire the loader's delta writes
      mbar_wait(bar_p_full + 8 * bf, (it >> 1) & 1);
      mbar_wait(bar_dp_full + 8 * bf, (it >> 1) & 1);
      tc_fence_after();
      uint32_t pb[32], dp[2][32];
      tmem_ld32(tP, pb);
      tmem_ld32(tDP, dp[0]);
      tmem_ld32(tDP + 32, dp[1]);
      tmem_wait_ld();
      mbar_wait(bar_ds_empty + 8 * bf, ((it >> 1) & 1) ^ 1);  // dK / dQ MMAs of iteration it-2 have read sDs[bf]
      const uint32_t ds_row = sDs + bf * C::kDsBytes + key * 128;
#pragma unroll
      for (int c = 0; c < 8; ++c) {  // 16-byte chunk c = queries [8c, 8c+8)
        const float4 d0 = ld_shared_f4(vec + (c * 8) * 4);
        const float4 d1 = ld_shared_f4(vec + (c * 8 + 4) * 4);
        const float dl[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const int q = c * 8 + 2 * k;
          const uint32_t pp = pb[q >> 1];
          float a = __uint_as_float(pp << 16) * (__uint_as_float(dp[q >> 5][q & 31]) - dl[2 * k]);
          float bb = __uint_as_float(pp & 0xffff0000u) * (__uint_as_float(dp[(q + 1) >> 5][(q + 1) & 31]) - dl[2 * k + 1]);
          if (!key_valid) { a = 0.f; bb = 0.f; }
          w[k] = pack_bf16(a, bb);
        }
        st_shared_v4(ds_row + ((c ^ (key & 7)) << 4), w[0], w[1], w[2], w[3]);
      }
      fence_proxy_async_smem();
      tc_fence_before();
      mbar_arrive(bar_ds_full + 8 * bf);
    }
  } else if (warp < 12) {
    // ================================================= reduce warpgroup: dQ^T drain (thread = d), then dK epilogue
    const int wq = warp - 8;
    const int drow = wq * 32 + lane;  // TMEM lane = d index (dQ^T), later = key index (dK)
    const uint32_t lane_off = uint32_t(wq * 32) << 16;
    for (int it = 0; it < n_it; ++it) {
      const QTile qt = q_tile_of(it, n0, item, p.n_gen);
      mbar_wait(bar_dq_full + 8 * (it & 1), (it >> 1) & 1);
      tc_fence_after();
      uint32_t r[2][32];
      tmem_ld32(tmem + lane_off + C::kColDP + (it & 1) * QT, r[0]);
      tmem_ld32(tmem + lane_off + C::kColDP + (it & 1) * QT + 32, r[1]);
      tmem_wait_ld();
      tc_fence_before();
      mbar_arrive(bar_dq_empty);
      // dQ_it^T leaves the SM straight from registers: for a fixed query the 32 lanes of a warp hold 32
      // consecutive d, so each red.global.add.f32 is one coalesced 128-byte reduction into the fp32
      // workspace (no shared-memory staging: the kernel is bound by shared-memory bandwidth).
      float* dq_row = p.dq_ws + (size_t(bh) * p.n_pad + qt.cat0) * D + drow;
#pragma unroll
      for (int x = 0; x < 2; ++x)
#pragma unroll
        for (int c = 0; c < 32; ++c)
          if (drow < D && x * 32 + c < qt.valid) red_add_f32(dq_row + (x * 32 + c) * D, __uint_as_float(r[x][c]));
    }
    // ---------------------------------------------------- epilogue: dK = scale * acc (lanes = keys)
    mbar_wait(bar_acc_full, 0);
    tc_fence_after();
    {
      const int key = drow;
      const bool key_valid = key < item.k_rows;
      const int n_tok = item.k_is_ref ? p.n_ref : p.n_gen;
      const int grow = item.k_row0 + key;
      __nv_bfloat16* base = item.k_is_ref ? p.dk_ref : p.dk_gen;
      uint4* orow = reinterpret_cast<uint4*>(base + ((size_t(b) * n_tok + grow) * p.heads + h) * D);
      const float sc = p.scale;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(tmem + lane_off + C::kColDK + c * 32, o);
        tmem_wait_ld();
        if (key_valid) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint4 v;
            v.x = pack_bf16(__uint_as_float(o[8 * q + 0]) * sc, __uint_as_float(o[8 * q + 1]) * sc);
            v.y = pack_bf16(__uint_as_float(o[8 * q + 2]) * sc, __uint_as_float(o[8 * q + 3]) * sc);
            v.z = pack_bf16(__uint_as_float(o[8 * q + 4]) * sc, __uint_as_float(o[8 * q + 5]) * sc);
            v.w = pack_bf16(__uint_as_float(o[8 * q + 6]) * sc, __uint_as_float(o[8 * q + 7]) * sc);
            orow[c * 4 + q] = v;
          }
        }
      }
    }
    tc_fence_before();
  } else {
    if (warp == 13) {
      // ================================================= loader: K/V once, then the {Q_i, dO_i, lse2, delta} ring
      const bool k_hm = item.k_is_ref && p.ref_kv_head_major;
      if (lane == 0) {
        mbar_arrive_expect_tx(bar_kv_full, 2 * C::kKBytes);
        bwd_load_tile<D>(sK, C::kKBoxBytes, item.k_is_ref ? &tm_k_ref : &tm_k_gen, bar_kv_full, item.k_row0, h, b, k_hm);
        bwd_load_tile<D>(sV, C::kKBoxBytes, item.k_is_ref ? &tm_v_ref : &tm_v_gen, bar_kv_full, item.k_row0, h, b, k_hm);
      }
      const float* lse2 = p.lse2 + size_t(bh) * p.n_pad;
      const float* delta = p.delta + size_t(bh) * p.n_pad;
      for (int it = 0; it < n_it; ++it) {
        const int s = it % ST;
        const QTile qt = q_tile_of(it, n0, item, p.n_gen);
        mbar_wait(bar_q_empty + 8 * s, ((it / ST) & 1) ^ 1);
        const uint32_t vec = sVec + s * (2 * QT * 4);
#pragma unroll
        for (int r = lane; r < QT; r += 32) {
          const bool ok = r < qt.valid;
          st_shared_f32(vec + r * 4, ok ? lse2[qt.cat0 + r] : INFINITY);   // +inf => P = 0 for rows outside the tile
          st_shared_f32(vec + QT * 4 + r * 4, ok ? delta[qt.cat0 + r] : 0.f);
        }
        __syncwarp();
        if (lane == 0) {
          const uint32_t dst = sStage + s * C::kStageBytes;
          mbar_arrive_expect_tx(bar_q_full + 8 * s, 2 * C::kQBytes);
          bwd_load_tile<D>(dst, C::kQBoxBytes, qt.is_ref ? &tm_q_ref : &tm_q_gen, bar_q_full + 8 * s, qt.row0, h, b, false);
          bwd_load_tile<D>(dst + C::kQBytes, C::kQBoxBytes, qt.is_ref ? &tm_do_ref : &tm_do_gen, bar_q_full + 8 * s,
                           qt.row0, h, b, false);
        }
      }
    } else if (warp == 12 && elect_one()) {
      // ================================================= MMA issuer
      constexpr uint32_t idesc_st = make_idesc_bf16(kTile, QT, 0, 0);   // S^T, dP^T : [128 x 64], K = d
      constexpr uint32_t idesc_acc = make_idesc_bf16(kTile, D, 0, 1);   // dV, dK    : [128 x D],  K = 64 queries
      // dQ^T : [D x 64], K = 128 keys.  With D = 64 the MMA is still issued with M = 128 (the M = 64 accumulator layout
      // differs): its A operand then runs on from the K tile into the V tile behind it, TMEM lanes [64, 128) receive
      // finite garbage (V^T dS^T) and the drain ignores them.
      constexpr uint32_t idesc_dq = make_idesc_bf16(kTile, QT, 1, 1);
      const uint32_t tS0 = tmem + C::kColS, tDP0 = tmem + C::kColDP;
      const uint32_t tDV = tmem + C::kColDV, tDK = tmem + C::kColDK;
      // Descriptor low words (start address, LBO); stepping along K or to another stage is one 32-bit add.
      constexpr uint32_t kHi = desc_hi_sw128(1024);
      const uint32_t k_km = desc_lo(sK, 16), v_km = desc_lo(sV, 16);             // K, V as K-major A operands
      const uint32_t k_mn = desc_lo(sK, C::kKBoxBytes);                          // K as MN-major A operand (dQ^T)
      const uint32_t st_km = desc_lo(sStage, 16);                                // Q_i / dO_i as K-major B operands
      const uint32_t st_mn = desc_lo(sStage, C::kQBoxBytes);                     // Q_i / dO_i as MN-major B operands
      const uint32_t ds_km = desc_lo(sDs, 16), ds_mn = desc_lo(sDs, C::kDsBytes);
      // [128 x 64] = A[128 keys][d] (K-major) * B[64 queries][d]^T (K-major); b_off = byte offset inside sStage
      auto issue_kq = [&](uint32_t d_tmem, uint32_t a_lo, uint32_t b_off) {
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk)
          umma_ss(d_tmem, desc64(a_lo + (((kk / 4) * C::kKBoxBytes + (kk % 4) * 32) >> 4), kHi),
                  desc64(st_km + ((b_off + (kk / 4) * C::kQBoxBytes + (kk % 4) * 32) >> 4), kHi), idesc_st, kk > 0);
      };
      mbar_wait(bar_kv_full, 0);
      mbar_wait(bar_q_full, 0);
      tc_fence_after();
      issue_kq(tS0, k_km, 0);
      umma_commit(bar_s_full);
      issue_kq(tDP0, v_km, C::kQBytes);
      umma_commit(bar_dp_full);
      for (int it = 0; it < n_it; ++it) {
        const int bf = it & 1, s = it % ST;
        const uint32_t oQ = s * C::kStageBytes, oDO = oQ + C::kQBytes;  // byte offsets inside sStage
        const uint32_t ods = bf * C::kDsBytes;
        const bool more = it + 1 < n_it;
        const int s1 = (it + 1) % ST;
        const uint32_t oQ1 = s1 * C::kStageBytes;
        if (more) {
          mbar_wait(bar_q_full + 8 * s1, ((it + 1) / ST) & 1);
          tc_fence_after();
          issue_kq(tS0 + (bf ^ 1) * QT, k_km, oQ1);  // S^T(it+1); its buffer held P^T(it-1), consumed by dV(it-1)
          umma_commit(bar_s_full + 8 * (bf ^ 1));
          // dP^T(it+1) -> dP[bf ^ 1], which last held dQ^T(it-1): only the dQ warpgroup's drain of that tile gates it
          mbar_wait(bar_dq_empty, (it & 1) ^ 1);
          tc_fence_after();
          issue_kq(tDP0 + (bf ^ 1) * QT, v_km, oQ1 + C::kQBytes);
          umma_commit(bar_dp_full + 8 * (bf ^ 1));
        }
        // dV += P^T(it) dO_it : A = P^T from TMEM (16 queries = 8 columns per step), B = dO_it [queries][d] MN-major
        mbar_wait(bar_p_full + 8 * bf, (it >> 1) & 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < QT / 16; ++kk)
          umma_ts(tDV, tS0 + bf * QT + kk * 8, desc64(st_mn + ((oDO + kk * 2048) >> 4), kHi), idesc_acc,
                  (it > 0 || kk > 0) ? 1u : 0u);
        mbar_wait(bar_ds_full + 8 * bf, (it >> 1) & 1);  // dS^T(it) in smem; dP^T(it) has been read out of TMEM
        tc_fence_after();
        // dK += dS^T(it) Q_it : A = dS^T [keys][queries] K-major (one 128-byte box), B = Q_it [queries][d] MN-major
#pragma unroll
        for (int kk = 0; kk < QT / 16; ++kk)
          umma_ss(tDK, desc64(ds_km + ((ods + kk * 32) >> 4), kHi), desc64(st_mn + ((oQ + kk * 2048) >> 4), kHi),
                  idesc_acc, (it > 0 || kk > 0) ? 1u : 0u);
        // dQ_it^T = K^T dS^T(it) : A = K [keys][d] MN-major, B = dS^T [keys][queries] MN-major, K = 128 keys; written
        // over dP^T(it), which the dS warpgroup has read (ds_full)
#pragma unroll
        for (int kk = 0; kk < kTile / 16; ++kk)
          umma_ss(tDP0 + bf * QT, desc64(k_mn + ((kk * 2048) >> 4), kHi), desc64(ds_mn + ((ods + kk * 2048) >> 4), kHi), idesc_dq, kk > 0);
        umma_commit(bar_dq_full + 8 * bf);
        umma_commit(bar_q_empty + 8 * s);
        umma_commit(bar_ds_empty + 8 * bf);
      }
      umma_commit(bar_acc_full);
    }
  }
  __syncthreads();
  if (warp == 12) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

// a6: D_i = sum_c dO_ic O_ic and LSE_i * log2(e) for rows [G ; R]; one warp per (b, token, head) row.
template <int D>
__global__ void sra_bwd_preprocess_kernel(const __nv_bfloat16* __restrict__ o_gen, const __nv_bfloat16* __restrict__ do_gen,
                                          const float* __restrict__ lse_gen, const __nv_bfloat16* __restrict__ o_ref,
                                          const __nv_bfloat16* __restrict__ do_ref, const float* __restrict__ lse_ref,
                                          float* __restrict__ delta, float* __restrict__ lse2, int B, int H, int n_gen,
                                          int n_ref, int n_pad) {
  const int lane = threadIdx.x & 31;
  const size_t warp_id = (blockIdx.x * size_t(blockDim.x) + threadIdx.x) >> 5;
  const size_t n_warps = (gridDim.x * size_t(blockDim.x)) >> 5;
  const size_t n_cat = size_t(n_gen) + n_ref;
  const size_t total = size_t(B) * n_cat * H;
  for (size_t r = warp_id; r < total; r += n_warps) {
    const int h = int(r % H);
    const size_t t = r / H;
    const int n = int(t % n_cat);
    const int b = int(t / n_cat);
    const bool is_ref = n >= n_gen;
    const int row = is_ref ? n - n_gen : n;
    const int n_tok = is_ref ? n_ref : n_gen;
    const size_t off = ((size_t(b) * n_tok + row) * H + h) * D;
    const __nv_bfloat16* o = (is_ref ? o_ref : o_gen) + off;
    const __nv_bfloat16* d = (is_ref ? do_ref : do_gen) + off;
    float acc = 0.f;
    if (D == 128) {
      const uint2 a = reinterpret_cast<const uint2*>(o)[lane], c = reinterpret_cast<const uint2*>(d)[lane];
      const __nv_bfloat162* a2 = reinterpret_cast<const __nv_bfloat162*>(&a);
      const __nv_bfloat162* c2 = reinterpret_cast<const __nv_bfloat162*>(&c);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const float2 x = __bfloat1622float2(a2[k]), y = __bfloat1622float2(c2[k]);
        acc = fmaf(x.x, y.x, acc);
        acc = fmaf(x.y, y.y, acc);
      }
    } else {
      const uint32_t a = reinterpret_cast<const uint32_t*>(o)[lane], c = reinterpret_cast<const uint32_t*>(d)[lane];
      const float2 x = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&a));
      const float2 y = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&c));
      acc = fmaf(x.x, y.x, x.y * y.y);
    }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, m);
    if (lane == 0) {
      const size_t w = (size_t(b) * H + h) * n_pad + n;
      delta[w] = acc;
      const float l = (is_ref ? lse_ref : lse_gen)[(size_t(b) * H + h) * n_tok + row];
      lse2[w] = l * 1.4426950408889634f;
    }
  }
}

// a8: dQ[b, n, h, :] = scale * ws[b*H + h][n][:]  (fp32) -> bf16; 8 elements (32 B in, 16 B out) per thread.
template <int D>
__global__ void sra_bwd_dq_finalize_kernel(const float* __restrict__ ws, __nv_bfloat16* __restrict__ dq_gen,
                                           __nv_bfloat16* __restrict__ dq_ref, int B, int H, int n_gen, int n_ref,
                                           int n_pad, float scale) {
  constexpr int V = D / 8;  // 8-element vectors per row
  const size_t n_cat = size_t(n_gen) + n_ref;
  const size_t total = size_t(B) * H * n_cat * V;
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int v = int(i % V);
    size_t t = i / V;
    const int h = int(t % H);  // output-major order: consecutive threads write consecutive bytes of dQ
    t /= H;
    const size_t n = t % n_cat;
    const int b = int(t / n_cat);
    // visit rows in output order: all G rows of batch b, then all R rows
    const bool is_ref = n >= size_t(n_gen);
    const int row = int(is_ref ? n - n_gen : n);
    const int n_tok = is_ref ? n_ref : n_gen;
    const float4* src = reinterpret_cast<const float4*>(ws + ((size_t(b) * H + h) * n_pad + n) * D) + 2 * v;
    const float4 x = src[0], y = src[1];
    uint4 o;
    o.x = pack_bf16(x.x * scale, x.y * scale);
    o.y = pack_bf16(x.z * scale, x.w * scale);
    o.z = pack_bf16(y.x * scale, y.y * scale);
    o.w = pack_bf16(y.z * scale, y.w * scale);
    __nv_bfloat16* dst = (is_ref ? dq_ref : dq_gen) + ((size_t(b) * n_tok + row) * H + h) * D;
    reinterpret_cast<uint4*>(dst)[v] = o;
  }
}

template <int D>
cudaError_t launch_bwd(const CUtensorMap* m, const BwdParams& p, cudaStream_t stream) {
  using C = BwdCfg<D>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(sra_bwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid(p.n_items, p.heads, p.batch);
  sra_bwd_kernel<D><<<grid, C::kThreads, C::kSmemBytes, stream>>>(m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], p);
  return cudaGetLastError();
}

template cudaError_t launch_bwd<64>(const CUtensorMap*, const BwdParams&, cudaStream_t);
template cudaError_t launch_bwd<128>(const CUtensorMap*, const BwdParams&, cudaStream_t);

// ------------------------------------------------------------------------------------------------ host driver
static int run_backward_core(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream);

int run_backward(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream) {
  const sra_config& c = ctx->cfg;
  const int B = c.batch, H = c.heads, d = c.head_dim;
  if (!a->q_gen || !a->k_gen || !a->v_gen || !a->o_gen || !a->lse_gen || !a->do_gen || !a->dq_gen || !a->dk_gen || !a->dv_gen)
    return ctx_fail(ctx, SRA_ERR_INVALID_ARG, "sra_backward: generation tensors (q,k,v,o,lse,do,dq,dk,dv) are required");
  const bool has_ref = c.n_ref > 0;
  if (has_ref && (!a->q_ref || !a->o_ref || !a->lse_ref || !a->do_ref || !a->dq_ref || !a->dk_ref || !a->dv_ref))
    return ctx_fail(ctx, SRA_ERR_INVALID_ARG, "sra_backward: reference tensors (q,o,lse,do,dq,dk,dv) are required when n_ref > 0");
  if ((a->k_ref == nullptr) != (a->v_ref == nullptr))
    return ctx_fail(ctx, SRA_ERR_INVALID_ARG, "k_ref and v_ref must both be NULL or both non-NULL");
  const bool use_cache = has_ref && a->k_ref == nullptr;
  if (use_cache && !ctx->cache_valid) return ctx_fail(ctx, SRA_ERR_NO_REF_CACHE, "k_ref/v_ref NULL but no resident cache");
  const void* ptrs[] = {a->q_gen, a->k_gen, a->v_gen, a->q_ref, a->k_ref, a->v_ref, a->o_gen, a->o_ref, a->do_gen,
                        a->do_ref, a->dq_gen, a->dk_gen, a->dv_gen, a->dq_ref, a->dk_ref, a->dv_ref};
  for (const void* q : ptrs)
    if (q && (reinterpret_cast<uintptr_t>(q) & 15)) return ctx_fail(ctx, SRA_ERR_INVALID_ARG, "tensor pointers must be 16-byte aligned");

  if (!ctx->has_valid || c.n_ref == 0) return run_backward_core(ctx, a, stream);
  // Validity path: gather the valid reference rows, run on the compacted reference, scatter the
  // reference gradients back (rows of invalid tokens are zero).
  sra_bwd_args v = *a;
  int rc;
  if ((rc = compact_rows(ctx, 0, a->q_ref, &v.q_ref, stream))) return rc;
  if ((rc = compact_rows(ctx, 1, a->k_ref, &v.k_ref, stream))) return rc;
  if ((rc = compact_rows(ctx, 2, a->v_ref, &v.v_ref, stream))) return rc;
  if ((rc = compact_rows(ctx, 3, a->o_ref, &v.o_ref, stream))) return rc;
  if ((rc = compact_rows(ctx, 4, a->do_ref, &v.do_ref, stream))) return rc;
  if ((rc = compact_lse(ctx, a->lse_ref, &v.lse_ref, stream))) return rc;
  if ((rc = compact_out(ctx, 5, &v.dq_ref))) return rc;
  if ((rc = compact_out(ctx, 6, &v.dk_ref))) return rc;
  if ((rc = compact_out(ctx, 7, &v.dv_ref))) return rc;
  if ((rc = run_backward_core(ctx, &v, stream))) return rc;
  if ((rc = expand_rows(ctx, 5, a->dq_ref, stream))) return rc;
  if ((rc = expand_rows(ctx, 6, a->dk_ref, stream))) return rc;
  if ((rc = expand_rows(ctx, 7, a->dv_ref, stream))) return rc;
  return SRA_OK;
}

// The launches themselves, on the effective (validity-compacted) reference.
static int run_backward_core(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream) {
  const sra_config& c = ctx->cfg;
  const int B = c.batch, H = c.heads, d = c.head_dim;
  const int nr = ctx->nr;
  const bool has_ref = nr > 0;
  const bool use_cache = has_ref && a->k_ref == nullptr;
  cudaError_t e;
  const int n_cat = c.n_gen + nr;
  const int n_pad = (n_cat + 63) / 64 * 64;
  const size_t vec_bytes = size_t(B) * H * n_pad * 4;
  const size_t dq_bytes = vec_bytes * d;
  if (!ctx->ws_dq) {
    cudaError_t e = cudaMalloc(&ctx->ws_dq, dq_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->ws_delta, vec_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->ws_lse2, vec_bytes);
    if (e != cudaSuccess) {
      (void)cudaGetLastError();
      cudaFree(ctx->ws_dq); cudaFree(ctx->ws_delta); cudaFree(ctx->ws_lse2);
      ctx->ws_dq = ctx->ws_delta = ctx->ws_lse2 = nullptr;
      return ctx_fail(ctx, SRA_ERR_OOM, "backward workspace allocation failed");
    }
    ctx->ws_dq_bytes = dq_bytes;
  }
  e = cudaMemsetAsync(ctx->ws_dq, 0, dq_bytes, stream);
  if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "dQ workspace memset");

  {  // a6
    const size_t rows = size_t(B) * n_cat * H;
    const int threads = 256;
    const int blocks = int(std::min<size_t>((rows * 32 + threads - 1) / threads, size_t(148) * 32));
    KernelTimer kt(ctx, SRA_KERNEL_BWD_PREPROCESS, stream);
    auto launch = [&](auto kernel) {
      kernel<<<blocks, threads, 0, stream>>>(
          static_cast<const __nv_bfloat16*>(a->o_gen), static_cast<const __nv_bfloat16*>(a->do_gen), a->lse_gen,
          static_cast<const __nv_bfloat16*>(a->o_ref), static_cast<const __nv_bfloat16*>(a->do_ref), a->lse_ref,
          ctx->ws_delta, ctx->ws_lse2, B, H, c.n_gen, nr, n_pad);
    };
    if (d == 128) launch(sra_bwd_preprocess_kernel<128>); else launch(sra_bwd_preprocess_kernel<64>);
    if ((e = cudaGetLastError()) != cudaSuccess) return ctx_fail_cuda(ctx, e, "bwd preprocess launch");
    ctx->launches += 1;
  }

  CUtensorMap m[8];
  int rc;
  if ((rc = make_tmap_bf16(ctx, &m[0], a->q_gen, B, c.n_gen, H, d, false, kBwdQTile))) return rc;
  if ((rc = make_tmap_bf16(ctx, &m[1], a->do_gen, B, c.n_gen, H, d, false, kBwdQTile))) return rc;
  if ((rc = make_tmap_bf16(ctx, &m[4], a->k_gen, B, c.n_gen, H, d, false, kTile))) return rc;
  if ((rc = make_tmap_bf16(ctx, &m[5], a->v_gen, B, c.n_gen, H, d, false, kTile))) return rc;
  m[2] = m[0]; m[3] = m[1]; m[6] = m[4]; m[7] = m[5];
  if (has_ref) {
    if ((rc = make_tmap_bf16(ctx, &m[2], a->q_ref, B, nr, H, d, false, kBwdQTile))) return rc;
    if ((rc = make_tmap_bf16(ctx, &m[3], a->do_ref, B, nr, H, d, false, kBwdQTile))) return rc;
    const void* kr = use_cache ? ctx->cache_k : a->k_ref;
    const void* vr = use_cache ? ctx->cache_v : a->v_ref;
    if ((rc = make_tmap_bf16(ctx, &m[6], kr, B, nr, H, d, use_cache, kTile))) return rc;
    if ((rc = make_tmap_bf16(ctx, &m[7], vr, B, nr, H, d, use_cache, kTile))) return rc;
  }

  BwdParams p{};
  p.items = ctx->d_bwd_items;
  p.n_items = int(ctx->bwd_items.size());
  p.heads = H; p.batch = B; p.n_gen = c.n_gen; p.n_ref = nr; p.n_pad = n_pad;
  p.scale = ctx->scale;
  p.scale_log2 = ctx->scale * 1.4426950408889634f;
  p.lse2 = ctx->ws_lse2; p.delta = ctx->ws_delta; p.dq_ws = ctx->ws_dq;
  p.dk_gen = static_cast<__nv_bfloat16*>(a->dk_gen); p.dv_gen = static_cast<__nv_bfloat16*>(a->dv_gen);
  p.dk_ref = static_cast<__nv_bfloat16*>(a->dk_ref); p.dv_ref = static_cast<__nv_bfloat16*>(a->dv_ref);
  p.ref_kv_head_major = use_cache ? 1 : 0;
  {
    KernelTimer kt(ctx, SRA_KERNEL_BWD_MAIN, stream);
    e = d == 128 ? launch_bwd<128>(m, p, stream) : launch_bwd<64>(m, p, stream);
  }
  if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "sra_bwd_kernel launch");
  ctx->launches += 1;

  {  // a8
    const size_t total = size_t(B) * H * n_cat * (d / 8);
    const int threads = 256;
    const int blocks = int(std::min<size_t>((total + threads - 1) / threads, size_t(148) * 32));
    KernelTimer kt(ctx, SRA_KERNEL_BWD_DQ_FINALIZE, stream);
    auto launch = [&](auto kernel) {
      kernel<<<blocks, threads, 0, stream>>>(ctx->ws_dq, static_cast<__nv_bfloat16*>(a->dq_gen),
                                             static_cast<__nv_bfloat16*>(a->dq_ref), B, H, c.n_gen, nr, n_pad, ctx->scale);
    };
    if (d == 128) launch(sra_bwd_dq_finalize_kernel<128>); else launch(sra_bwd_dq_finalize_kernel<64>);
    if ((e = cudaGetLastError()) != cudaSuccess) return ctx_fail_cuda(ctx, e, "dQ finalize launch");
    ctx->launches += 1;
  }
  return SRA_OK;
}

}  // namespace sra
