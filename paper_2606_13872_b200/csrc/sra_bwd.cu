// SRA backward for sm_100a (PAPER.md:173 - SFT trains through SRA).
//
//   a6  sra_bwd_preprocess_kernel   D_i = sum_c dO_ic O_ic and LSE_i * log2(e), rows [G ; R] concatenated
//   a7  sra_bwd_kernel<D>           one CTA = one 128-key tile x one (batch, head); it loops over the 128-row
//                                   query tiles that may see the tile (all G queries; for a reference key tile
//                                   also the R queries of its own block - the transposed SRA mask), 5 MMAs each,
//                                   every one of them M = 128, N = 128 (full tensor rate):
//         S^T  = K   Q_i^T      [keys x queries]   SS            -> TMEM S
//         dP^T = V   dO_i^T     [keys x queries]   SS            -> TMEM dPdQ
//         dV  += P^T dO_i       [keys x d]         A = P^T (bf16) from TMEM, written over S^T
//         dQ_i^T = K^T dS^T     [d x queries]      A = K (MN-major), B = dS^T (MN-major) -> TMEM dPdQ (over dP^T)
//         dK  += dS^T Q_i       [keys x d]         A = dS^T (bf16) from shared memory
//       Thread = key = TMEM lane for the elementwise math.  The compute warps (one per SM sub-partition; two with
//       SRA_BWD_SPLIT = 2) form P^T = exp2(S^T * scale*log2e - LSE*log2e), keep it in registers, and then dS^T = P^T o
//       (dP^T - D) of the same tile.  dQ_i^T is drained by another warpgroup (thread = d = TMEM lane): registers ->
//       a shared-memory staging buffer [query][d] -> cp.reduce.async.bulk .add.f32 into the fp32 workspace
//       [B*H][n_pad][d] (many key tiles add into the same query rows; the summation order is not deterministic -
//       SURVEY.md 8c A13).
//       TMEM is exactly full at d = 128 (S 128 | dPdQ 128 | dV 128 | dK 128 columns), so nothing is double-buffered
//       there; the issue order  dV(i), S^T(i+1), dQ^T(i), dK(i), dP^T(i+1)  gives every elementwise stage the
//       shadow of at least one other tile-sized MMA: exp(i+1) runs under dQ^T(i), dK(i), dP^T(i+1); dS(i+1) under
//       dV(i+1), S^T(i+2); the dQ^T(i) drain under dK(i).  Shared memory (226 KB at d = 128): K, V, dS^T, a 2-stage
//       Q ring (Q_i is read first by S^T(i) and last by dK(i)), one dO buffer (read by dP^T(i) and dV(i), both early
//       in a tile), two slots of {LSE_i log2e, D_i} and 32 KB of dQ staging.
//   a8  sra_bwd_dq_finalize_kernel  workspace * scale -> bf16 dQ [B, N, H, d]
#include <type_traits>

#include "ptx.cuh"
#include "sra_common.h"
#include "sra_ctx.h"

namespace sra {

// Development aid (-DSRA_BWD_TRACE): clock64 timestamps of the pipeline events of one CTA over a few iterations.
#ifdef SRA_BWD_TRACE
__device__ long long* g_bwd_trace = nullptr;
#define TR(role, ev)                                                                                                 \
  do {                                                                                                               \
    if (tr_on && it >= 100 && it < 108 && g_bwd_trace) g_bwd_trace[((role) * 8 + (it - 100)) * 16 + (ev)] = clock64(); \
  } while (0)
#else
#define TR(role, ev) do { } while (0)
#endif

// dQ^T leaves the SM through a shared-memory staging buffer and cp.reduce.async.bulk (1, the default), or as per-thread
// red.global.add.f32 straight from registers (0: the round-1 / early round-2 form, kept for A/B).
#ifndef SRA_BWD_BULK
#define SRA_BWD_BULK 1
#endif
#ifndef SRA_BWD_BULK_NQ
#define SRA_BWD_BULK_NQ 4  // pieces per 128-query tile
#endif
#ifndef SRA_BWD_BULK_NB
#define SRA_BWD_BULK_NB 2  // staging buffers
#endif
#ifndef SRA_BWD_RED_GAP
#define SRA_BWD_RED_GAP 28  // cycles per dQ reduction instruction of a drain warp (0 = unpaced)
#endif
#ifndef SRA_BWD_SPLIT
#define SRA_BWD_SPLIT 1
#endif
#ifndef SRA_BWD_CHUNK
#define SRA_BWD_CHUNK 32  // score columns per tcgen05.ld of the compute warps (16 or 32)
#endif
#ifndef SRA_BWD_EMU
#define SRA_BWD_EMU 0  // of every 8 column pairs, this many take exp2 on the FMA/ALU pipes (ex2_emu2) instead of MUFU
#endif

template <int D>
struct BwdCfg {
  static constexpr int kQT = kBwdQTile;                 // 128 query rows per iteration
  static constexpr int kKBytes = kTile * D * 2;         // K or V tile
  static constexpr int kQBytes = kQT * D * 2;           // Q_i or dO_i tile
  static constexpr int kBoxBytes = kTile * 128;         // one 64-column (128 B) box of a 128-row tile
#if SRA_BWD_BULK
  static constexpr int kQStages = 2;                    // Q_i ring (Q_i is read first by S^T(i), last by dK(i))
  static constexpr int kStageBytes = SRA_BWD_BULK_NB * (kBwdQTile / SRA_BWD_BULK_NQ) * D * 4;  // dQ staging: kNB x [kRP queries][D] fp32
#else
  static constexpr int kQStages = 3;
  static constexpr int kStageBytes = 0;
#endif
  static constexpr int kVecSlots = 2;                   // {-LSE_i log2e [128], D_i [128]} ring
  static constexpr int kDsBytes = kTile * kQT * 2;      // dS^T tile: 2 boxes of [128 keys][64 queries] bf16
  static constexpr int kVecBytes = kVecSlots * 2 * kQT * 4;
  static constexpr int kNumBars = 1 + 2 * kQStages + 2 + 2 * kVecSlots + 8;
  static constexpr int kSmemBytes = 2 * kKBytes + (kQStages + 1) * kQBytes + kDsBytes + kVecBytes + kNumBars * 8 + 16 + kStageBytes + (kStageBytes ? 128 : 0);
  // kSplit compute warps per SM sub-partition share a key row's 128 query columns.  Warps [0, 4 kSplit): compute (P^T,
  // dS^T; dV epilogue) | next 4: dQ^T drain (dK epilogue) | then the MMA issuer, the loader and 2 idle warps (the register
  // file is allocated per 4 warps).  A drain thread holds a whole 128-column row of dQ^T, so that the TMEM columns are
  // released before its first reduction: kSplit = 1 is a 384-thread launch (168 registers each); kSplit = 2 is a
  // 512-thread launch whose 128 registers per thread are re-cut per warpgroup with setmaxnreg.
  static constexpr int kSplit = SRA_BWD_SPLIT;
  static constexpr int kCols = kQT / kSplit;            // query columns per compute thread
  static constexpr int kComputeWarps = 4 * kSplit;
  static constexpr int kMmaWarp = kComputeWarps + 4, kLoadWarp = kComputeWarps + 5;
  static constexpr int kThreads = (kComputeWarps + 8) * 32;
  static constexpr bool kRecut = kSplit == 2;
  static constexpr int kRegsCompute = 120, kRegsDrain = 160, kRegsMisc = 80;  // kSplit = 2: (2 x 120 + 160 + 80) x 128 <= 64 K
  // TMEM columns: S^T (P^T bf16 over it) | dP^T (later dQ^T) | dV | dK
  static constexpr int kColS = 0, kColDP = 128, kColDV = 256, kColDK = 256 + D;
  static_assert(kSmemBytes <= 232448, "shared memory budget");
};

template <int D>
__device__ __forceinline__ void bwd_load_tile(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int row, int h, int b,
                                              bool head_major) {
#pragma unroll
  for (int x = 0; x < D / 64; ++x) {
    if (head_major)
      tma_load_4d(dst + x * BwdCfg<D>::kBoxBytes, tm, bar, x * 64, row, h, b);
    else
      tma_load_4d(dst + x * BwdCfg<D>::kBoxBytes, tm, bar, x * 64, h, row, b);
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
  constexpr int ST = C::kQStages;
  constexpr int VS = C::kVecSlots;
  extern __shared__ __align__(1024) uint8_t smem_raw[];  // 128-byte-swizzled tiles need 1024-byte alignment
  const uint32_t smem_base = smem_u32(smem_raw);
  if ((smem_base & 1023u) != 0) __trap();
  const uint32_t sK = smem_base;
  const uint32_t sV = sK + C::kKBytes;                          // directly behind K (the d = 64 dQ^T MMA runs on into it)
  const uint32_t sQ = sV + C::kKBytes;                          // [ST] Q_i
  const uint32_t sDO = sQ + ST * C::kQBytes;                    // dO_i
  const uint32_t sDs = sDO + C::kQBytes;                        // dS^T
  const uint32_t sVec = sDs + C::kDsBytes;                      // [VS] x {-lse2[128], delta[128]}
  const uint32_t sBar = sVec + C::kVecBytes;
  const uint32_t bar_kv_full = sBar;
  const uint32_t bar_q_full = sBar + 8;                         // [ST] TMA transaction
  const uint32_t bar_q_empty = bar_q_full + 8 * ST;             // [ST] commit after dK(i)
  const uint32_t bar_do_full = bar_q_empty + 8 * ST;
  const uint32_t bar_do_empty = bar_do_full + 8;                // commit after dV(i)
  const uint32_t bar_vec_full = bar_do_empty + 8;               // [VS] loader warp
  const uint32_t bar_vec_empty = bar_vec_full + 8 * VS;         // [VS] 8 compute warps, after dS(i)
  const uint32_t bar_s_full = bar_vec_empty + 8 * VS;
  const uint32_t bar_p_full = bar_s_full + 8;                   // 8 compute warps
  const uint32_t bar_dp_full = bar_p_full + 8;
  const uint32_t bar_ds_full = bar_dp_full + 8;                 // 8 compute warps
  const uint32_t bar_dq_full = bar_ds_full + 8;
  const uint32_t bar_dq_empty = bar_dq_full + 8;                // 4 drain warps
  const uint32_t bar_acc_full = bar_dq_empty + 8;
  const uint32_t s_tmem_ptr = bar_acc_full + 16;
  const uint32_t sStage = (s_tmem_ptr + 16 + 127) & ~127u;      // (SRA_BWD_BULK) dQ staging: [64 queries][D] fp32
  uint32_t* tmem_ptr_generic = reinterpret_cast<uint32_t*>(smem_raw + (s_tmem_ptr - smem_base));

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const BwdItem item = p.items[blockIdx.x + size_t(blockIdx.z) * p.item_batch_stride];
  if (item.k_rows == 0) return;  // padding of a per-sample schedule (whole CTA, nothing is set up yet)
  const int h = blockIdx.y;
  const int b = blockIdx.z;
  const int bh = b * p.heads + h;
  const int n0 = (item.g_len + QT - 1) / QT;  // generation query tiles that see this key tile
  const int n1 = (item.seg1_len + QT - 1) / QT;
  const int n_it = n0 + n1;
  // Every CTA of a head walks the same query tiles and adds into the same dQ rows; starting each CTA at a different
  // tile spreads the L2 reductions over addresses (the L2 serialises atomics per address) - the order of a
  // CTA's query tiles is otherwise free.
  const int rot = int((blockIdx.x * 2654435761u) >> 8) % n_it;
  auto tile_of = [&](int i) { const int x = i + rot; return x >= n_it ? x - n_it : x; };
#ifdef SRA_BWD_TRACE
  const bool tr_on = blockIdx.x == 5 && blockIdx.y == 0 && blockIdx.z == 0 && (threadIdx.x & 31) == 0;
#endif

  if (threadIdx.x == 0) {
    mbar_init(bar_kv_full, 1);
    for (int s = 0; s < ST; ++s) {
      mbar_init(bar_q_full + 8 * s, 1);
      mbar_init(bar_q_empty + 8 * s, 1);
    }
    mbar_init(bar_do_full, 1);
    mbar_init(bar_do_empty, 1);
    for (int s = 0; s < VS; ++s) {
      mbar_init(bar_vec_full + 8 * s, 1);
      mbar_init(bar_vec_empty + 8 * s, C::kComputeWarps);
    }
    mbar_init(bar_s_full, 1);
    mbar_init(bar_p_full, C::kComputeWarps);
    mbar_init(bar_dp_full, 1);
    mbar_init(bar_ds_full, C::kComputeWarps);
    mbar_init(bar_dq_full, 1);
    mbar_init(bar_dq_empty, 4);
    mbar_init(bar_acc_full, 1);
    fence_mbar_init();
  }
  if (warp == C::kLoadWarp && lane == 0) {
    tma_prefetch_desc(&tm_q_gen);
    tma_prefetch_desc(&tm_do_gen);
    tma_prefetch_desc(item.k_is_ref ? &tm_k_ref : &tm_k_gen);
    tma_prefetch_desc(item.k_is_ref ? &tm_v_ref : &tm_v_gen);
  }
  if (warp == C::kMmaWarp) tmem_alloc(s_tmem_ptr, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr_generic;

  if (warp < C::kComputeWarps) {
    // ================================================= compute warps (thread = key = TMEM lane)
    // Warps w and w + 4 sit on the same SM sub-partition and own the same 32 keys; warp w takes query columns [0, 64) of
    // every tile, warp w + 4 columns [64, 128).  Per tile: P^T = exp2(S^T sl2 - LSE log2e) -> bf16 -> TMEM (the A operand
    // of dV) and kept in registers; then, once dP^T has landed, dS^T = P^T o (dP^T - D) -> bf16 -> the swizzled
    // shared-memory tile that is the A operand of dK and the B operand of dQ^T.  A single warp is dispatch-bound on its
    // own instruction stream (MUFU.EX2 8 cycles, FFMA2 / FADD2 ~3.5, measured); two per sub-partition overlap.
    if (C::kRecut) reg_dec<C::kRegsCompute>();
    constexpr int NC = C::kCols;
    const int hh = warp >> 2;
    const int key = (warp & 3) * 32 + lane;
    const bool key_valid = key < item.k_rows;
    const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + lane_off + C::kColS + hh * NC;
    const uint32_t tDP = tmem + lane_off + C::kColDP + hh * NC;
    uint8_t* const ds_row_g = smem_raw + (sDs - smem_base) + (hh * NC / 64) * C::kBoxBytes + key * 128;  // box x = queries [64 x, +64)
    const float sl2 = p.scale_log2;
    const uint64_t sl2_2 = pack2(sl2, sl2);
    for (int it = 0; it < n_it; ++it) {
      const int vs = it % VS;
      // -lse2 of this warp's queries; delta at + QT floats.  Plain (non-volatile) shared-memory loads, so that the
      // compiler batches them ahead of the arithmetic instead of exposing one load latency per four elements.
      const float4* vec = reinterpret_cast<const float4*>(smem_raw + (sVec - smem_base) + vs * (2 * QT * 4) + hh * NC * 4);
      const int tq = tile_of(it);
      const int valid_h = (tq < n0 ? min(QT, item.g_len - tq * QT) : min(QT, item.seg1_len - (tq - n0) * QT)) - NC * hh;
      if ((warp & 3) == 0) TR(1 + hh, 0);
      mbar_wait(bar_vec_full + 8 * vs, (it / VS) & 1);  // acquire the loader's -lse2 / delta stores
      mbar_wait(bar_s_full, it & 1);
      if ((warp & 3) == 0) TR(1 + hh, 1);
      tc_fence_after();
      // The columns stream through two 32-column register buffers: the tcgen05.ld of the next chunk is in flight
      // while this one is exponentiated.
      uint32_t sv[2][32];
      uint32_t pk[NC / 2];
      tmem_ld32(tS, sv[0]);
#pragma unroll
      for (int c = 0; c < NC / 32; ++c) {
        tmem_wait_ld();
        if (c + 1 < NC / 32) tmem_ld32(tS + (c + 1) * 32, sv[(c + 1) & 1]);
        const uint32_t(&sc)[32] = sv[c & 1];
#pragma unroll
        for (int q4 = 0; q4 < 8; ++q4) {
#ifdef SRA_BWD_NOVEC  // (ablation builds only: no shared-memory loads of the row constants, results are wrong)
          const float4 nl = make_float4(-8.f, -8.f, -8.f, -8.f);
#else
          const float4 nl = vec[c * 8 + q4];
#endif
          const uint64_t x01 = fma2(pack2(__uint_as_float(sc[q4 * 4 + 0]), __uint_as_float(sc[q4 * 4 + 1])), sl2_2, pack2(nl.x, nl.y));
          const uint64_t x23 = fma2(pack2(__uint_as_float(sc[q4 * 4 + 2]), __uint_as_float(sc[q4 * 4 + 3])), sl2_2, pack2(nl.z, nl.w));
          float p0, p1, p2, p3;
          if ((((2 * q4) * SRA_BWD_EMU) & 7) < SRA_BWD_EMU) ex2_emu2(x01, p0, p1);
          else { float a, bb; unpack2(x01, a, bb); p0 = ex2(a); p1 = ex2(bb); }
          if ((((2 * q4 + 1) * SRA_BWD_EMU) & 7) < SRA_BWD_EMU) ex2_emu2(x23, p2, p3);
          else { float a, bb; unpack2(x23, a, bb); p2 = ex2(a); p3 = ex2(bb); }
          pk[c * 16 + q4 * 2 + 0] = pack_bf16(p0, p1);
          pk[c * 16 + q4 * 2 + 1] = pack_bf16(p2, p3);
        }
      }
      if (valid_h < NC) {
        // ragged last query tile of a segment: the rows behind it belong to a neighbour (or are TMA zero fill);
        // their P^T columns are forced to 0 by selection, whatever the scores were
#pragma unroll
        for (int k = 0; k < NC / 2; ++k) {
          if (2 * k >= valid_h) pk[k] = 0u;
          else if (2 * k + 1 >= valid_h) pk[k] &= 0xffffu;
        }
      }
      // P^T: bf16 pairs over the first half of the score columns this warp has read (columns [kCols hh, + kCols / 2) of
      // S), so no warp of a key row overwrites scores a partner may still be loading
#pragma unroll
      for (int x = 0; x < NC / 64; ++x) tmem_st32(tS + x * 32, *reinterpret_cast<uint32_t(*)[32]>(&pk[x * 32]));
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_p_full);
      if ((warp & 3) == 0) TR(1 + hh, 2);
      // ---- dS^T(it)
      mbar_wait(bar_dp_full, it & 1);  // dP^T(it) has landed; every earlier MMA (dQ^T / dK of it-1, readers of sDs) is done
      if ((warp & 3) == 0) TR(1 + hh, 3);
      tc_fence_after();
      // dS^T pair = P^T pair (bf16x2, as the dV MMA consumes it) * bf16x2(dP^T pair - D pair): one packed subtract, one
      // conversion and one packed bf16 multiply per two elements.  (The selections of the masked form cost an
      // instruction per pair, so the aligned interior takes the plain loop.)
      auto form_ds = [&](auto masked) {
        tmem_ld32(tDP, sv[0]);
#pragma unroll
        for (int c = 0; c < NC / 32; ++c) {
          tmem_wait_ld();
          if (c + 1 < NC / 32) tmem_ld32(tDP + (c + 1) * 32, sv[(c + 1) & 1]);
          const uint32_t(&dp)[32] = sv[c & 1];
#pragma unroll
          for (int e = 0; e < 4; ++e) {  // 8 queries = one 16-byte chunk of the dS^T row
#ifdef SRA_BWD_NOVEC
            const float4 d0 = make_float4(0.f, 0.f, 0.f, 0.f), d1 = d0;
#else
            const float4 d0 = vec[QT / 4 + c * 8 + e * 2];
            const float4 d1 = vec[QT / 4 + c * 8 + e * 2 + 1];
#endif
            const uint64_t dl[4] = {pack2(d0.x, d0.y), pack2(d0.z, d0.w), pack2(d1.x, d1.y), pack2(d1.z, d1.w)};
            uint32_t w[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const int q = c * 32 + e * 8 + 2 * k;  // query column of this half
              float a, bb;
              unpack2(sub2(pack2(__uint_as_float(dp[e * 8 + 2 * k]), __uint_as_float(dp[e * 8 + 2 * k + 1])), dl[k]), a, bb);
              w[k] = mul_bf16x2(pk[q >> 1], pack_bf16(a, bb));
              if (decltype(masked)::value) {
                if (!key_valid || q >= valid_h) w[k] = 0u;
                else if (q + 1 >= valid_h) w[k] &= 0xffffu;
              }
            }
            const int ch16 = c * 4 + e;  // 16-byte chunk of this thread's dS^T row range
            *reinterpret_cast<uint4*>(ds_row_g + (ch16 / 8) * C::kBoxBytes + (((ch16 & 7) ^ (key & 7)) << 4)) =
                make_uint4(w[0], w[1], w[2], w[3]);
          }
        }
      };
      if (__any_sync(0xffffffffu, !key_valid) || valid_h < NC) form_ds(std::true_type{}); else form_ds(std::false_type{});
      tc_fence_before();  // the dP^T columns may be overwritten by dQ^T(it) once ds_full completes
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(bar_ds_full);
        mbar_arrive(bar_vec_empty + 8 * vs);
      }
      if ((warp & 3) == 0) TR(1 + hh, 4);
    }
    // ---------------------------------------------------- epilogue: dV (lanes = keys), D / kSplit columns per warp
    mbar_wait(bar_acc_full, 0);
    tc_fence_after();
    {
      const int n_tok = item.k_is_ref ? p.n_ref : p.n_gen;
      const int grow = item.k_row0 + key;
      __nv_bfloat16* base = item.k_is_ref ? p.dv_ref : p.dv_gen;
      uint4* orow = reinterpret_cast<uint4*>(base + ((size_t(b) * n_tok + grow) * p.heads + h) * D + hh * (D / C::kSplit));
#pragma unroll
      for (int c = 0; c < D / C::kSplit / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(tmem + lane_off + C::kColDV + hh * (D / C::kSplit) + c * 32, o);
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
  } else if (warp < C::kComputeWarps + 4) {
    // ================================================= drain warps: dQ^T (thread = d = TMEM lane), then the dK epilogue
    if (C::kRecut) reg_inc<C::kRegsDrain>();
    const int wq = warp - C::kComputeWarps;
    const int key = wq * 32 + lane;
    const bool key_valid = key < item.k_rows;
    const uint32_t lane_off = uint32_t(wq * 32) << 16;
    for (int it = 0; it < n_it; ++it) {
      const QTile qt = q_tile_of(tile_of(it), n0, item, p.n_gen);
      if (wq == 0) TR(3, 0);
      mbar_wait(bar_dq_full, it & 1);
      if (wq == 0) TR(3, 1);
      tc_fence_after();
      // All 128 columns of dQ_it^T are taken into registers first, so that the TMEM columns are released (dq_empty)
      // before the first reduction - the reductions run at the L2's rate, far longer than dP^T(it+1) may wait.
      const int drow = key;
      uint32_t r[4][32];
#pragma unroll
      for (int x = 0; x < 4; ++x) tmem_ld32(tmem + lane_off + C::kColDP + x * 32, r[x]);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_dq_empty);  // dQ^T(it) is in registers: the columns are free for dP^T(it+1)
      if (wq == 0) TR(3, 2);
#if SRA_BWD_BULK
      // dQ_it leaves as kNQ bulk reductions of 128 / kNQ query rows each: registers -> shared-memory staging [query][d]
      // (thread = d, so the 32 lanes of a store hit 32 consecutive words: conflict-free) -> cp.reduce.async.bulk .add.f32
      // into the workspace rows of the tile, which are contiguous.  The reductions go through the TMA unit, not through the
      // memory-instruction queue the compute warps' tcgen05.ld / st and shared-memory stores need (per-thread
      // red.global.add.f32 had to be paced to 18 B/clk/SM for that reason; the L2 takes 23-24 from either source).  kNB
      // staging buffers: the stores of piece q overlap the bulk reads of the pieces before it; a buffer is rewritten once
      // the reduction issued kNB pieces earlier has read it.  (Many key tiles add into the same rows: the summation
      // order is not deterministic - SURVEY.md 8c A13.)
      constexpr int kNQ = SRA_BWD_BULK_NQ, kNB = SRA_BWD_BULK_NB, kRP = QT / kNQ;
      static_assert(kNB * kRP * D * 4 <= C::kStageBytes, "staging budget");
#pragma unroll
      for (int qr = 0; qr < kNQ; ++qr) {
        const uint32_t stg = sStage + (qr % kNB) * (kRP * D * 4);
        if (wq == 0 && lane == 0) tma_wait_group_read<kNB - 1>();
        named_bar_sync(1, 128);
        if (drow < D) {
#pragma unroll
          for (int cc = 0; cc < kRP; ++cc) {
            const int col = qr * kRP + cc;
            st_shared_f32(stg + (cc * D + drow) * 4, __uint_as_float(r[col >> 5][col & 31]));
          }
        }
        fence_proxy_async_smem();
        named_bar_sync(1, 128);
        if (wq == 0 && lane == 0) {
          const int rows = min(kRP, qt.valid - qr * kRP);
          if (rows > 0) bulk_reduce_add_f32(p.dq_ws + (size_t(bh) * p.n_pad + qt.cat0 + qr * kRP) * D, stg, uint32_t(rows) * D * 4);
          tma_commit_group();
        }
      }
#else
      // (A/B form: dQ_it^T straight from registers - for a fixed query the 32 lanes of a warp hold 32 consecutive d, so each
      //  red.global.add.f32 is one coalesced 128-byte reduction)
      float* dq_row = p.dq_ws + (size_t(bh) * p.n_pad + qt.cat0) * D + drow;
      if (drow < D) {
        if (qt.valid == QT) {
          // The reductions share each sub-partition's memory-instruction queue with the compute warp's tcgen05.ld / st and
          // shared-memory accesses; issued back to back they fill it (the LSU -> L2 path drains ~22 B/clk/SM) and the
          // compute warp stalls behind them.  They are paced instead: groups of 8, kRedGap cycles apart.
          long long t_next = clock64();
#pragma unroll
          for (int x = 0; x < 4; ++x)
#pragma unroll
            for (int c = 0; c < 32; ++c) {
              if (SRA_BWD_RED_GAP > 0 && (c & 7) == 0) {
                while (clock64() < t_next) { }
                t_next += 8 * SRA_BWD_RED_GAP;
              }
#ifndef SRA_BWD_NORED  // (ablation builds only: drop the reductions, dQ is then wrong)
              red_add_f32(dq_row + (x * 32 + c) * D, __uint_as_float(r[x][c]));
#else
              if (r[x][c] == 0x7fc12345u) red_add_f32(dq_row, 1.f);
#endif
            }
        } else {
#pragma unroll
          for (int x = 0; x < 4; ++x)
#pragma unroll
            for (int c = 0; c < 32; ++c)
              if (x * 32 + c < qt.valid) red_add_f32(dq_row + (x * 32 + c) * D, __uint_as_float(r[x][c]));
        }
      }
#endif
      if (wq == 0) TR(3, 3);
    }
#if SRA_BWD_BULK
    if (wq == 0 && lane == 0) tma_wait_group<0>();
#endif
    // ---------------------------------------------------- epilogue: dK = scale * acc (lanes = keys)
    mbar_wait(bar_acc_full, 0);
    tc_fence_after();
    {
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
    if (C::kRecut) reg_dec<C::kRegsMisc>();
    if (warp == C::kLoadWarp) {
      // ================================================= loader: K/V once, then per tile Q_i (3 stages), {-lse2, delta}
      // (2 slots, written by the 32 lanes) and dO_i (one buffer, free once dV(i-1) is done)
      const bool k_hm = item.k_is_ref && p.ref_kv_head_major;
      // Ragged tiles whose segment ends inside its tensor go through the maps bounded at the segment end
      // (sra_common.h BoundMaps): the rows behind the end read as zero, not as the neighbouring block's or frame's.
      const CUtensorMap* tk = item.k_is_ref ? &tm_k_ref : &tm_k_gen;
      const CUtensorMap* tv = item.k_is_ref ? &tm_v_ref : &tm_v_gen;
      if (p.bound.maps != nullptr && item.k_rows < kTile) {
        const int ix = bound_index(p.bound, item.k_is_ref != 0, p.item_batch_stride ? b : 0, item.k_row0 + item.k_rows);
        if (ix >= 0) { tk = p.bound.maps + (item.k_is_ref ? 6 : 2) * p.bound.n_total + ix; tv = tk + p.bound.n_total; }
      }
      // (the ragged last query tile of a segment: searched when it comes up, once per segment)
      auto tail_q = [&](const QTile& qt) -> const CUtensorMap* {
        if (p.bound.maps == nullptr || qt.valid == QT) return nullptr;
        const int ix = bound_index(p.bound, qt.is_ref != 0, p.item_batch_stride ? b : 0, qt.row0 + qt.valid);
        return ix >= 0 ? p.bound.maps + (qt.is_ref ? 4 : 0) * p.bound.n_total + ix : nullptr;
      };
      if (lane == 0) {
        mbar_arrive_expect_tx(bar_kv_full, 2 * C::kKBytes);
        bwd_load_tile<D>(sK, tk, bar_kv_full, item.k_row0, h, b, k_hm);
        bwd_load_tile<D>(sV, tv, bar_kv_full, item.k_row0, h, b, k_hm);
      }
      const float* lse2 = p.lse2 + size_t(bh) * p.n_pad;
      const float* delta = p.delta + size_t(bh) * p.n_pad;
      for (int it = 0; it < n_it; ++it) {
        const int s = it % ST, vs = it % VS;
        const QTile qt = q_tile_of(tile_of(it), n0, item, p.n_gen);
        const CUtensorMap* tq_tail = tail_q(qt);  // Q map; the dO map of the same end sits n_total entries behind it
        // the tile's row constants, fetched before any wait so that their latency hides behind it
        float nl[QT / 32], dl[QT / 32];
#pragma unroll
        for (int r = 0; r < QT / 32; ++r) {
          const int row = r * 32 + lane;
          const bool ok = row < qt.valid;
          nl[r] = ok ? -__ldg(lse2 + qt.cat0 + row) : -INFINITY;  // -inf => P = 0 for rows outside the tile
          dl[r] = ok ? __ldg(delta + qt.cat0 + row) : 0.f;
        }
        TR(4, 0);
        mbar_wait(bar_q_empty + 8 * s, ((it / ST) & 1) ^ 1);
        TR(4, 1);
        if (lane == 0) {
          mbar_arrive_expect_tx(bar_q_full + 8 * s, C::kQBytes);
          bwd_load_tile<D>(sQ + s * C::kQBytes, tq_tail ? tq_tail : (qt.is_ref ? &tm_q_ref : &tm_q_gen), bar_q_full + 8 * s, qt.row0, h, b, false);
        }
        mbar_wait(bar_vec_empty + 8 * vs, ((it / VS) & 1) ^ 1);
        TR(4, 2);
        const uint32_t vec = sVec + vs * (2 * QT * 4);
#pragma unroll
        for (int r = 0; r < QT / 32; ++r) {
          st_shared_f32(vec + (r * 32 + lane) * 4, nl[r]);
          st_shared_f32(vec + QT * 4 + (r * 32 + lane) * 4, dl[r]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_vec_full + 8 * vs);
        mbar_wait(bar_do_empty, (it & 1) ^ 1);
        TR(4, 3);
        if (lane == 0) {
          mbar_arrive_expect_tx(bar_do_full, C::kQBytes);
          bwd_load_tile<D>(sDO, tq_tail ? tq_tail + p.bound.n_total : (qt.is_ref ? &tm_do_ref : &tm_do_gen), bar_do_full, qt.row0, h, b, false);
        }
      }
    } else if (warp == C::kMmaWarp && elect_one()) {
      // ================================================= MMA issuer
      constexpr uint32_t idesc_st = make_idesc_bf16(kTile, QT, 0, 0);   // S^T, dP^T : [128 x 128], A, B K-major, K = d
      constexpr uint32_t idesc_acc = make_idesc_bf16(kTile, D, 0, 1);   // dV, dK    : [128 x D], B MN-major, K = 128 queries
      // dQ^T : [D x 128], A, B MN-major, K = 128 keys.  With D = 64 the MMA is still issued with M = 128 (the M = 64
      // accumulator layout differs): its A operand then runs on from the K tile into the V tile behind it, TMEM lanes
      // [64, 128) receive finite garbage (V^T dS^T) and the drain ignores them.
      constexpr uint32_t idesc_dq = make_idesc_bf16(kTile, QT, 1, 1);
      const uint32_t tS = tmem + C::kColS, tDP = tmem + C::kColDP, tDV = tmem + C::kColDV, tDK = tmem + C::kColDK;
      // Descriptor low words (start address, LBO); stepping along K or to another stage is one 32-bit add.
      constexpr uint32_t kHi = desc_hi_sw128(1024);
      const uint32_t k_km = desc_lo(sK, 16), v_km = desc_lo(sV, 16);             // K, V as K-major A operands
      const uint32_t k_mn = desc_lo(sK, C::kBoxBytes);                           // K as MN-major A operand (dQ^T)
      const uint32_t q_km = desc_lo(sQ, 16), do_km = desc_lo(sDO, 16);           // Q_i / dO_i as K-major B operands
      const uint32_t q_mn = desc_lo(sQ, C::kBoxBytes), do_mn = desc_lo(sDO, C::kBoxBytes);  // ... as MN-major B operands
      const uint32_t ds_km = desc_lo(sDs, 16), ds_mn = desc_lo(sDs, C::kBoxBytes);
      // [128 keys x 128 queries] = A[keys][d] (K-major) * B[queries][d]^T (K-major)
      auto issue_kq = [&](uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo) {
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t off = ((kk / 4) * C::kBoxBytes + (kk % 4) * 32) >> 4;
          umma_ss(d_tmem, desc64(a_lo + off, kHi), desc64(b_lo + off, kHi), idesc_st, kk > 0);
        }
      };
      mbar_wait(bar_kv_full, 0);
      mbar_wait(bar_q_full, 0);
      tc_fence_after();
      issue_kq(tS, k_km, q_km);
      umma_commit(bar_s_full);
      mbar_wait(bar_do_full, 0);
      tc_fence_after();
      issue_kq(tDP, v_km, do_km);
      umma_commit(bar_dp_full);
      for (int it = 0; it < n_it; ++it) {
        const int s = it % ST;
        const uint32_t oQ = (s * C::kQBytes) >> 4;
        const bool more = it + 1 < n_it;
        // dV += P^T(it) dO_it : A = P^T bf16 from TMEM (16 queries = 8 columns per step; the pairs of compute warp
        // group x sit at column kCols x), B = dO_it [queries][d] MN-major
        TR(0, 0);
        mbar_wait(bar_p_full, it & 1);
        TR(0, 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < QT / 16; ++kk)
          umma_ts(tDV, tS + ((kk * 16) / C::kCols) * C::kCols + ((kk * 16) % C::kCols) / 2, desc64(do_mn + ((kk * 2048) >> 4), kHi), idesc_acc,
                  (it > 0 || kk > 0) ? 1u : 0u);
        umma_commit(bar_do_empty);  // dO_it has been read by dP^T(it) and dV(it)
        TR(0, 2);
        if (more) {
          // S^T(it+1) overwrites S^T / P^T(it): in order behind dV(it); the compute warps have read S^T(it) (p_full)
          const int s1 = (it + 1) % ST;
          mbar_wait(bar_q_full + 8 * s1, ((it + 1) / ST) & 1);
          TR(0, 3);
          tc_fence_after();
          issue_kq(tS, k_km, q_km + ((s1 * C::kQBytes) >> 4));
          umma_commit(bar_s_full);
          TR(0, 4);
        }
        mbar_wait(bar_ds_full, it & 1);  // dS^T(it) in shared memory; dP^T(it) has been read out of TMEM
        TR(0, 5);
        tc_fence_after();
        // dQ_it^T = K^T dS^T(it) : A = K [keys][d] MN-major, B = dS^T [keys][queries] MN-major, K = 128 keys; lands over
        // dP^T(it).  Issued before dK so that its drain runs under the dK MMA.
#pragma unroll
        for (int kk = 0; kk < kTile / 16; ++kk)
          umma_ss(tDP, desc64(k_mn + ((kk * 2048) >> 4), kHi), desc64(ds_mn + ((kk * 2048) >> 4), kHi), idesc_dq, kk > 0);
        umma_commit(bar_dq_full);
        TR(0, 6);
        // dK += dS^T(it) Q_it : A = dS^T [keys][queries] K-major (two 64-query boxes), B = Q_it [queries][d] MN-major
#pragma unroll
        for (int kk = 0; kk < QT / 16; ++kk)
          umma_ss(tDK, desc64(ds_km + (((kk / 4) * C::kBoxBytes + (kk % 4) * 32) >> 4), kHi),
                  desc64(q_mn + oQ + ((kk * 2048) >> 4), kHi), idesc_acc, (it > 0 || kk > 0) ? 1u : 0u);
        umma_commit(bar_q_empty + 8 * s);
        TR(0, 7);
        if (more) {
          mbar_wait(bar_do_full, (it + 1) & 1);
          TR(0, 8);
          mbar_wait(bar_dq_empty, it & 1);
          TR(0, 9);  // dQ^T(it) is in registers: the columns are free for dP^T(it+1)
          tc_fence_after();
          issue_kq(tDP, v_km, do_km);
          umma_commit(bar_dp_full);
          TR(0, 10);
        }
      }
      umma_commit(bar_acc_full);
    }
  }
  __syncthreads();
  if (warp == C::kMmaWarp) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

// a6: D_i = sum_c dO_ic O_ic and LSE_i * log2(e) for rows [G ; R].  A row of O or dO is D bf16 = D / 8 16-byte vectors:
// D / 8 lanes per row (16 for d = 128, 8 for d = 64), 32 / (D / 8) rows per warp pass, 16 bytes per lane per tensor.
template <int D>
__global__ void sra_bwd_preprocess_kernel(const __nv_bfloat16* __restrict__ o_gen, const __nv_bfloat16* __restrict__ do_gen,
                                          const float* __restrict__ lse_gen, const __nv_bfloat16* __restrict__ o_ref,
                                          const __nv_bfloat16* __restrict__ do_ref, const float* __restrict__ lse_ref,
                                          float* __restrict__ delta, float* __restrict__ lse2, int B, int H, int n_gen,
                                          int n_ref, int n_pad) {
  constexpr int LPR = D / 8;        // lanes per row
  constexpr int RPW = 32 / LPR;     // rows per warp pass
  const int lane = threadIdx.x & 31;
  const int sub = lane / LPR, li = lane % LPR;
  const size_t warp_id = (blockIdx.x * size_t(blockDim.x) + threadIdx.x) >> 5;
  const size_t n_warps = (gridDim.x * size_t(blockDim.x)) >> 5;
  const size_t n_cat = size_t(n_gen) + n_ref;
  const size_t total = size_t(B) * n_cat * H;
  for (size_t r0 = warp_id * RPW; r0 < total; r0 += n_warps * RPW) {
    const size_t r = r0 + sub;
    const bool ok = r < total;
    const size_t rr = ok ? r : total - 1;
    const int h = int(rr % H);
    const size_t t = rr / H;
    const int n = int(t % n_cat);
    const int b = int(t / n_cat);
    const bool is_ref = n >= n_gen;
    const int row = is_ref ? n - n_gen : n;
    const int n_tok = is_ref ? n_ref : n_gen;
    const size_t off = ((size_t(b) * n_tok + row) * H + h) * D;
    const uint4 a = reinterpret_cast<const uint4*>((is_ref ? o_ref : o_gen) + off)[li];
    const uint4 c = reinterpret_cast<const uint4*>((is_ref ? do_ref : do_gen) + off)[li];
    const __nv_bfloat162* a2 = reinterpret_cast<const __nv_bfloat162*>(&a);
    const __nv_bfloat162* c2 = reinterpret_cast<const __nv_bfloat162*>(&c);
    float acc = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float2 x = __bfloat1622float2(a2[k]), y = __bfloat1622float2(c2[k]);
      acc = fmaf(x.x, y.x, acc);
      acc = fmaf(x.y, y.y, acc);
    }
#pragma unroll
    for (int m = LPR / 2; m > 0; m >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, m);
    if (ok && li == 0) {
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
  bool* configured = smem_configured_flag(D == 128 ? 4 : 5);  // per device
  if (!*configured) {
    cudaError_t e = cudaFuncSetAttribute(sra_bwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes);
    if (e != cudaSuccess) return e;
    *configured = true;
  }
  dim3 grid(p.n_items, p.heads, p.batch);
  sra_bwd_kernel<D><<<grid, C::kThreads, C::kSmemBytes, stream>>>(m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], p);
  return cudaGetLastError();
}

#ifdef SRA_BWD_TRACE
extern "C" void sra_dbg_set_bwd_trace(long long* p) { cudaMemcpyToSymbol(g_bwd_trace, &p, sizeof(p)); }
#endif
template cudaError_t launch_bwd<64>(const CUtensorMap*, const BwdParams&, cudaStream_t);
template cudaError_t launch_bwd<128>(const CUtensorMap*, const BwdParams&, cudaStream_t);

// ------------------------------------------------------------------------------------------------ host driver
static int run_backward_core(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream);

int run_backward(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream) {
  const sra_config& c = ctx->cfg;
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
  // the workspace is sized once, for the unmasked reference (sra_reserve(SRA_RESERVE_BACKWARD), or here on first use)
  if (int rc = reserve(ctx, SRA_RESERVE_BACKWARD)) return rc;
  if (int rc = sync_schedule(ctx, stream)) return rc;
  e = cudaMemsetAsync(ctx->ws_dq, 0, dq_bytes, stream);
  if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "dQ workspace memset");

  {  // a6
    const size_t rows = size_t(B) * n_cat * H;
    const int threads = 256;
    const int blocks = grid_for(ctx, rows * (d / 8), threads, 32);  // d / 8 lanes per row
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
  p.items = ctx->d_bwd_items[ctx->sched_buf];
  p.n_items = ctx->bwd_stride;
  p.item_batch_stride = ctx->n_masks > 1 ? ctx->bwd_stride : 0;
  p.heads = H; p.batch = B; p.n_gen = c.n_gen; p.n_ref = nr; p.n_pad = n_pad;
  p.scale = ctx->scale;
  p.scale_log2 = ctx->scale * 1.4426950408889634f;
  p.lse2 = ctx->ws_lse2; p.delta = ctx->ws_delta; p.dq_ws = ctx->ws_dq;
  p.dk_gen = static_cast<__nv_bfloat16*>(a->dk_gen); p.dv_gen = static_cast<__nv_bfloat16*>(a->dv_gen);
  p.dk_ref = static_cast<__nv_bfloat16*>(a->dk_ref); p.dv_ref = static_cast<__nv_bfloat16*>(a->dv_ref);
  p.ref_kv_head_major = use_cache ? 1 : 0;
  {
    const void* kr = has_ref ? (use_cache ? ctx->cache_k : a->k_ref) : nullptr;
    const void* vr = has_ref ? (use_cache ? ctx->cache_v : a->v_ref) : nullptr;
    const sra_ctx::BoundRole roles[8] = {
        {a->q_gen, c.n_gen, false, false, kBwdQTile}, {a->do_gen, c.n_gen, false, false, kBwdQTile},
        {a->k_gen, c.n_gen, false, false, kTile},     {a->v_gen, c.n_gen, false, false, kTile},
        {has_ref ? a->q_ref : nullptr, nr, true, false, kBwdQTile}, {has_ref ? a->do_ref : nullptr, nr, true, false, kBwdQTile},
        {kr, nr, true, use_cache, kTile},             {vr, nr, true, use_cache, kTile}};
    if ((rc = bound_maps(ctx, ctx->bnd_bwd, roles, 8, stream, &p.bound))) return rc;
  }
  {
    KernelTimer kt(ctx, SRA_KERNEL_BWD_MAIN, stream);
    e = d == 128 ? launch_bwd<128>(m, p, stream) : launch_bwd<64>(m, p, stream);
  }
  if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "sra_bwd_kernel launch");
  ctx->launches += 1;

  {  // a8
    const size_t total = size_t(B) * H * n_cat * (d / 8);
    const int threads = 256;
    const int blocks = grid_for(ctx, total, threads, 32);
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
