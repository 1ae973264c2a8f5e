// SRA forward kernel for sm_100a.
//
// One CTA = one work item (a 256-row query slab of G or of one R block) x one (batch, head).
// The slab is two 128-row Q tiles that ping-pong on the tensor core:
//
//   warps 0-7   softmax: warps w and w + 4 share the 32 query rows (TMEM lanes) of sub-partition w & 3; warp w takes
//               key columns [0, 64) of every score tile, warp w + 4 columns [64, 128), for both Q tiles in turn
//   warp  8     MMA issuer (one elected thread): S_i = Q_i K_j^T (SS), O_i += P_i V_j (A = P from TMEM)
//   warp  9     TMA loader (one elected thread): Q once, then the K/V tile ring
//   warps 10-11 idle (they only pad the third warpgroup for setmaxnreg)
//
// TMEM (512 columns x 128 lanes x fp32): S0 @0, S1 @128, O0 @256, O1 @256+D.  P_i (bf16) overwrites S_i in two
// pieces, each written by the warp that read the scores underneath it: keys [0, 64) -> columns [0, 32) of S_i,
// keys [64, 128) -> columns [64, 96); the PV MMA takes its K steps from there.
// Masked tiles are never visited: the key-tile loop walks only the item's visible segments;
// only the last tile of a segment pays for a column mask (n_valid < 128).
//
// CG = 2 (head_dim 128, the default wherever two consecutive slabs see the same keys): a CTA PAIR - a cluster of two
// CTAs on one TPC - works on a 512-row slab (128-row tile t of the slab belongs to CTA t & 1, slot t >> 1) with
// tcgen05.mma.cta_group::2, M = 256: each MMA drives both SMs' tensor cores, rows [0, 128) of A / D in CTA 0's shared
// memory / TMEM, rows [128, 256) in CTA 1's.  The B operand is split between the two: CTA r loads keys [64 r, 64 r + 64)
// of every K tile (QK^T: N = 128 keys) and head-dim columns [64 r, 64 r + 64) of every V tile (PV: N = 128 columns), so
// each SM pulls HALF of the K/V bytes out of L2 and reads half of the B operand from shared memory; the hardware
// exchanges the halves inside the TPC.  Only the leader (CTA 0) issues MMAs; its tcgen05.commit is multicast to both
// CTAs' mbarriers, both CTAs' TMA loads report their bytes to the leader's kv_full barriers, and CTA 1's softmax
// warps arrive remotely on the leader's p_full barriers.
#include <algorithm>
#include <type_traits>

#include "ptx.cuh"
#include "sra_common.h"

namespace sra {

// Of every 8 column pairs of a score tile, this many take their exp2 on the FMA/ALU pipes
// (ex2_emu2) instead of MUFU: per key tile the two MMAs and the 16 K MUFU exponentials need the
// same number of SM cycles, so without the split the softmax sits on the critical path.
#ifndef SRA_FWD_EMU
#define SRA_FWD_EMU 3
#endif
constexpr int kEmuPairsPer8 = SRA_FWD_EMU;

// Development aid (-DSRA_FWD_TRACE): clock64 timestamps of the pipeline events of one CTA over a few key tiles.
#ifdef SRA_FWD_TRACE
__device__ long long* g_fwd_trace = nullptr;
#define FTR(role, step, ev)                                                                                         \
  do {                                                                                                              \
    if (ftr_on && (step) >= 100 && (step) < 108 && g_fwd_trace) g_fwd_trace[((role) * 8 + ((step) - 100)) * 16 + (ev)] = clock64(); \
  } while (0)
#else
#define FTR(role, step, ev) do { } while (0)
#endif

template <int D, int CG>
struct FwdCfg {
  static_assert(CG == 1 || (CG == 2 && D == 128), "the CTA-pair kernel is built for head_dim 128");
  static constexpr int kTileBytes = kTile * D * 2;          // one Q tile in smem
  static constexpr int kStageBytes = kTileBytes / CG;       // this CTA's share of a K or V tile
  static constexpr int kBoxes = D / 64;                      // 64-column (128 B) TMA boxes per tile
  static constexpr int kBoxBytes = kTile * 128;              // 16 KB: [128 rows][64 columns]
  static constexpr int kKRows = kTile / CG;                  // key rows of a K tile held by this CTA
  static constexpr int kKBoxBytes = kKRows * 128;            // [kKRows][64 columns]
  static constexpr int kStages = (D == 128) ? 5 * CG : 10;   // K/V ring depth (tiles)
  static constexpr int kNumBars = 1 + 2 * kStages + 6 + 4;
  static constexpr int kXchBytes = 2 * 2 * kTile * 4;       // (slot, half, row) floats swapped by the two threads of a row
  static constexpr int kSmemBytes = 2 * kTileBytes + kStages * kStageBytes + kNumBars * 8 + 16 + kXchBytes;
  static constexpr int kTmemCols = 512;
  static constexpr int kThreads = 384;
  static_assert(kSmemBytes <= 232448, "shared memory budget");
};

// One 128-row tile of a [.., d] tensor (Q; with CG = 1 also K and V): D / 64 boxes of [128 rows][64 columns].
template <int D, int CG>
__device__ __forceinline__ void load_tile(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int row, int h, int b,
                                          bool head_major) {
#pragma unroll
  for (int x = 0; x < D / 64; ++x) {
    const uint32_t dx = dst + x * FwdCfg<D, CG>::kBoxBytes;
    if (CG == 1) {
      if (head_major) tma_load_4d(dx, tm, bar, x * 64, row, h, b); else tma_load_4d(dx, tm, bar, x * 64, h, row, b);
    } else {
      if (head_major) tma_load_4d_pair(dx, tm, bar, x * 64, row, h, b); else tma_load_4d_pair(dx, tm, bar, x * 64, h, row, b);
    }
  }
}
// CTA-pair shares of a key tile.  K (B operand of QK^T, N = keys): this CTA's 64 keys, all of d, as two
// [64 rows][64 columns] boxes (the tensor map's box is 64 rows).  V (B operand of PV, N = head-dim columns): all
// 128 keys, this CTA's 64 columns - one ordinary [128 rows][64 columns] box.
template <int D>
__device__ __forceinline__ void load_k_half(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int row, int h, int b,
                                            bool head_major, int rank) {
#pragma unroll
  for (int x = 0; x < D / 64; ++x) {
    const uint32_t dx = dst + x * FwdCfg<D, 2>::kKBoxBytes;
    if (head_major) tma_load_4d_pair(dx, tm, bar, x * 64, row + 64 * rank, h, b);
    else tma_load_4d_pair(dx, tm, bar, x * 64, h, row + 64 * rank, b);
  }
}
template <int D>
__device__ __forceinline__ void load_v_half(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int row, int h, int b,
                                            bool head_major, int rank) {
  if (head_major) tma_load_4d_pair(dst, tm, bar, 64 * rank, row, h, b);
  else tma_load_4d_pair(dst, tm, bar, 64 * rank, h, row, b);
}

// Map of `role` bounded at `end_row`, or null (sra_common.h BoundMaps).
__device__ __forceinline__ const CUtensorMap* bound_lookup(const BoundMaps& bm, int role, bool is_ref, int mask, int end_row) {
  const int ix = bound_index(bm, is_ref, mask, end_row);
  return ix >= 0 ? bm.maps + role * bm.n_total + ix : nullptr;
}

template <int D, int CG>
__global__ void __launch_bounds__(FwdCfg<D, CG>::kThreads, 1)
    sra_fwd_kernel(const __grid_constant__ CUtensorMap tm_q_gen, const __grid_constant__ CUtensorMap tm_k_gen,
                   const __grid_constant__ CUtensorMap tm_v_gen, const __grid_constant__ CUtensorMap tm_q_ref,
                   const __grid_constant__ CUtensorMap tm_k_ref, const __grid_constant__ CUtensorMap tm_v_ref,
                   const FwdParams p) {
  using C = FwdCfg<D, CG>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];  // 128-byte-swizzled tiles need 1024-byte alignment
  const uint32_t smem_base = smem_u32(smem_raw);
  if ((smem_base & 1023u) != 0) __trap();
  const uint32_t sQ = smem_base;                         // 2 tiles
  const uint32_t sKV = smem_base + 2 * C::kTileBytes;    // kStages tiles
  const uint32_t sBar = sKV + C::kStages * C::kStageBytes;
  const uint32_t bar_q_full = sBar;
  const uint32_t bar_kv_full = sBar + 8;
  const uint32_t bar_kv_empty = bar_kv_full + 8 * C::kStages;
  const uint32_t bar_s_full = bar_kv_empty + 8 * C::kStages;
  const uint32_t bar_p_full = bar_s_full + 16;
  const uint32_t bar_o_full = bar_p_full + 16;
  const uint32_t bar_x = bar_o_full + 16;                // [4] one per row group: the two warps of a row swap a float
  const uint32_t s_tmem_ptr = bar_x + 32;
  const uint32_t sXch = s_tmem_ptr + 16;
  uint32_t* tmem_ptr_generic = reinterpret_cast<uint32_t*>(smem_raw + (s_tmem_ptr - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  // CG = 2: blockIdx.x = 2 * (pair item) + rank; 128-row tile t of the pair's slab belongs to CTA t & 1, slot t >> 1
  const int rank = CG == 2 ? int(cluster_ctarank()) : 0;
  const FwdItem item = p.items[(CG == 2 ? blockIdx.x >> 1 : blockIdx.x) + size_t(blockIdx.z) * p.item_batch_stride];
  if (item.q_rows == 0) return;  // padding of a per-sample schedule (the whole CTA / CTA pair: nothing is set up yet)
  const bool q_is_ref = (item.q_is_ref & 1) != 0;
  const int split = item.q_is_ref >> 8;  // 0: final output; s + 1: key split s of a short-query G slab
  const int h = blockIdx.y;
  const int b = blockIdx.z;
  const int n0 = (item.seg0_len + kTile - 1) / kTile;
  const int n1 = (item.seg1_len + kTile - 1) / kTile;
  const int n_kv = n0 + n1;
  // DUAL (a slab with one Q tile per CTA: the short-query regime, and the last slab of a frame or block): the second
  // slot of TMEM would idle and every key tile would wait for the S -> softmax -> P -> PV chain of the one before it.
  // Instead both slots work on the SAME Q tile: slot i takes the key tiles j = i (mod 2) with its own running
  // (m_ref, l, O), and the epilogue merges the two partial softmax states.  Two key tiles are then in flight, as with
  // two Q tiles.  (The same decision in both CTAs of a pair: it depends on the item only.)
  const bool dual = item.q_rows <= kTile * CG && n_kv >= 2;
  const int n_qt = (item.q_rows > kTile * CG || dual) ? 2 : 1;  // TMEM slots in use (the same in both CTAs of a pair)
  const int n_steps = dual ? (n_kv + 1) / 2 : n_kv;             // iterations of the (step, slot) loops
  auto slot_row = [&](int i) { return dual ? rank * kTile : (CG * i + rank) * kTile; };  // first slab row of this CTA's slot i

#ifdef SRA_FWD_TRACE
  const bool ftr_on = blockIdx.x == 4 && blockIdx.y == 0 && blockIdx.z == 0 && (threadIdx.x & 31) == 0;
#endif
  if (threadIdx.x == 0) {
    mbar_init(bar_q_full, 1);
    for (int s = 0; s < C::kStages; ++s) {
      mbar_init(bar_kv_full + 8 * s, 1);
      mbar_init(bar_kv_empty + 8 * s, 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_s_full + 8 * i, 1);
      mbar_init(bar_p_full + 8 * i, 8 * CG);  // one elected arrive per softmax warp (of both CTAs of a pair)
      mbar_init(bar_o_full + 8 * i, 1);
    }
    for (int g = 0; g < 4; ++g) mbar_init(bar_x + 8 * g, 2);  // one elected arrive per warp of the pair
    fence_mbar_init();
  }
  if (warp == 9 && lane == 0) {
    tma_prefetch_desc(q_is_ref ? &tm_q_ref : &tm_q_gen);
    tma_prefetch_desc(item.seg0_is_ref ? &tm_k_ref : &tm_k_gen);
    tma_prefetch_desc(item.seg0_is_ref ? &tm_v_ref : &tm_v_gen);
  }
  if (warp == 8) tmem_alloc<CG>(s_tmem_ptr, C::kTmemCols);
  tc_fence_before();
  if (CG == 2) cluster_sync(); else __syncthreads();  // (pair: the peer's mbarriers are initialised before anything signals them)
  tc_fence_after();
  // p_full lives in the leader CTA (its MMA thread waits for the P tiles of both CTAs)
  const uint32_t bar_p_full_leader = CG == 2 ? mapa_cluster(bar_p_full, 0) : bar_p_full;
  const uint32_t tmem = *tmem_ptr_generic;
  const uint32_t tS0 = tmem, tO0 = tmem + 256;

  if (warp < 8) {
    // ======================================================= softmax warps
    // Warps w and w + 4 sit on the same SM sub-partition and own the same 32 TMEM lanes (query rows);
    // warp w takes key columns [0, 64) of every score tile, warp w + 4 columns [64, 128), for BOTH Q
    // tiles in turn.  Two warps per sub-partition work on one tile at a time, so the hardware scheduler
    // interleaves their MUFU / FMA / ALU streams (one warp alone issues its exp2 back to back and leaves
    // the other pipes idle), and the softmax of a tile takes about half as long, which is what bounds the
    // S -> P -> PV -> QK dependency ring of that tile.
    reg_inc<224>();
    const int hh = warp >> 2;  // column half
    const int row_in_tile = (warp & 3) * 32 + lane;
    const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
    const float sl2 = p.scale_log2;
    // Online softmax with a *lagging* lazy rescale.  m_ref is the reference max the exponentials are
    // taken against; it is stale on purpose: P = exp2((s - m_ref) * sl2) is exact for any m_ref (bf16 and
    // fp32 keep their relative precision), so a tile never waits for its own row max before its first
    // exp2.  The tile max mt is reduced alongside the exponentials (FMNMX3 in the shadow of MUFU) and
    // only (a) moves m_ref at the start of a later tile once it leads by more than 2^8 (O and l are
    // rescaled then), (b) forces a second, exact pass over this tile when it leads by more than 2^64
    // (always on the first tile, where m_ref = -inf; otherwise only for adversarial score jumps).
    float m_ref[2] = {-INFINITY, -INFINITY};
    float m_seen[2] = {-INFINITY, -INFINITY};  // max raw score over the tiles processed so far
    float l[2] = {0.f, 0.f};                   // this thread's half of sum exp2((s - m_ref) * sl2)
    uint32_t slot = 0;                         // exchange-buffer parity, toggles at every swap
    // One float per (slot, half, row): the two threads of a row swap their half-row maxima (and, at the end, their
    // half-row sums) through shared memory.  The swap is split: post() publishes this thread's value and arrives on the
    // row group's mbarrier (64 arrivals) without blocking - it is called as soon as the half-row max is known, in the
    // middle of the tile's exponentials - and fetch() waits for the partner's arrival only when the value is needed,
    // at the end of the pass, by when the partner has normally long arrived.  (A blocking 64-thread barrier here
    // made the two warps of a row run in lock-step.)  Slots alternate; a slot is rewritten two swaps later, which the
    // partner cannot reach before this thread's next arrival, i.e. after this thread has read the slot.
    const uint32_t bx = bar_x + 8 * (warp & 3);
    uint32_t xphase = 0;
    auto post = [&](float mine) {
      st_shared_f32(sXch + ((slot * 2 + hh) * kTile + row_in_tile) * 4, mine);
      __syncwarp();
      if (lane == 0) mbar_arrive(bx);
    };
    auto fetch = [&]() -> float {
      mbar_wait(bx, xphase);
      const float other = ld_shared_f32(sXch + ((slot * 2 + (hh ^ 1)) * kTile + row_in_tile) * 4);
      slot ^= 1;
      xphase ^= 1;
      return other;
    };
    for (int t = 0; t < n_steps; ++t) {
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int j = dual ? 2 * t + i : t;  // key tile of slot i at this step
        if (i < n_qt && j < n_kv) {
          const int n_valid = (j < n0) ? min(kTile, item.seg0_len - j * kTile) : min(kTile, item.seg1_len - (j - n0) * kTile);
          const int n_valid_h = n_valid - 64 * hh;  // valid columns of this thread's 64-column half (may be <= 0)
          const uint32_t tS = tS0 + i * 128 + lane_off;
          const uint32_t tO = tO0 + i * D + lane_off + hh * (D / 2);
          auto rescale_to = [&](float m_new) {
            const float alpha = ex2((m_ref[i] - m_new) * sl2);
            m_ref[i] = m_new;
            l[i] *= alpha;
#pragma unroll
            for (int c = 0; c < D / 64; ++c) {  // this thread's half of the O_i row
              uint32_t o[32];
              tmem_ld32(tO + c * 32, o);
              tmem_wait_ld();
#pragma unroll
              for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
              tmem_st32(tO + c * 32, o);
            }
            tmem_wait_st();
          };
          if ((warp & 3) == 0) FTR(2 * hh + i, t, 0);
          mbar_wait(bar_s_full + 8 * i, t & 1);
          tc_fence_after();
          if ((warp & 3) == 0) FTR(2 * hh + i, t, 1);
#ifndef SRA_FWD_SKEL  // (ablation builds only: MMAs, TMA and barriers without the softmax arithmetic; results are wrong)
          // s_full completed => every earlier MMA, including this slot's previous O_i += P_i V, is complete.
          if (t > 0 && __any_sync(0xffffffffu, (m_seen[i] - m_ref[i]) * sl2 > 8.0f)) rescale_to(fmaxf(m_ref[i], m_seen[i]));
          uint32_t pk[2][16];
          float l_tile = 0.f, mt = -INFINITY;
#pragma unroll 1
          for (int pass = 0; pass < 2; ++pass) {
            // The half row streams through two 32-column register buffers: the tcgen05.ld of the second
            // chunk is in flight while the first is exponentiated.
            uint32_t s[2][32];
            const float neg_m = -m_ref[i] * sl2;
            const uint64_t sl2_2 = pack2(sl2, sl2), neg_m2 = pack2(neg_m, neg_m);
            uint64_t la = pack2(0.f, 0.f), lb = pack2(0.f, 0.f);
            float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
            float mt_h = -INFINITY;
            tmem_ld32(tS + hh * 64, s[0]);
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              tmem_wait_ld();
              if (c == 0) tmem_ld32(tS + hh * 64 + 32, s[1]);
              uint32_t(&sc)[32] = s[c];
              if (n_valid < kTile) {
#pragma unroll
                for (int k = 0; k < 32; ++k)
                  if (c * 32 + k >= n_valid_h) sc[k] = 0xff800000u;  // -inf
              }
#pragma unroll
              for (int k = 0; k < 16; ++k)
                mx[k & 3] = fmaxf(mx[k & 3], fmaxf(__uint_as_float(sc[2 * k]), __uint_as_float(sc[2 * k + 1])));
              if (c == 1) {  // half-row max known: publish it now, the exponentials of this chunk follow
                mt_h = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3]));
                post(mt_h);
              }
#pragma unroll
              for (int k = 0; k < 16; ++k) {
                const float s0 = __uint_as_float(sc[2 * k]), s1 = __uint_as_float(sc[2 * k + 1]);
                // x = s * scale * log2(e) - m_ref * scale * log2(e) for a pair of columns (one FFMA2)
                const uint64_t x = fma2(pack2(s0, s1), sl2_2, neg_m2);
                float p0, p1;
                if (((k * kEmuPairsPer8) & 7) < kEmuPairsPer8) {
                  ex2_emu2(x, p0, p1);  // FMA/ALU pipes
                } else {
                  float x0, x1;
                  unpack2(x, x0, x1);
                  p0 = ex2(x0);  // MUFU
                  p1 = ex2(x1);
                }
                if (k & 1) lb = add2(lb, pack2(p0, p1)); else la = add2(la, pack2(p0, p1));
                pk[c][k] = pack_bf16(p0, p1);
              }
            }
            float l0, l1, l2, l3;
            unpack2(la, l0, l1);
            unpack2(lb, l2, l3);
            l_tile = (l0 + l1) + (l2 + l3);
            if ((warp & 3) == 0) FTR(2 * hh + i, t, 2);
            // Full-row tile max = max of the two halves.
            mt = fmaxf(mt_h, fetch());
            if ((warp & 3) == 0) FTR(2 * hh + i, t, 3);
            // exact unless the tile leads m_ref by more than 2^64 (or m_ref is still -inf); the decision is
            // the same in both warps of a row (same mt, same m_ref)
            if (pass == 1 || !__any_sync(0xffffffffu, !((mt - m_ref[i]) * sl2 <= 64.0f))) break;
            const float m_new = fmaxf(m_ref[i], mt);
            if (t > 0) rescale_to(m_new); else m_ref[i] = m_new;
          }
          m_seen[i] = fmaxf(m_seen[i], mt);
          l[i] += l_tile;
          if (n_valid < kTile) {
            // the emulated exp2 returns ~2^-125 (not 0) for a masked column: force P = 0 exactly
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
              for (int k = 0; k < 16; ++k) {
                const int col = c * 32 + 2 * k;
                if (col >= n_valid_h) pk[c][k] = 0u;
                else if (col + 1 >= n_valid_h) pk[c][k] &= 0xffffu;
              }
          }
          // P_i: bf16 pairs; this half's 64 keys go over the first 32 columns of the 64 score columns this same warp
          // has read (columns [64 hh, 64 hh + 32) of the S_i region), so neither warp of a row ever overwrites
          // scores its partner may still be loading and no barrier is needed between the loads and this store.
#pragma unroll
          for (int c = 0; c < 2; ++c) tmem_st16(tS + hh * 64 + c * 16, pk[c]);
          tmem_wait_st();
#endif
          tc_fence_before();
          __syncwarp();
          if (lane == 0) {
            if (CG == 2) mbar_arrive_cluster(bar_p_full_leader + 8 * i); else mbar_arrive(bar_p_full + 8 * i);
          }
          if ((warp & 3) == 0) FTR(2 * hh + i, t, 4);
        }
      }
    }
    // ---------------------------------------------------- epilogue (a5): O / l -> bf16, LSE
    // (DUAL: one output tile from the two slots' partial states: O = a_0 O_0 + a_1 O_1, l = a_0 l_0 + a_1 l_1 with
    //  a_i = 2^((m_ref_i - m) sl2), m = max(m_ref_0, m_ref_1))
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      if (i < (dual ? 1 : n_qt)) {
        const uint32_t tO = tO0 + i * D + lane_off + hh * (D / 2);
        mbar_wait(bar_o_full + 8 * i, 0);
        if (dual) mbar_wait(bar_o_full + 8, 0);
        tc_fence_after();
        float a0 = 1.f, a1 = 0.f, m_out = m_ref[i];
        if (dual) {
          m_out = fmaxf(m_ref[0], m_ref[1]);
          a0 = ex2((m_ref[0] - m_out) * sl2);
          a1 = ex2((m_ref[1] - m_out) * sl2);
        }
        const float l_mine = dual ? l[0] * a0 + l[1] * a1 : l[i];
        post(l_mine);
        const float l_row = l_mine + fetch();
        const int row = slot_row(i) + row_in_tile;
        const bool valid = row < item.q_rows;
        const int n_tok = q_is_ref ? p.n_ref : p.n_gen;
        const int grow = item.q_row0 + row;
        __nv_bfloat16* obase = q_is_ref ? p.o_ref : p.o_gen;
        uint4* orow = reinterpret_cast<uint4*>(obase + ((size_t(b) * n_tok + grow) * p.heads + h) * D + hh * (D / 2));
        const float inv_l = 1.0f / l_row;
        const float w0 = a0 * inv_l, w1 = a1 * inv_l;
        // this thread's half row of O, 32 columns at a time, normalised (and merged)
        auto load_o = [&](int c, uint32_t (&o)[32]) {
          tmem_ld32(tO + c * 32, o);
          tmem_wait_ld();
          if (dual) {
            uint32_t o1[32];
            tmem_ld32(tO + D + c * 32, o1);
            tmem_wait_ld();
#pragma unroll
            for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * w0 + __uint_as_float(o1[k]) * w1);
          } else {
#pragma unroll
            for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * inv_l);
          }
        };
        if (split == 0) {
#pragma unroll
          for (int c = 0; c < D / 64; ++c) {
            uint32_t o[32];
            load_o(c, o);
            if (valid) {
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
          float* lse = q_is_ref ? p.lse_ref : p.lse_gen;
          if (lse != nullptr && valid && hh == 0) lse[(size_t(b) * p.heads + h) * n_tok + grow] = m_out * p.scale + __logf(l_row);
        } else {
          // key split: fp32 partial (O_s, LSE_s) of generation rows, head-major so the merge kernel streams it
          const size_t prow = ((size_t(split - 1) * p.batch + b) * p.heads + h) * p.n_gen + grow;
          float4* dst = reinterpret_cast<float4*>(p.part_o + prow * D + hh * (D / 2));
#pragma unroll
          for (int c = 0; c < D / 64; ++c) {
            uint32_t o[32];
            load_o(c, o);
            if (valid) {
#pragma unroll
              for (int q = 0; q < 8; ++q)
                dst[c * 8 + q] = make_float4(__uint_as_float(o[4 * q + 0]), __uint_as_float(o[4 * q + 1]),
                                             __uint_as_float(o[4 * q + 2]), __uint_as_float(o[4 * q + 3]));
            }
          }
          if (valid && hh == 0) p.part_lse[prow] = m_out * p.scale + __logf(l_row);
        }
        tc_fence_before();
      }
    }
  } else {
    reg_dec<56>();
    if (warp == 9 && elect_one()) {
      // ===================================================== TMA loader
      // Pair: every load of either CTA reports its bytes to the LEADER's barriers (the leader's MMA thread is the
      // only consumer); the leader alone arrives, expecting the bytes of both CTAs.
      const CUtensorMap* tq = q_is_ref ? &tm_q_ref : &tm_q_gen;
      const uint32_t q_full_l = CG == 2 ? mapa_cluster(bar_q_full, 0) : bar_q_full;
      const uint32_t kv_full_l = CG == 2 ? mapa_cluster(bar_kv_full, 0) : bar_kv_full;
      // Two copies of the loader, chosen once per CTA.  BND: an item whose query slab or key segments can end INSIDE a
      // tensor - a reference block (R items), a frame of a temporal window - loads its ragged tiles through the maps
      // bounded at those ends (sra_common.h BoundMaps): the rows behind an end read as zero, not as the neighbouring
      // block's or frame's (0 * Inf in the PV MMA; the softmax's warp-wide rescale votes would otherwise depend on a
      // neighbour's Q rows).  Every other item runs the plain loop, whose per-tile latency is measurable in the step time
      // (any run-time map selection in it costs 0.4-0.8 % at 720p).
      auto run_loader = [&](auto bnd_tag) {
        constexpr bool BND = decltype(bnd_tag)::value;
        const int mask = p.item_batch_stride ? b : 0;
        if (rank == 0) mbar_arrive_expect_tx(bar_q_full, n_qt * C::kTileBytes * CG);
        const CUtensorMap* tq_tail = tq;
        if (BND && slot_row(n_qt - 1) + kTile > item.q_rows) {
          const CUtensorMap* m = bound_lookup(p.bound, q_is_ref ? 5 : 4, q_is_ref, mask, item.q_row0 + item.q_rows);
          if (m != nullptr) tq_tail = m;
        }
        for (int i = 0; i < n_qt; ++i)
          load_tile<D, CG>(sQ + i * C::kTileBytes, (BND && slot_row(i) + kTile > item.q_rows) ? tq_tail : tq, q_full_l,
                           item.q_row0 + slot_row(i), h, b, false);
        int it = 0;
        for (int j = 0; j < n_kv; ++j) {
          const bool first = j < n0;
          const bool is_ref = first ? (item.seg0_is_ref != 0) : true;
          const int row = first ? item.seg0_start + j * kTile : item.seg1_start + (j - n0) * kTile;
          const bool hm = is_ref && p.ref_kv_head_major;
          // (the table is searched when the ragged tile comes up: the loader runs a ring ahead of the MMAs)
          const CUtensorMap* tk_tail = nullptr;
          if (BND && (first ? j == n0 - 1 : j == n_kv - 1)) {
            const int len = first ? item.seg0_len : item.seg1_len;
            if (len % kTile != 0) tk_tail = bound_lookup(p.bound, is_ref ? 2 : 0, is_ref, mask, (first ? item.seg0_start : item.seg1_start) + len);
          }
#pragma unroll
          for (int kv = 0; kv < 2; ++kv, ++it) {
            const int s = it % C::kStages;
            const uint32_t ph = (it / C::kStages) & 1;
            const CUtensorMap* tm = kv == 0 ? (is_ref ? &tm_k_ref : &tm_k_gen) : (is_ref ? &tm_v_ref : &tm_v_gen);
            if (BND && tk_tail != nullptr) tm = tk_tail + kv * p.bound.n_total;
            mbar_wait(bar_kv_empty + 8 * s, ph ^ 1);
            if (rank == 0) mbar_arrive_expect_tx(bar_kv_full + 8 * s, C::kTileBytes);
            const uint32_t dst = sKV + s * C::kStageBytes;
            if constexpr (CG == 1) {
              load_tile<D, 1>(dst, tm, kv_full_l + 8 * s, row, h, b, hm);
            } else {
              if (kv == 0) load_k_half<D>(dst, tm, kv_full_l + 8 * s, row, h, b, hm, rank);
              else load_v_half<D>(dst, tm, kv_full_l + 8 * s, row, h, b, hm, rank);
            }
          }
        }
      };
      if (p.bound.maps != nullptr && (q_is_ref || p.bound.n_gen_ends > 0)) run_loader(std::true_type{});
      else run_loader(std::false_type{});
    } else if (warp == 8 && rank == 0 && elect_one()) {
      // ===================================================== MMA issuer (pair: the leader CTA only, M = 256)
      constexpr uint32_t idesc_qk = make_idesc_bf16(kTile * CG, kTile, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc_bf16(kTile * CG, D, 0, 1);
      // Descriptor low words: Q/K tiles are K-major (LBO unused), V is MN-major (LBO = one 64-column box).
      constexpr uint32_t kDescHi = desc_hi_sw128(1024);
      constexpr uint32_t kQStep = C::kTileBytes >> 4, kStageStep = C::kStageBytes >> 4;
      const uint32_t q_lo = desc_lo(sQ, 16), k_lo = desc_lo(sKV, 16), v_lo = desc_lo(sKV, C::kBoxBytes);
      auto issue_qk = [&](int i, int stage) {
        const uint32_t q = q_lo + i * kQStep, k = k_lo + stage * kStageStep;
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t qoff = ((kk / 4) * C::kBoxBytes + (kk % 4) * 32) >> 4;
          const uint32_t koff = ((kk / 4) * C::kKBoxBytes + (kk % 4) * 32) >> 4;
          umma_ss<CG>(tS0 + i * 128, desc64(q + qoff, kDescHi), desc64(k + koff, kDescHi), idesc_qk, kk > 0);
        }
      };
      auto issue_pv = [&](int i, int stage, bool acc) {
        const uint32_t v = v_lo + stage * kStageStep;
#pragma unroll
        for (int kk = 0; kk < kTile / 16; ++kk)
          umma_ts<CG>(tO0 + i * D, tS0 + i * 128 + (kk / 4) * 64 + (kk % 4) * 8, desc64(v + kk * (2048 >> 4), kDescHi), idesc_pv,
                      (acc || kk > 0) ? 1u : 0u);
      };
      auto stage_of = [&](int it) { return it % C::kStages; };
      auto phase_of = [&](int it) { return uint32_t((it / C::kStages) & 1); };

      mbar_wait(bar_q_full, 0);
      if (dual) {
        // slot i = j & 1 takes key tile j (K_j at ring position 2 j, V_j at 2 j + 1); both Q slots hold the same tile
        for (int i = 0; i < 2; ++i) {
          mbar_wait(bar_kv_full + 8 * stage_of(2 * i), phase_of(2 * i));
          tc_fence_after();
          issue_qk(i, stage_of(2 * i));
          umma_commit<CG>(bar_s_full + 8 * i);
          umma_commit<CG>(bar_kv_empty + 8 * stage_of(2 * i));
        }
        for (int j = 0; j < n_kv; ++j) {
          const int i = j & 1, t = j >> 1, itv = 2 * j + 1, itk = 2 * (j + 2);
          mbar_wait(bar_kv_full + 8 * stage_of(itv), phase_of(itv));
          mbar_wait(bar_p_full + 8 * i, t & 1);
          tc_fence_after();
          issue_pv(i, stage_of(itv), t > 0);
          if (j + 2 >= n_kv) umma_commit<CG>(bar_o_full + 8 * i);
          umma_commit<CG>(bar_kv_empty + 8 * stage_of(itv));
          if (j + 2 < n_kv) {
            mbar_wait(bar_kv_full + 8 * stage_of(itk), phase_of(itk));
            tc_fence_after();
            issue_qk(i, stage_of(itk));
            umma_commit<CG>(bar_s_full + 8 * i);
            umma_commit<CG>(bar_kv_empty + 8 * stage_of(itk));
          }
        }
      } else {
      int it = 0;
      mbar_wait(bar_kv_full + 8 * stage_of(it), phase_of(it));
      tc_fence_after();
      for (int i = 0; i < n_qt; ++i) {
        issue_qk(i, stage_of(it));
        umma_commit<CG>(bar_s_full + 8 * i);
      }
      umma_commit<CG>(bar_kv_empty + 8 * stage_of(it));
      ++it;
      for (int j = 0; j < n_kv; ++j) {
        const int sv = stage_of(it);
        mbar_wait(bar_kv_full + 8 * sv, phase_of(it));
        ++it;
        const bool more = j + 1 < n_kv;
        const int sk = stage_of(it);
        for (int i = 0; i < n_qt; ++i) {
          FTR(4 + i, j, 0);
          if (CG == 2) mbar_wait_cluster(bar_p_full + 8 * i, j & 1); else mbar_wait(bar_p_full + 8 * i, j & 1);
          FTR(4 + i, j, 1);
          tc_fence_after();
          issue_pv(i, sv, j > 0);
          FTR(4 + i, j, 2);
          if (!more) umma_commit<CG>(bar_o_full + 8 * i);
          if (i == n_qt - 1) umma_commit<CG>(bar_kv_empty + 8 * sv);
          if (more) {
            if (i == 0) {
              mbar_wait(bar_kv_full + 8 * sk, phase_of(it));
              tc_fence_after();
            }
            issue_qk(i, sk);
            umma_commit<CG>(bar_s_full + 8 * i);
            FTR(4 + i, j, 3);
            if (i == n_qt - 1) umma_commit<CG>(bar_kv_empty + 8 * sk);
          }
        }
        if (more) ++it;
      }
      }
    }
  }
  // Pair: neither CTA may leave (or free its TMEM) while the other can still read its shared memory / TMEM or signal
  // its mbarriers.
  tc_fence_before();
  if (CG == 2) cluster_sync(); else __syncthreads();
  if (warp == 8) {
    tc_fence_after();
    tmem_dealloc<CG>(tmem, C::kTmemCols);
  }
}

// The dynamic shared-memory opt-in is a per-device function attribute: remembered per device ordinal.
bool* smem_configured_flag(int which) {
  static bool flags[8][64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) dev = 0;
  return &flags[which][dev];
}

template <int D, int CG>
cudaError_t launch_fwd(const CUtensorMap* maps, const FwdParams& p, cudaStream_t stream) {
  using C = FwdCfg<D, CG>;
  bool* configured = smem_configured_flag((D == 128 ? 0 : 1) + 2 * (CG - 1));
  if (!*configured) {
    cudaError_t e = cudaFuncSetAttribute(sra_fwd_kernel<D, CG>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes);
    if (e != cudaSuccess) return e;
    *configured = true;
  }
  // p.n_items counts launched items: 256-row slabs (CG = 1) or 512-row pair slabs, two CTAs each (CG = 2)
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(p.n_items * CG, p.heads, p.batch);
  cfg.blockDim = dim3(C::kThreads);
  cfg.dynamicSmemBytes = C::kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = CG == 2 ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, sra_fwd_kernel<D, CG>, maps[0], maps[1], maps[2], maps[3], maps[4], maps[5], p);
}

// a5' (short-query schedules only): O = sum_s exp(LSE_s - LSE) O_s with LSE = log sum_s exp(LSE_s); one warp per
// (batch, token, head) output row, fp32 partials in, bf16 O (RNE) and fp32 LSE out.  HBM-bound and tiny.
template <int D>
__global__ void sra_fwd_merge_kernel(const float* __restrict__ part_o, const float* __restrict__ part_lse,
                                     __nv_bfloat16* __restrict__ o_gen, float* __restrict__ lse_gen, int n_split, int B,
                                     int H, int n_gen, int row0, int n_rows) {
  const int lane = threadIdx.x & 31;
  const size_t warp_id = (blockIdx.x * size_t(blockDim.x) + threadIdx.x) >> 5;
  const size_t n_warps = (gridDim.x * size_t(blockDim.x)) >> 5;
  const size_t rows = size_t(B) * n_rows * H;  // generation rows [row0, row0 + n_rows) of every batch item and head
  const size_t split_stride = size_t(B) * H * n_gen;
  constexpr int V = D / 32;  // floats per lane
  for (size_t r = warp_id; r < rows; r += n_warps) {
    const int h = int(r % H);
    const size_t t = r / H;
    const int n = row0 + int(t % n_rows);
    const int b = int(t / n_rows);
    const size_t prow = (size_t(b) * H + h) * n_gen + n;
    float m = -INFINITY;
    for (int s = 0; s < n_split; ++s) m = fmaxf(m, part_lse[s * split_stride + prow]);
    float acc[V];
#pragma unroll
    for (int k = 0; k < V; ++k) acc[k] = 0.f;
    float wsum = 0.f;
    for (int s = 0; s < n_split; ++s) {
      const float w = __expf(part_lse[s * split_stride + prow] - m);
      wsum += w;
      const float* src = part_o + (s * split_stride + prow) * D + lane * V;
      if (V == 4) {
        const float4 x = *reinterpret_cast<const float4*>(src);
        acc[0] = fmaf(w, x.x, acc[0]); acc[1] = fmaf(w, x.y, acc[1]); acc[2] = fmaf(w, x.z, acc[2]); acc[3 % V] = fmaf(w, x.w, acc[3 % V]);
      } else {
        const float2 x = *reinterpret_cast<const float2*>(src);
        acc[0] = fmaf(w, x.x, acc[0]); acc[1] = fmaf(w, x.y, acc[1]);
      }
    }
    const float inv = 1.0f / wsum;
    __nv_bfloat16* dst = o_gen + ((size_t(b) * n_gen + n) * H + h) * D + lane * V;
    if (V == 4) {
      uint2 o;
      o.x = pack_bf16(acc[0] * inv, acc[1] * inv);
      o.y = pack_bf16(acc[2 % V] * inv, acc[3 % V] * inv);
      *reinterpret_cast<uint2*>(dst) = o;
    } else {
      *reinterpret_cast<uint32_t*>(dst) = pack_bf16(acc[0] * inv, acc[1] * inv);
    }
    if (lse_gen != nullptr && lane == 0) lse_gen[prow] = m + __logf(wsum);
  }
}

cudaError_t launch_fwd_merge(const FwdParams& p, int head_dim, int n_split, cudaStream_t stream, int n_ctas, int row0,
                             int n_rows) {
  if (n_rows < 0) { row0 = 0; n_rows = p.n_gen; }
  if (n_rows == 0) return cudaSuccess;
  const size_t rows = size_t(p.batch) * n_rows * p.heads;
  const int threads = 256;
  const int blocks = int(std::min<size_t>((rows * 32 + threads - 1) / threads, size_t(n_ctas)));
  if (head_dim == 128)
    sra_fwd_merge_kernel<128><<<blocks, threads, 0, stream>>>(p.part_o, p.part_lse, p.o_gen, p.lse_gen, n_split, p.batch, p.heads, p.n_gen, row0, n_rows);
  else
    sra_fwd_merge_kernel<64><<<blocks, threads, 0, stream>>>(p.part_o, p.part_lse, p.o_gen, p.lse_gen, n_split, p.batch, p.heads, p.n_gen, row0, n_rows);
  return cudaGetLastError();
}

#ifdef SRA_FWD_TRACE
extern "C" void sra_dbg_set_fwd_trace(long long* p) { cudaMemcpyToSymbol(g_fwd_trace, &p, sizeof(p)); }
#endif
template cudaError_t launch_fwd<64, 1>(const CUtensorMap*, const FwdParams&, cudaStream_t);
template cudaError_t launch_fwd<128, 1>(const CUtensorMap*, const FwdParams&, cudaStream_t);
template cudaError_t launch_fwd<128, 2>(const CUtensorMap*, const FwdParams&, cudaStream_t);

}  // namespace sra
