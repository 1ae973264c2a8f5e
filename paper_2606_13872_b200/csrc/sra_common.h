// Shared host/device definitions of the SRA CUDA path (work items, kernel parameters).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace sra {

constexpr int kTile = 128;         // rows per MMA tile (UMMA M = 128; key tile N = 128)
constexpr int kQRowsPerCta = 256;  // two ping-ponged Q tiles per CTA (forward)

// Forward work item: a 256-row query slab and the (up to two) key
// segments it may see.  G slab: seg0 = all generation keys, seg1 = all reference keys.
// R slab of block j: seg0 = reference keys [off[j], off[j+1]), seg1 empty.
struct FwdItem {
  int32_t q_is_ref;     // bit 0: 0 = rows of Q_g / O_g, 1 = rows of Q_r / O_r;  bits 8..: 0 = the item sees all of
                        // its keys and writes O / LSE; s + 1 = key split s of a short-query G slab, writes the
                        // fp32 partial (O_s, LSE_s) that sra_fwd_merge_kernel combines
  int32_t q_row0;       // first row (token index inside its tensor)
  int32_t q_rows;       // valid rows in this slab, 1..256
  int32_t seg0_is_ref;  // which K/V tensors seg0 reads
  int32_t seg0_start, seg0_len;
  int32_t seg1_start, seg1_len;  // always reference K/V; len 0 = absent
};

// Backward work item: a 128-key tile and the (up to two) query segments that see it.
// G key tile: generation queries [g_start, g_start + g_len) (all of them, or - with a temporal window - the frames
// whose window holds the tile's frame).  R key tile of block j: all generation queries, plus seg1 = reference
// queries [off[j], off[j+1]).
struct BwdItem {
  int32_t k_is_ref;
  int32_t k_row0;
  int32_t k_rows;  // valid keys 1..128
  int32_t seg1_start, seg1_len;  // reference-query segment (len 0 = absent)
  int32_t g_start, g_len;        // generation-query segment that sees this tile (all of G unless a temporal window is set)
  int32_t pad[1];
};

// Bounded tensor maps (mask isolation also for non-finite data).  The last tile of a key or query segment that ends
// INSIDE its tensor (a reference block, a frame of a temporal window) is loaded through a copy of the tensor map whose
// row dimension ends at the segment end: TMA then zero-fills the rows behind it instead of fetching the neighbouring
// block's or frame's, so a masked P = 0 never meets a neighbour's Inf / NaN in an MMA (0 * Inf = NaN).
struct BoundMaps {
  const CUtensorMap* maps;  // global memory, [roles][n_total]; null = no segment ends inside a tensor
  const int32_t* ends;      // [n_gen_ends | n_masks x ref_stride] end rows, each list ascending (padding INT32_MAX)
  int32_t n_gen_ends, ref_stride, n_total;
};
#ifdef __CUDACC__
// Index of the map bounded at `end_row` (generation list, or reference list of mask `mask`), -1 = none (the end is the
// tensor's own: the ordinary map already zero-fills there).
__device__ __forceinline__ int bound_index(const BoundMaps& bm, bool is_ref, int mask, int end_row) {
  if (bm.maps == nullptr) return -1;
  const int base = is_ref ? bm.n_gen_ends + mask * bm.ref_stride : 0;
  const int n = is_ref ? bm.ref_stride : bm.n_gen_ends;
  int lo = 0, hi = n;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (bm.ends[base + mid] < end_row) lo = mid + 1; else hi = mid;
  }
  return (lo < n && bm.ends[base + lo] == end_row) ? base + lo : -1;
}
#endif

struct FwdParams {
  const FwdItem* items;
  int32_t n_items;
  int32_t item_batch_stride;  // 0: one list for every batch item; else batch item b reads items + b * stride (per-sample
                              // validity masks: lists padded to a common length with empty items, q_rows = 0)
  int32_t heads, batch;
  int32_t n_gen, n_ref;
  float scale_log2;  // softmax_scale * log2(e)
  float scale;       // softmax_scale
  __nv_bfloat16* o_gen;
  __nv_bfloat16* o_ref;
  float* lse_gen;  // may be null
  float* lse_ref;  // may be null
  // coordinate order of the K/V reference tensor maps: 1 = head-major cache [B,H,N,d] => (c, n, h, b)
  int32_t ref_kv_head_major;
  // key-split partials of short-query G slabs (null when the schedule has no splits)
  float* part_o;    // fp32 [n_split][B][H][n_gen][d]: O_s = P_s V_s / l_s
  float* part_lse;  // fp32 [n_split][B][H][n_gen]:    LSE_s (natural log of the scaled scores)
  BoundMaps bound;  // roles: 0 K_g, 1 V_g, 2 K_r, 3 V_r, 4 Q_g, 5 Q_r
};

constexpr int kBwdQTile = 128;  // query rows per backward iteration (keys per CTA = kTile)

struct BwdParams {
  const BwdItem* items;
  int32_t n_items;
  int32_t item_batch_stride;  // as in FwdParams (empty item: k_rows = 0)
  int32_t heads, batch;
  int32_t n_gen, n_ref;
  int32_t n_pad;       // row length of the [G ; R]-concatenated fp32 workspaces (multiple of 64)
  float scale_log2;    // softmax_scale * log2(e)
  float scale;         // softmax_scale
  const float* lse2;   // ws [B*H][n_pad]: LSE * log2(e)           (written by the preprocess kernel)
  const float* delta;  // ws [B*H][n_pad]: D_i = sum_c dO_ic O_ic  (written by the preprocess kernel)
  float* dq_ws;        // ws [B*H][n_pad][d] fp32 dQ accumulators (zeroed before the launch)
  __nv_bfloat16* dk_gen;
  __nv_bfloat16* dv_gen;
  __nv_bfloat16* dk_ref;
  __nv_bfloat16* dv_ref;
  int32_t ref_kv_head_major;
  BoundMaps bound;  // roles: 0 Q_g, 1 dO_g, 2 K_g, 3 V_g, 4 Q_r, 5 dO_r, 6 K_r, 7 V_r
};

}  // namespace sra
