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
};

}  // namespace sra
