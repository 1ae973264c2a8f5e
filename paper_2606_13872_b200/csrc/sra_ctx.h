// Private definition of sra_ctx (shared by the API and the backward driver).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/sra.h"
#include "sra_common.h"

struct sra_ctx {
  sra_config cfg{};
  std::vector<int32_t> off;  // n_ref_blocks + 1
  // Reference validity (sra_set_reference_validity): kernels, schedule, cache and workspaces see the
  // COMPACTED reference (valid tokens only, blocks shrunk, empty blocks dropped); nr / offe equal n_ref / off
  // when every token is valid.
  // Sparse temporal attention (sra_set_temporal_window): generation frame offsets and window (frames on
  // each side); window < 0 = off (every generation row sees every generation key)
  std::vector<int32_t> gen_frames;
  int window = -1;
  int nr = 0;                  // effective reference tokens
  std::vector<int32_t> offe;   // effective block offsets
  bool has_valid = false;
  std::vector<int32_t> h_gidx; // compact index -> reference token
  int32_t* d_gidx = nullptr;   // [nr]
  int32_t* d_cidx = nullptr;   // [n_ref]: reference token -> compact index, -1 = invalid
  void* cbuf[9] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // compact q,k,v,o,do,dq,dk,dv (bf16) + lse (fp32)
  float scale = 0.f;
  int device = -1;       // -1: host-only context (no usable CUDA device)
  bool sm100 = false;
  std::vector<sra::FwdItem> fwd_items;  // G items first, then R items
  int n_gen_items = 0, n_ref_items = 0;
  std::vector<sra::BwdItem> bwd_items;
  sra::FwdItem* d_fwd_items = nullptr;
  // CTA-pair launch list (head_dim 128, no key split): consecutive slabs that see the same keys are merged into
  // 512-row pair items (a slab without such a neighbour stays alone, q_rows <= 256); G pairs first, then R pairs.
  // pair_of_item[i] = pair holding fwd_items[i]; pair_of_item[n_items] = n_pairs.
  std::vector<sra::FwdItem> pair_items;
  std::vector<int32_t> pair_of_item;
  int n_gen_pairs = 0, n_ref_pairs = 0;
  sra::FwdItem* d_pair_items = nullptr;
  bool use_pairs = false;
  // Short-query regime (few G slabs): every G slab is cut into n_split key ranges so that all SMs stream the
  // K/V cache; split_items = the n_gen_items * n_split split slabs followed by the R items.
  int n_split = 1;
  std::vector<sra::FwdItem> split_items;
  sra::FwdItem* d_split_items = nullptr;
  float* ws_part_o = nullptr;
  float* ws_part_lse = nullptr;
  sra::BwdItem* d_bwd_items = nullptr;
  __nv_bfloat16* cache_k = nullptr;  // [B, H, n_ref, d]
  __nv_bfloat16* cache_v = nullptr;
  bool cache_valid = false;
  // backward workspace (lazy)
  float* ws_dq = nullptr;     // fp32 [B*H, n_pad, d] dQ accumulators
  float* ws_delta = nullptr;  // fp32 [B*H, n_pad]   D_i
  float* ws_lse2 = nullptr;   // fp32 [B*H, n_pad]   LSE_i * log2(e)
  size_t ws_dq_bytes = 0;
  // host-buffer staging of sra_forward_host (lazy): q,k,v,o gen; q,o ref; lse gen/ref
  void* stage[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  // sra_forward_host pipeline (lazy): copy streams and events; sub-range override of the forward launch
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  std::vector<cudaEvent_t> pipe_ev;
  int sub_first = 0, sub_count = -1;  // forward_core launches items [sub_first, sub_first + sub_count) when sub_count >= 0
  // "reference keys first" (sra_forward_host): every G slab once against the reference segment only (A items,
  // needs nothing but Q and the resident cache) and once against the generation segment only (B items), as fp32
  // partials merged per slab range; sub_items != nullptr makes forward_core launch from it (no merge).
  sra::FwdItem* d_seg_items = nullptr;  // [2 * n_gen_items]: A items, then B items (with use_pairs: [2 * n_gen_pairs] pair items)
  float* ws_seg_o = nullptr;            // fp32 [2][B][H][n_gen][d]
  float* ws_seg_lse = nullptr;          // fp32 [2][B][H][n_gen]
  const sra::FwdItem* sub_items = nullptr;
  int64_t launches = 0;
  // optional per-kernel timing (sra_set_kernel_timing)
  bool timing = false;
  cudaEvent_t ev[SRA_NUM_KERNELS][2] = {};
  bool ev_recorded[SRA_NUM_KERNELS] = {};
  std::string err;
};

namespace sra {
// Brackets one kernel launch with CUDA events on its stream when ctx->timing is on.
struct KernelTimer {
  sra_ctx* ctx;
  int id;
  cudaStream_t stream;
  KernelTimer(sra_ctx* c, int which, cudaStream_t s) : ctx(c), id(which), stream(s) {
    if (ctx->timing) cudaEventRecord(ctx->ev[id][0], stream);
  }
  ~KernelTimer() {
    if (ctx->timing) {
      cudaEventRecord(ctx->ev[id][1], stream);
      ctx->ev_recorded[id] = true;
    }
  }
};
int ctx_fail(sra_ctx* ctx, int code, const std::string& msg);
int ctx_fail_cuda(sra_ctx* ctx, cudaError_t e, const char* what);
int make_tmap_bf16(sra_ctx* ctx, CUtensorMap* out, const void* ptr, int B, int N, int H, int d, bool head_major,
                   int box_rows);
template <int D>
cudaError_t launch_bwd(const CUtensorMap* maps, const BwdParams& p, cudaStream_t stream);
template <int D, int CG>
cudaError_t launch_fwd(const CUtensorMap* maps, const FwdParams& p, cudaStream_t stream);
cudaError_t launch_fwd_merge(const FwdParams& p, int head_dim, int n_split, cudaStream_t stream, int row0 = 0,
                             int n_rows = -1);  // n_rows < 0: every generation row
int run_backward(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream);
// compaction helpers of the validity path (sra_api.cu)
int compact_rows(sra_ctx* ctx, int slot, const void* src, const void** out, cudaStream_t stream);
int compact_lse(sra_ctx* ctx, const float* src, const float** out, cudaStream_t stream);
int compact_out(sra_ctx* ctx, int slot, void** out);
int expand_rows(sra_ctx* ctx, int slot, void* dst, cudaStream_t stream);
int expand_lse(sra_ctx* ctx, float* dst, cudaStream_t stream);
}  // namespace sra
