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
  // Sparse temporal attention (sra_set_temporal_window): generation frame offsets and window (frames on
  // each side); window < 0 = off (every generation row sees every generation key)
  std::vector<int32_t> gen_frames;
  int window = -1;
  // Reference validity (sra_set_reference_validity[_batched]): kernels, schedule, cache and workspaces
  // see the COMPACTED reference (valid tokens only, blocks shrunk, empty blocks dropped).  n_masks = 1: one compaction
  // shared by the batch; n_masks = batch: one per batch item (reading A12).  Compacted tensors have `nr` rows per
  // batch item (nr = max over the masks; rows [nr_b[m], nr) of item m are zero padding, never scheduled).
  bool has_valid = false;
  int n_masks = 1;
  std::vector<int> nr_b;                       // [n_masks] valid reference tokens
  std::vector<std::vector<int32_t>> offe_b;    // [n_masks] effective block offsets
  int nr = 0;                                  // rows of the compacted reference tensors (= n_ref without a mask)
  std::vector<int32_t> h_gidx;                 // [B][nr]: compact row -> reference token, -1 = padding
  std::vector<int32_t> h_cidx;                 // [B][n_ref]: reference token -> compact row, -1 = invalid
  int32_t* d_gidx = nullptr;                   // capacity B * n_ref
  int32_t* d_cidx = nullptr;                   // B * n_ref
  bool idx_dirty = false;                      // host index arrays changed: uploaded by the next launch, on its stream
  void* cbuf[9] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // compact q,k,v,o,do,dq,dk,dv (bf16) + lse (fp32), capacity n_ref rows
  float scale = 0.f;
  int device = -1;       // -1: host-only context (no usable CUDA device)
  bool sm100 = false;
  int num_sms = 148;     // multiProcessorCount of the ctx's device (148 for a host-only ctx: the B200's)
  // ---- schedules (host).  Mask 0's lists (the only ones when n_masks == 1) are what the schedule queries return.
  std::vector<sra::FwdItem> fwd_items;  // G items first, then R items
  int n_gen_items = 0, n_ref_items = 0;
  std::vector<sra::BwdItem> bwd_items;
  // CTA-pair launch list (head_dim 128, no key split): consecutive slabs that see the same keys are merged into
  // 512-row pair items (a slab without such a neighbour stays alone, q_rows <= 256); G pairs first, then R pairs.
  // pair_of_item[i] = pair holding fwd_items[i]; pair_of_item[n_items] = n_pairs.
  std::vector<sra::FwdItem> pair_items;
  std::vector<int32_t> pair_of_item;
  int n_gen_pairs = 0, n_ref_pairs = 0;
  bool use_pairs = false;
  // Short-query regime (few G slabs): every G slab is cut into n_split key ranges so that all SMs stream the
  // K/V cache; split_items = the n_gen_items * n_split split slabs followed by the R items.
  int n_split = 1;
  std::vector<sra::FwdItem> split_items;
  // What the kernels read: the lists of every mask stacked [n_masks][stride], shorter lists padded with empty items
  // (q_rows = 0 / k_rows = 0: the CTA returns at once).  With n_masks == 1 the stride is irrelevant (batch stride 0).
  std::vector<sra::FwdItem> st_fwd, st_pair;
  std::vector<sra::BwdItem> st_bwd;
  int fwd_stride = 0, pair_stride = 0, bwd_stride = 0;   // items per mask in the stacks (max over the masks)
  int max_ref_items = 0, max_ref_pairs = 0;              // max over the masks (G counts are the same for every mask)
  // Device copies, double-buffered: sra_set_temporal_window / sra_set_reference_validity only rebuild the host lists
  // and flip `sched_buf`; the next launch uploads them on ITS stream into the other buffer, so a kernel still in
  // flight keeps reading the list it was launched with and no call synchronises the device.
  bool sched_dirty = true;
  int sched_buf = 0;
  sra::FwdItem* d_fwd_items[2] = {nullptr, nullptr};
  sra::FwdItem* d_pair_items[2] = {nullptr, nullptr};
  sra::FwdItem* d_split_items[2] = {nullptr, nullptr};
  sra::BwdItem* d_bwd_items[2] = {nullptr, nullptr};
  size_t cap_fwd = 0, cap_pair = 0, cap_split = 0, cap_bwd = 0;  // capacities (items) of each buffer of the pair
  float* ws_part_o = nullptr;
  float* ws_part_lse = nullptr;
  size_t cap_part_rows = 0;
  __nv_bfloat16* cache_k = nullptr;  // [B, H, n_ref, d] capacity; the tensor maps see [B, H, nr, d]
  __nv_bfloat16* cache_v = nullptr;
  bool cache_valid = false;
  // backward workspace (sra_reserve(SRA_RESERVE_BACKWARD) or first sra_backward), sized for the unmasked reference
  float* ws_dq = nullptr;     // fp32 [B*H, n_pad, d] dQ accumulators
  float* ws_delta = nullptr;  // fp32 [B*H, n_pad]   D_i
  float* ws_lse2 = nullptr;   // fp32 [B*H, n_pad]   LSE_i * log2(e)
  // host-buffer staging of sra_forward_host (sra_reserve(SRA_RESERVE_HOST) or first sra_forward_host):
  // q,k,v,o gen; q,o ref; lse gen/ref
  void* stage[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  // sra_forward_host pipeline: copy streams and events; sub-range override of the forward launch
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  std::vector<cudaEvent_t> pipe_ev;
  double h2d_gbs = 50.0;          // measured when the staging is reserved (pinned -> device); sizes the reference-first phase
  double fwd_flops_per_s = 1e15;  // measured from the previous pipelined call's middle launch
  cudaEvent_t rate_ev[2] = {nullptr, nullptr};
  bool rate_pending = false;
  double rate_flops = 0.0;
  int seg_buf = 0;
  int sub_first = 0, sub_count = -1;  // forward_core launches items [sub_first, sub_first + sub_count) when sub_count >= 0
  // "reference keys first" (sra_forward_host): every G slab once against the reference segment only (A items,
  // needs nothing but Q and the resident cache) and once against the generation segment only (B items), as fp32
  // partials merged per slab range; sub_seg makes forward_core launch from the segment list (no merge).
  sra::FwdItem* d_seg_items[2] = {nullptr, nullptr};  // [2 * n_gen_items] (with use_pairs: [2 * n_gen_pairs] pair items): A items, then B items
  size_t cap_seg = 0;
  bool seg_dirty = true;
  int seg_kc = 1;                       // generation-key chunks of the B items in the device list ([A ; B_0 ; ... ; B_kc-1])
  float* ws_seg_o = nullptr;            // fp32 [3][B][H][n_gen][d]  (A, B_0, B_1)
  float* ws_seg_lse = nullptr;          // fp32 [3][B][H][n_gen]
  bool sub_seg = false;
  // encoded tensor maps, keyed by what they describe (cuTensorMapEncodeTiled is ~1 us of host time each)
  struct TmapEntry {
    const void* ptr; int B, N, H, d, box_rows; bool head_major; CUtensorMap map;
  };
  std::vector<TmapEntry> tmaps;
  size_t tmap_next = 0;
  // Bounded tensor maps (sra_common.h BoundMaps): the segment ends that fall inside a tensor - frame ends of a
  // temporal window, block ends of the (compacted) reference per mask - and, per kernel family, the device copies of
  // the ends and of the maps encoded for the pointers of the last call (re-encoded only when a pointer or the
  // schedule changes; double-buffered like the schedule).
  std::vector<int32_t> bound_ends;  // [n_gen_ends | n_masks x ref_end_stride]
  int n_gen_ends = 0, ref_end_stride = 0;
  uint64_t bound_version = 0;
  struct BoundRole {
    const void* ptr; int N; bool is_ref, head_major; int box_rows;
    bool operator==(const BoundRole& o) const { return ptr == o.ptr && N == o.N && is_ref == o.is_ref && head_major == o.head_major && box_rows == o.box_rows; }
  };
  struct BoundSet {
    CUtensorMap* d_maps[2] = {nullptr, nullptr};
    int32_t* d_ends[2] = {nullptr, nullptr};
    size_t cap_maps = 0, cap_ends = 0;
    int buf = 0;
    uint64_t version = ~uint64_t(0);  // bound_version the device copy was built for
    std::vector<BoundRole> roles;     // ... and the tensors
    std::vector<CUtensorMap> h_maps;
  } bnd_fwd, bnd_bwd;
  uint32_t reserved = 0;  // SRA_RESERVE_* already done
  int64_t launches = 0;
  // optional per-kernel timing (sra_set_kernel_timing)
  bool timing = false;
  cudaEvent_t ev[SRA_NUM_KERNELS][2] = {};
  bool ev_recorded[SRA_NUM_KERNELS] = {};
  std::string err;

  int mask_of(int b) const { return n_masks == 1 ? 0 : b; }
};

namespace sra {
// Makes the ctx's device current for the duration of an entry point and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  bool changed = false;
  explicit DeviceGuard(int dev) {
    if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (changed) cudaSetDevice(prev);
  }
};
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
int sync_schedule(sra_ctx* ctx, cudaStream_t stream);  // uploads a changed schedule / index arrays on `stream`
// Device table of bounded maps for the given role tensors (encoded and uploaded on `stream` only when they differ
// from the last call's); out->maps = null when no segment ends inside a tensor.
int bound_maps(sra_ctx* ctx, sra_ctx::BoundSet& bs, const sra_ctx::BoundRole* roles, int n_roles, cudaStream_t stream,
               BoundMaps* out);
int reserve(sra_ctx* ctx, uint32_t what);
int grid_for(const sra_ctx* ctx, size_t total, int threads = 256, int ctas_per_sm = 16);
template <int D>
cudaError_t launch_bwd(const CUtensorMap* maps, const BwdParams& p, cudaStream_t stream);
template <int D, int CG>
cudaError_t launch_fwd(const CUtensorMap* maps, const FwdParams& p, cudaStream_t stream);
cudaError_t launch_fwd_merge(const FwdParams& p, int head_dim, int n_split, cudaStream_t stream, int n_ctas, int row0 = 0,
                             int n_rows = -1);  // n_rows < 0: every generation row
bool* smem_configured_flag(int which);  // per-device "dynamic shared memory opt-in done" flags (which < 8)
int run_backward(sra_ctx* ctx, const sra_bwd_args* a, cudaStream_t stream);
// compaction helpers of the validity path (sra_api.cu)
int compact_rows(sra_ctx* ctx, int slot, const void* src, const void** out, cudaStream_t stream);
int compact_lse(sra_ctx* ctx, const float* src, const float** out, cudaStream_t stream);
int compact_out(sra_ctx* ctx, int slot, void** out);
int expand_rows(sra_ctx* ctx, int slot, void* dst, cudaStream_t stream);
int expand_lse(sra_ctx* ctx, float* dst, cudaStream_t stream);
}  // namespace sra
