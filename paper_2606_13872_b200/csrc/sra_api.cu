// C-ABI implementation of include/sra.h: context, tile schedule (host), TMA tensor maps,
// reference-KV cache build and kernel launches.  No CPU compute path exists here.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "sra_ctx.h"

using sra::BwdItem;
using sra::FwdItem;
using sra::kQRowsPerCta;
using sra::kTile;


namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<EncodeTiledFn>(p);
  return fn;
}

// NVTX range around an entry point (visible in Nsight timelines; header-only NVTX3, a no-op without a tool)
struct nvtx_range {
  explicit nvtx_range(const char* name) { nvtxRangePushA(name); }
  ~nvtx_range() { nvtxRangePop(); }
};

int fail(sra_ctx* ctx, int code, const std::string& msg) { return sra::ctx_fail(ctx, code, msg); }
int fail_cuda(sra_ctx* ctx, cudaError_t e, const char* what) { return sra::ctx_fail_cuda(ctx, e, what); }

}  // namespace

namespace sra {

int ctx_fail(sra_ctx* ctx, int code, const std::string& msg) {
  if (ctx) ctx->err = msg;
  return code;
}
int ctx_fail_cuda(sra_ctx* ctx, cudaError_t e, const char* what) {
  return ctx_fail(ctx, SRA_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// bf16 tensor map over a [B, N, H, d] (token-major) or [B, H, N, d] (head-major) tensor; box = box_rows x 64
// columns, 128-byte swizzle, OOB rows read as zero.  Token-major coordinates: (c, h, n, b); head-major: (c, n, h, b).
// Encoded maps are kept in the ctx, keyed by everything they describe: a steady-state step re-encodes nothing.
// (rows_bound < N: the same tensor, but rows [rows_bound, N) read as zero - sra_common.h BoundMaps)
static int encode_tmap_bf16(sra_ctx* ctx, CUtensorMap* out, const void* ptr, int B, int N, int H, int d, bool head_major,
                            int box_rows, int rows_bound) {
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return fail(ctx, SRA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t dims[4], strides[3];
  cuuint32_t box[4], estr[4] = {1, 1, 1, 1};
  const cuuint64_t row = cuuint64_t(d) * 2;
  if (head_major) {
    dims[0] = d; dims[1] = rows_bound; dims[2] = H; dims[3] = B;
    strides[0] = row; strides[1] = row * N; strides[2] = row * N * H;
    box[0] = 64; box[1] = box_rows; box[2] = 1; box[3] = 1;
  } else {
    dims[0] = d; dims[1] = H; dims[2] = rows_bound; dims[3] = B;
    strides[0] = row; strides[1] = row * H; strides[2] = row * H * N;
    box[0] = 64; box[1] = 1; box[2] = box_rows; box[3] = 1;
  }
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(ptr), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(ctx, SRA_ERR_CUDA, "cuTensorMapEncodeTiled failed: " + std::to_string(int(r)));
  return SRA_OK;
}

int make_tmap_bf16(sra_ctx* ctx, CUtensorMap* out, const void* ptr, int B, int N, int H, int d, bool head_major,
                   int box_rows) {
  if (ctx) {
    for (const sra_ctx::TmapEntry& e : ctx->tmaps)
      if (e.ptr == ptr && e.N == N && e.box_rows == box_rows && e.head_major == head_major && e.B == B && e.H == H && e.d == d) {
        *out = e.map;
        return SRA_OK;
      }
  }
  if (int rc = encode_tmap_bf16(ctx, out, ptr, B, N, H, d, head_major, box_rows, N)) return rc;
  if (ctx) {
    constexpr size_t kMaxCached = 48;
    sra_ctx::TmapEntry e{ptr, B, N, H, d, box_rows, head_major, *out};
    if (ctx->tmaps.size() < kMaxCached) ctx->tmaps.push_back(e);
    else { ctx->tmaps[ctx->tmap_next] = e; ctx->tmap_next = (ctx->tmap_next + 1) % kMaxCached; }
  }
  return SRA_OK;
}

// [B, N, H, d] -> [B, H, N, d], 16 bytes per thread (a1: pure HBM copy, 2 * bytes of traffic).
__global__ void relayout_head_major_kernel(const uint4* __restrict__ src0, const uint4* __restrict__ src1,
                                           uint4* __restrict__ dst0, uint4* __restrict__ dst1, int N, int H, int vec,
                                           size_t total, const int32_t* __restrict__ gidx, int n_src) {
  // gidx != null: only the valid reference tokens are cached (row n of batch item b = source token gidx[b][n];
  // -1 = padding behind the item's last valid token: zeros, so that a masked tile tail never multiplies 0 by garbage)
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int c = int(i % vec);
    size_t t = i / vec;
    const int hh = int(t % H);
    t /= H;
    const int n = int(t % N);
    const size_t bb = t / N;
    const size_t o = ((bb * H + hh) * size_t(N) + n) * vec + c;
    const int tok = gidx ? gidx[bb * N + n] : n;
    const size_t in = gidx ? ((bb * n_src + tok) * H + hh) * size_t(vec) + c : i;
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    dst0[o] = tok >= 0 ? src0[in] : z;
    dst1[o] = tok >= 0 ? src1[in] : z;
  }
}

// RoPE (reading A18): 8 bf16 = 4 interleaved pairs, each multiplied as a complex number by
// (cos, sin)[4 pairs] in fp32 and rounded back to bf16.
__device__ __forceinline__ uint32_t rope_pair(uint32_t w, float c, float s) {
  const float a = __uint_as_float(w << 16), b = __uint_as_float(w & 0xffff0000u);
  const __nv_bfloat162 r = __floats2bfloat162_rn(fmaf(a, c, -b * s), fmaf(a, s, b * c));
  return *reinterpret_cast<const uint32_t*>(&r);
}
__device__ __forceinline__ uint4 rope_vec(uint4 x, float4 c, float4 s) {
  return make_uint4(rope_pair(x.x, c.x, s.x), rope_pair(x.y, c.y, s.y), rope_pair(x.z, c.z, s.z), rope_pair(x.w, c.w, s.w));
}

// The fused cache producer: relayout_head_major_kernel with the rotation of K folded into the copy
// (K: read pre-RoPE [B, N, H, d], write rotated [B, H, N, d]; V: plain relayout).  cos/sin rows are indexed by the
// ORIGINAL token (gidx[n] under a validity mask).  Traffic = 2 * bytes(K, V) + the table once per head from L2.
__global__ void relayout_rope_head_major_kernel(const uint4* __restrict__ src0, const uint4* __restrict__ src1,
                                                uint4* __restrict__ dst0, uint4* __restrict__ dst1, int N, int H, int vec,
                                                size_t total, const int32_t* __restrict__ gidx, int n_src,
                                                const float4* __restrict__ cs, const float4* __restrict__ sn) {
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int c = int(i % vec);
    size_t t = i / vec;
    const int hh = int(t % H);
    t /= H;
    const int n = int(t % N);
    const size_t bb = t / N;
    const int tok = gidx ? gidx[bb * N + n] : n;
    const size_t o = ((bb * H + hh) * size_t(N) + n) * vec + c;
    if (tok < 0) {  // padding row of a per-sample compaction
      dst0[o] = make_uint4(0u, 0u, 0u, 0u);
      dst1[o] = make_uint4(0u, 0u, 0u, 0u);
      continue;
    }
    const size_t in = gidx ? ((bb * n_src + tok) * H + hh) * size_t(vec) + c : i;
    const size_t tb = size_t(tok) * vec + c;  // float4 index: row tok of [n_src, d/2], pairs [4c, 4c + 4)
    dst0[o] = rope_vec(src0[in], __ldg(cs + tb), __ldg(sn + tb));
    dst1[o] = src1[in];
  }
}

// In-place rotation of one or two [B, N, H, d] tensors (the per-step Q_g / K_g side).
__global__ void rope_inplace_kernel(uint4* __restrict__ x0, uint4* __restrict__ x1, int N, int H, int vec, size_t total,
                                    const float4* __restrict__ cs, const float4* __restrict__ sn) {
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int c = int(i % vec);
    const int tok = int((i / (size_t(vec) * H)) % N);
    const size_t tb = size_t(tok) * vec + c;
    const float4 cc = __ldg(cs + tb), ss = __ldg(sn + tb);
    x0[i] = rope_vec(x0[i], cc, ss);
    if (x1) x1[i] = rope_vec(x1[i], cc, ss);
  }
}

// Validity path.  dst[b, i, :, :] = src[b, gidx[b][i], :, :], zeros where gidx[b][i] < 0
// (rows of H*d bf16, 16 B per thread)
__global__ void gather_rows_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, const int32_t* __restrict__ gidx,
                                   int n_src, int n_dst, int row_vec, size_t total) {
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int c = int(i % row_vec);
    const size_t t = i / row_vec;
    const int n = int(t % n_dst);
    const size_t b = t / n_dst;
    const int k = gidx[b * n_dst + n];
    dst[i] = k >= 0 ? src[(b * n_src + k) * row_vec + c] : make_uint4(0u, 0u, 0u, 0u);
  }
}
// dst[b, n, :, :] = cidx[b][n] >= 0 ? src[b, cidx[b][n], :, :] : 0   (every row of dst is written)
__global__ void expand_rows_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, const int32_t* __restrict__ cidx,
                                   int n_src, int n_dst, int row_vec, size_t total) {
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int c = int(i % row_vec);
    const size_t t = i / row_vec;
    const int n = int(t % n_dst);
    const size_t b = t / n_dst;
    const int k = cidx[b * n_dst + n];
    dst[i] = k >= 0 ? src[(b * n_src + k) * row_vec + c] : make_uint4(0u, 0u, 0u, 0u);
  }
}
// LSE [B*H, n]: gather (compact = 1) or expand with -inf for invalid rows (the empty-row convention)
__global__ void lse_map_kernel(const float* __restrict__ src, float* __restrict__ dst, const int32_t* __restrict__ idx,
                               int n_src, int n_dst, int H, size_t total) {
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const int n = int(i % n_dst);
    const size_t bh = i / n_dst;
    const int k = idx[(bh / H) * n_dst + n];  // the index array of this row's batch item
    dst[i] = k >= 0 ? src[bh * n_src + k] : -INFINITY;
  }
}

int grid_for(const sra_ctx* ctx, size_t total, int threads, int ctas_per_sm) {
  return int(std::max<size_t>(1, std::min<size_t>((total + threads - 1) / threads, size_t(ctx->num_sms) * ctas_per_sm)));
}

static int cbuf_get(sra_ctx* ctx, int slot, void** out) {
  if (!ctx->cbuf[slot])  // (slots 4-7 hold dO / dQ / dK / dV: only a context that also runs the backward needs them)
    if (int rc = reserve(ctx, SRA_RESERVE_VALIDITY | (slot >= 4 && slot <= 7 ? SRA_RESERVE_BACKWARD : 0))) return rc;
  *out = ctx->cbuf[slot];
  return SRA_OK;
}

int compact_rows(sra_ctx* ctx, int slot, const void* src, const void** out, cudaStream_t stream) {
  *out = nullptr;
  if (!src) return SRA_OK;
  void* dst;
  if (int rc = cbuf_get(ctx, slot, &dst)) return rc;
  *out = dst;
  const sra_config& c = ctx->cfg;
  const int row_vec = c.heads * c.head_dim / 8;
  const size_t total = size_t(c.batch) * ctx->nr * row_vec;
  if (total == 0) return SRA_OK;
  gather_rows_kernel<<<grid_for(ctx, total), 256, 0, stream>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst), ctx->d_gidx,
                                                              c.n_ref, ctx->nr, row_vec, total);
  ctx->launches += 1;
  return cudaGetLastError() == cudaSuccess ? SRA_OK : ctx_fail(ctx, SRA_ERR_CUDA, "gather_rows launch failed");
}
int compact_lse(sra_ctx* ctx, const float* src, const float** out, cudaStream_t stream) {
  *out = nullptr;
  if (!src) return SRA_OK;
  void* dst;
  if (int rc = cbuf_get(ctx, 8, &dst)) return rc;
  *out = static_cast<const float*>(dst);
  const sra_config& c = ctx->cfg;
  const size_t total = size_t(c.batch) * c.heads * ctx->nr;
  if (total == 0) return SRA_OK;
  lse_map_kernel<<<grid_for(ctx, total), 256, 0, stream>>>(src, static_cast<float*>(dst), ctx->d_gidx, c.n_ref, ctx->nr, c.heads, total);
  ctx->launches += 1;
  return cudaGetLastError() == cudaSuccess ? SRA_OK : ctx_fail(ctx, SRA_ERR_CUDA, "lse gather launch failed");
}
int compact_out(sra_ctx* ctx, int slot, void** out) { return cbuf_get(ctx, slot, out); }
int expand_rows(sra_ctx* ctx, int slot, void* dst, cudaStream_t stream) {
  if (!dst) return SRA_OK;
  const sra_config& c = ctx->cfg;
  const int row_vec = c.heads * c.head_dim / 8;
  const size_t total = size_t(c.batch) * c.n_ref * row_vec;
  expand_rows_kernel<<<grid_for(ctx, total), 256, 0, stream>>>(static_cast<const uint4*>(ctx->cbuf[slot]), static_cast<uint4*>(dst),
                                                              ctx->d_cidx, ctx->nr, c.n_ref, row_vec, total);
  ctx->launches += 1;
  return cudaGetLastError() == cudaSuccess ? SRA_OK : ctx_fail(ctx, SRA_ERR_CUDA, "expand_rows launch failed");
}
int expand_lse(sra_ctx* ctx, float* dst, cudaStream_t stream) {
  if (!dst) return SRA_OK;
  const sra_config& c = ctx->cfg;
  const size_t total = size_t(c.batch) * c.heads * c.n_ref;
  lse_map_kernel<<<grid_for(ctx, total), 256, 0, stream>>>(static_cast<const float*>(ctx->cbuf[8]), dst, ctx->d_cidx, ctx->nr, c.n_ref, c.heads, total);
  ctx->launches += 1;
  return cudaGetLastError() == cudaSuccess ? SRA_OK : ctx_fail(ctx, SRA_ERR_CUDA, "lse expand launch failed");
}

}  // namespace sra

// ------------------------------------------------------------------------------------------------ schedule
namespace {

struct Sched {
  std::vector<FwdItem> fwd, pair, split;
  std::vector<int32_t> pair_of_item;
  std::vector<BwdItem> bwd;
  int n_gen_items = 0, n_ref_items = 0, n_gen_pairs = 0, n_ref_pairs = 0, n_split = 1;
};

// Work items of ONE compaction of the reference: nr valid tokens in blocks `off`.
Sched build_one(const sra_ctx* ctx, int Nr, const std::vector<int32_t>& off, bool allow_split) {
  Sched S;
  const int Ng = ctx->cfg.n_gen;
  const int num_sms = ctx->num_sms;
  // G slabs: every generation key tile, then every reference key tile.  With a temporal window
  // ("restricts each frame's receptive field to a local neighborhood") a slab never straddles a frame
  // and walks only the generation keys of frames [f - w, f + w]; the reference stays fully visible.
  std::vector<int32_t> fr = {0, Ng};
  const bool windowed = ctx->window >= 0 && ctx->gen_frames.size() >= 2;
  if (windowed) fr = ctx->gen_frames;
  const int F = int(fr.size()) - 1;
  for (int f = 0; f < F; ++f) {
    const int lo = windowed ? fr[std::max(0, f - ctx->window)] : 0;
    const int hi = windowed ? fr[std::min(F, f + ctx->window + 1)] : Ng;
    for (int r0 = fr[f]; r0 < fr[f + 1]; r0 += kQRowsPerCta) {
      FwdItem it{};
      it.q_is_ref = 0; it.q_row0 = r0; it.q_rows = std::min(kQRowsPerCta, fr[f + 1] - r0);
      it.seg0_is_ref = 0; it.seg0_start = lo; it.seg0_len = hi - lo;
      it.seg1_start = 0; it.seg1_len = Nr;
      S.fwd.push_back(it);
    }
  }
  S.n_gen_items = int(S.fwd.size());
  // R slabs: only the keys of the slab's own block ("reference tokens only self-attend").
  for (int j = 0; j + 1 < int(off.size()); ++j) {
    const int s = off[j], e = off[j + 1];
    for (int r0 = s; r0 < e; r0 += kQRowsPerCta) {
      FwdItem it{};
      it.q_is_ref = 1; it.q_row0 = r0; it.q_rows = std::min(kQRowsPerCta, e - r0);
      it.seg0_is_ref = 1; it.seg0_start = s; it.seg0_len = e - s;
      it.seg1_start = 0; it.seg1_len = 0;
      S.fwd.push_back(it);
    }
  }
  S.n_ref_items = int(S.fwd.size()) - S.n_gen_items;
  // Short-query regime (north_star: "cache-bound short-query cases"; SURVEY.md 8d auxiliary sweep): with fewer G
  // slabs than ~2 per SM the tensor cores are idle and the step is bound by streaming K/V (mostly the resident
  // reference cache) out of HBM, so every G slab is cut into n_split key ranges of whole tiles; each range runs
  // as its own CTA and writes an fp32 partial (O_s, LSE_s), merged by sra_fwd_merge_kernel (flash-decoding).
  if (allow_split) {
    const long base = long(S.n_gen_items) * ctx->cfg.heads * ctx->cfg.batch;
    const int t0 = (Ng + kTile - 1) / kTile, t1 = (Nr + kTile - 1) / kTile;
    const int tiles = t0 + t1;
    const long waves0 = (base + num_sms - 1) / num_sms;
    const bool few = base < 2 * num_sms;                                                    // cache-bound regime
    const bool ragged_waves = base < 8 * num_sms && double(base) / double(waves0 * num_sms) < 0.85;  // e.g. 2.16 waves
    if ((few || ragged_waves) && tiles >= 16 && !windowed) {
      // Candidates keep >= 8 key tiles per split.  Take the smallest split count that fills whole waves of
      // num_sms CTAs to >= 92 % (fewer partials to write and merge); if even the largest cannot occupy every SM
      // once, take the largest.
      const int n_max = std::min(64, tiles / 8);
      int best = n_max;
      if (base * n_max >= num_sms) {
        double best_eff = 0.0;
        for (int n = 2; n <= n_max; ++n) {
          const long ctas = base * n;
          if (ctas < num_sms) continue;
          const long waves = (ctas + num_sms - 1) / num_sms;
          const double eff = double(ctas) / double(waves * num_sms);
          if (eff >= 0.92) { best = n; break; }
          if (eff > best_eff) { best_eff = eff; best = n; }
        }
      }
      S.n_split = best;
    }
    if (S.n_split > 1) {
      for (int g = 0; g < S.n_gen_items; ++g)
        for (int sp = 0; sp < S.n_split; ++sp) {
          FwdItem it = S.fwd[g];
          const int a = int(long(tiles) * sp / S.n_split), b = int(long(tiles) * (sp + 1) / S.n_split);  // tiles [a, b)
          const int g0 = std::min(a, t0), g1 = std::min(b, t0);           // generation key tiles [g0, g1)
          const int r0 = std::max(a, t0) - t0, r1 = std::max(b, t0) - t0; // reference key tiles [r0, r1)
          it.q_is_ref = (sp + 1) << 8;
          it.seg0_start = g0 * kTile; it.seg0_len = g1 > g0 ? std::min(Ng, g1 * kTile) - g0 * kTile : 0;
          it.seg1_start = r0 * kTile; it.seg1_len = r1 > r0 ? std::min(Nr, r1 * kTile) - r0 * kTile : 0;
          S.split.push_back(it);
        }
      for (int r = 0; r < S.n_ref_items; ++r) S.split.push_back(S.fwd[S.n_gen_items + r]);
    }
  }
  // CTA pairs (sra_fwd_kernel<128, 2>): two consecutive slabs of the same kind that see the same keys and tile 512
  // consecutive rows run as one cluster of two CTAs sharing every K/V tile.
  S.pair_of_item.assign(S.fwd.size() + 1, 0);
  for (size_t i = 0; i < S.fwd.size();) {
    FwdItem it = S.fwd[i];
    size_t used = 1;
    if (i + 1 < S.fwd.size()) {
      const FwdItem& nx = S.fwd[i + 1];
      if (nx.q_is_ref == it.q_is_ref && it.q_rows == kQRowsPerCta && nx.q_row0 == it.q_row0 + kQRowsPerCta &&
          nx.seg0_is_ref == it.seg0_is_ref && nx.seg0_start == it.seg0_start && nx.seg0_len == it.seg0_len &&
          nx.seg1_start == it.seg1_start && nx.seg1_len == it.seg1_len) {
        it.q_rows += nx.q_rows;
        used = 2;
      }
    }
    for (size_t k = 0; k < used; ++k) S.pair_of_item[i + k] = int32_t(S.pair.size());
    (it.q_is_ref ? S.n_ref_pairs : S.n_gen_pairs) += 1;
    S.pair.push_back(it);
    i += used;
  }
  S.pair_of_item[S.fwd.size()] = int32_t(S.pair.size());
  // Backward: key tiles.  G key tiles are seen by all G queries; R key tiles of block j additionally by block j's
  // R queries.  Tiles never straddle a block boundary.  (With a temporal window, G key tiles do not straddle frames
  // either and are seen by the queries of frames [f - w, f + w] only.)
  for (int f = 0; f < F; ++f) {
    const int lo = windowed ? fr[std::max(0, f - ctx->window)] : 0;
    const int hi = windowed ? fr[std::min(F, f + ctx->window + 1)] : Ng;
    for (int k0 = fr[f]; k0 < fr[f + 1]; k0 += kTile) {
      BwdItem it{};
      it.k_is_ref = 0; it.k_row0 = k0; it.k_rows = std::min(kTile, fr[f + 1] - k0);
      it.g_start = lo; it.g_len = hi - lo;
      S.bwd.push_back(it);
    }
  }
  for (int j = 0; j + 1 < int(off.size()); ++j) {
    const int s = off[j], e = off[j + 1];
    for (int k0 = s; k0 < e; k0 += kTile) {
      BwdItem it{};
      it.k_is_ref = 1; it.k_row0 = k0; it.k_rows = std::min(kTile, e - k0);
      it.g_start = 0; it.g_len = Ng;
      it.seg1_start = s; it.seg1_len = e - s;
      S.bwd.push_back(it);
    }
  }
  return S;
}

// Rebuilds every host list from (window, validity) and marks the device copies stale.  Per-sample masks (n_masks ==
// batch): one schedule per batch item, stacked with a common stride and padded with empty items; the G parts have the
// same length for every item (only their reference segment length differs), so "G items first" holds for the stack.
void build_schedule(sra_ctx* ctx) {
  const int M = ctx->n_masks;
  std::vector<Sched> all;
  for (int m = 0; m < M; ++m) all.push_back(build_one(ctx, ctx->nr_b[m], ctx->offe_b[m], /*allow_split=*/M == 1));
  const Sched& S0 = all[0];
  ctx->fwd_items = S0.fwd; ctx->pair_items = S0.pair; ctx->pair_of_item = S0.pair_of_item; ctx->bwd_items = S0.bwd;
  ctx->split_items = S0.split; ctx->n_split = S0.n_split;
  ctx->n_gen_items = S0.n_gen_items; ctx->n_ref_items = S0.n_ref_items;
  ctx->n_gen_pairs = S0.n_gen_pairs; ctx->n_ref_pairs = S0.n_ref_pairs;
  ctx->use_pairs = ctx->cfg.head_dim == 128 && ctx->n_split == 1;
#ifdef SRA_NO_PAIRS  // (A/B builds: the single-CTA kernel everywhere)
  ctx->use_pairs = false;
#endif
  ctx->max_ref_items = ctx->max_ref_pairs = 0;
  size_t max_bwd = 0;
  for (const Sched& S : all) {
    ctx->max_ref_items = std::max(ctx->max_ref_items, S.n_ref_items);
    ctx->max_ref_pairs = std::max(ctx->max_ref_pairs, S.n_ref_pairs);
    max_bwd = std::max(max_bwd, S.bwd.size());
  }
  ctx->fwd_stride = ctx->n_gen_items + ctx->max_ref_items;
  ctx->pair_stride = ctx->n_gen_pairs + ctx->max_ref_pairs;
  ctx->bwd_stride = int(max_bwd);
  ctx->st_fwd.assign(size_t(M) * ctx->fwd_stride, FwdItem{});
  ctx->st_pair.assign(size_t(M) * ctx->pair_stride, FwdItem{});
  ctx->st_bwd.assign(size_t(M) * ctx->bwd_stride, BwdItem{});
  for (int m = 0; m < M; ++m) {
    std::copy(all[m].fwd.begin(), all[m].fwd.end(), ctx->st_fwd.begin() + size_t(m) * ctx->fwd_stride);
    std::copy(all[m].pair.begin(), all[m].pair.end(), ctx->st_pair.begin() + size_t(m) * ctx->pair_stride);
    std::copy(all[m].bwd.begin(), all[m].bwd.end(), ctx->st_bwd.begin() + size_t(m) * ctx->bwd_stride);
  }
  // Segment ends that fall inside a tensor (sra_common.h BoundMaps): frame ends of a temporal window; block ends of
  // each mask's compacted reference (the last block ends with the item's valid rows - zero padding or the tensor's own
  // end follows, nothing to bound).
  ctx->bound_ends.clear();
  if (ctx->window >= 0 && ctx->gen_frames.size() >= 2)
    for (size_t f = 1; f + 1 < ctx->gen_frames.size(); ++f) ctx->bound_ends.push_back(ctx->gen_frames[f]);
  ctx->n_gen_ends = int(ctx->bound_ends.size());
  ctx->ref_end_stride = 0;
  for (int m = 0; m < M; ++m) ctx->ref_end_stride = std::max(ctx->ref_end_stride, int(ctx->offe_b[m].size()) - 2);
  ctx->ref_end_stride = std::max(ctx->ref_end_stride, 0);
  for (int m = 0; m < M; ++m)
    for (int j = 0; j < ctx->ref_end_stride; ++j)
      ctx->bound_ends.push_back(j + 2 < int(ctx->offe_b[m].size()) ? ctx->offe_b[m][j + 1] : INT32_MAX);
  ctx->bound_version += 1;
  ctx->sched_dirty = true;
  ctx->seg_dirty = true;
}

template <typename T>
cudaError_t ensure_pair(T* (&buf)[2], size_t& cap, size_t need) {
  if (need <= cap) return cudaSuccess;
  // growth (a schedule with more items than any before it - e.g. a temporal window over many frames): the one place a
  // sra_set_* call may allocate; the old buffers are released only after the device has finished with them
  const size_t ncap = need + need / 4 + 16;
  T* nb[2] = {nullptr, nullptr};
  cudaError_t e = cudaMalloc(&nb[0], ncap * sizeof(T));
  if (e == cudaSuccess) e = cudaMalloc(&nb[1], ncap * sizeof(T));
  if (e != cudaSuccess) { cudaFree(nb[0]); (void)cudaGetLastError(); return e; }
  if (buf[0] || buf[1]) { cudaDeviceSynchronize(); cudaFree(buf[0]); cudaFree(buf[1]); }
  buf[0] = nb[0]; buf[1] = nb[1];
  cap = ncap;
  return cudaSuccess;
}

// Device buffers for the current host lists (no-op unless a list outgrew its buffers).
int ensure_schedule_capacity(sra_ctx* ctx) {
  const sra_config& c = ctx->cfg;
  cudaError_t e = ensure_pair(ctx->d_fwd_items, ctx->cap_fwd, ctx->st_fwd.size());
  if (e == cudaSuccess) e = ensure_pair(ctx->d_pair_items, ctx->cap_pair, ctx->st_pair.size());
  if (e == cudaSuccess) e = ensure_pair(ctx->d_bwd_items, ctx->cap_bwd, ctx->st_bwd.size());
  if (e == cudaSuccess && ctx->n_split > 1) {
    e = ensure_pair(ctx->d_split_items, ctx->cap_split, ctx->split_items.size());
    const size_t prow = size_t(ctx->n_split) * c.batch * c.heads * c.n_gen;
    if (e == cudaSuccess && prow > ctx->cap_part_rows) {
      if (ctx->ws_part_o) { cudaDeviceSynchronize(); cudaFree(ctx->ws_part_o); cudaFree(ctx->ws_part_lse); ctx->ws_part_o = ctx->ws_part_lse = nullptr; }
      e = cudaMalloc(&ctx->ws_part_o, prow * c.head_dim * sizeof(float));
      if (e == cudaSuccess) e = cudaMalloc(&ctx->ws_part_lse, prow * sizeof(float));
      if (e == cudaSuccess) ctx->cap_part_rows = prow;
    }
  }
  // bounded tensor maps: 6 roles forward, 8 backward
  const size_t n_ends = ctx->bound_ends.size();
  if (e == cudaSuccess) e = ensure_pair(ctx->bnd_fwd.d_ends, ctx->bnd_fwd.cap_ends, n_ends);
  if (e == cudaSuccess) e = ensure_pair(ctx->bnd_fwd.d_maps, ctx->bnd_fwd.cap_maps, 6 * n_ends);
  if (e == cudaSuccess) e = ensure_pair(ctx->bnd_bwd.d_ends, ctx->bnd_bwd.cap_ends, n_ends);
  if (e == cudaSuccess) e = ensure_pair(ctx->bnd_bwd.d_maps, ctx->bnd_bwd.cap_maps, 8 * n_ends);
  if (e != cudaSuccess) { (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? SRA_ERR_OOM : SRA_ERR_CUDA; }
  return SRA_OK;
}

}  // namespace

namespace sra {

// Called at the head of every launching entry point: if sra_set_temporal_window / sra_set_reference_validity changed
// the host lists, copies them into the OTHER device buffer on `stream` and flips to it.  The copies are from pageable
// host memory (staged by the runtime before the call returns), ordered before this call's kernels on the same stream;
// kernels launched earlier keep reading the buffer they were given.
int sync_schedule(sra_ctx* ctx, cudaStream_t stream) {
  if (!ctx->sched_dirty && !ctx->idx_dirty) return SRA_OK;
  cudaError_t e = cudaSuccess;
  if (ctx->sched_dirty) {
    if (int rc = ensure_schedule_capacity(ctx)) return ctx_fail(ctx, rc, "schedule buffer allocation failed");
    const int nb = ctx->sched_buf ^ 1;
    auto up = [&](void* dst, const void* src, size_t bytes) {
      if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);
    };
    up(ctx->d_fwd_items[nb], ctx->st_fwd.data(), ctx->st_fwd.size() * sizeof(FwdItem));
    up(ctx->d_pair_items[nb], ctx->st_pair.data(), ctx->st_pair.size() * sizeof(FwdItem));
    up(ctx->d_bwd_items[nb], ctx->st_bwd.data(), ctx->st_bwd.size() * sizeof(BwdItem));
    if (ctx->n_split > 1) up(ctx->d_split_items[nb], ctx->split_items.data(), ctx->split_items.size() * sizeof(FwdItem));
    if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "schedule upload");
    ctx->sched_buf = nb;
    ctx->sched_dirty = false;
  }
  if (ctx->idx_dirty) {
    if (ctx->has_valid) {
      if (int rc = reserve(ctx, SRA_RESERVE_VALIDITY)) return rc;
      if (!ctx->h_gidx.empty()) e = cudaMemcpyAsync(ctx->d_gidx, ctx->h_gidx.data(), ctx->h_gidx.size() * 4, cudaMemcpyHostToDevice, stream);
      if (e == cudaSuccess && !ctx->h_cidx.empty()) e = cudaMemcpyAsync(ctx->d_cidx, ctx->h_cidx.data(), ctx->h_cidx.size() * 4, cudaMemcpyHostToDevice, stream);
      if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "validity index upload");
    }
    ctx->idx_dirty = false;
  }
  return SRA_OK;
}

int bound_maps(sra_ctx* ctx, sra_ctx::BoundSet& bs, const sra_ctx::BoundRole* roles, int n_roles, cudaStream_t stream,
               BoundMaps* out) {
  const size_t n_total = ctx->bound_ends.size();
  *out = BoundMaps{};
#ifdef SRA_NO_BOUND  // (A/B builds: the kernels see no bounded maps)
  return SRA_OK;
#endif
  if (n_total == 0) return SRA_OK;
  // (a role the call does not pass - q_ref on a cached step - keeps the maps of the last call that did)
  bool same = bs.version == ctx->bound_version && int(bs.roles.size()) == n_roles;
  for (int r = 0; same && r < n_roles; ++r) same = roles[r].ptr == nullptr || bs.roles[r] == roles[r];
  if (!same) {
    std::vector<sra_ctx::BoundRole> merged(roles, roles + n_roles);
    if (bs.version == ctx->bound_version && int(bs.roles.size()) == n_roles)
      for (int r = 0; r < n_roles; ++r)
        if (merged[r].ptr == nullptr) merged[r] = bs.roles[r];
    roles = merged.data();
    if (bs.cap_ends < n_total || bs.cap_maps < size_t(n_roles) * n_total)
      return ctx_fail(ctx, SRA_ERR_CUDA, "bounded tensor-map buffers were not sized by the schedule build");
    const sra_config& c = ctx->cfg;
    bs.h_maps.assign(size_t(n_roles) * n_total, CUtensorMap{});
    for (int r = 0; r < n_roles; ++r) {
      if (!roles[r].ptr) continue;
      const size_t i0 = roles[r].is_ref ? size_t(ctx->n_gen_ends) : 0, i1 = roles[r].is_ref ? n_total : size_t(ctx->n_gen_ends);
      for (size_t i = i0; i < i1; ++i) {
        const int end = ctx->bound_ends[i];
        if (end <= 0 || end >= roles[r].N) continue;  // padding, or the tensor's own end
        if (int rc = encode_tmap_bf16(ctx, &bs.h_maps[size_t(r) * n_total + i], roles[r].ptr, c.batch, roles[r].N, c.heads,
                                      c.head_dim, roles[r].head_major, roles[r].box_rows, end))
          return rc;
      }
    }
    const int nb = bs.buf ^ 1;
    cudaError_t e = cudaMemcpyAsync(bs.d_ends[nb], ctx->bound_ends.data(), n_total * sizeof(int32_t), cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess)
      e = cudaMemcpyAsync(bs.d_maps[nb], bs.h_maps.data(), bs.h_maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "bounded tensor-map upload");
    bs.buf = nb;
    bs.version = ctx->bound_version;
    bs.roles.assign(roles, roles + n_roles);
  }
  out->maps = bs.d_maps[bs.buf];
  out->ends = bs.d_ends[bs.buf];
  out->n_gen_ends = ctx->n_gen_ends;
  out->ref_stride = ctx->ref_end_stride;
  out->n_total = int(n_total);
  return SRA_OK;
}

// One-time allocations of the optional paths.  Everything is sized from the config for the largest case (unmasked
// reference), so nothing is ever re-allocated when a mask or window changes.
int reserve(sra_ctx* ctx, uint32_t what) {
  const sra_config& c = ctx->cfg;
  what &= ~ctx->reserved;
  if (!what) return SRA_OK;
  cudaError_t e = cudaSuccess;
  const size_t row = size_t(c.heads) * c.head_dim * 2;
  if (what & SRA_RESERVE_BACKWARD) {
    const int n_pad = (c.n_gen + c.n_ref + 63) / 64 * 64;
    const size_t vec_bytes = size_t(c.batch) * c.heads * n_pad * 4;
    e = cudaMalloc(&ctx->ws_dq, vec_bytes * c.head_dim);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->ws_delta, vec_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->ws_lse2, vec_bytes);
    if (e != cudaSuccess) {
      (void)cudaGetLastError();
      cudaFree(ctx->ws_dq); cudaFree(ctx->ws_delta); cudaFree(ctx->ws_lse2);
      ctx->ws_dq = ctx->ws_delta = ctx->ws_lse2 = nullptr;
      return ctx_fail(ctx, SRA_ERR_OOM, "backward workspace allocation failed");
    }
    ctx->reserved |= SRA_RESERVE_BACKWARD;
  }
  if (what & SRA_RESERVE_VALIDITY) {
    const size_t rows = size_t(c.batch) * std::max(c.n_ref, 1);
    for (int slot : {0, 1, 2, 3, 8})
      if (e == cudaSuccess && !ctx->cbuf[slot]) e = cudaMalloc(&ctx->cbuf[slot], slot == 8 ? rows * c.heads * 4 : rows * row);
    if (e == cudaSuccess && !ctx->d_gidx) e = cudaMalloc(&ctx->d_gidx, rows * 4);
    if (e == cudaSuccess && !ctx->d_cidx) e = cudaMalloc(&ctx->d_cidx, rows * 4);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return ctx_fail(ctx, SRA_ERR_OOM, "validity compaction buffer allocation failed"); }
    ctx->reserved |= SRA_RESERVE_VALIDITY;
  }
  if ((ctx->reserved & (SRA_RESERVE_VALIDITY | SRA_RESERVE_BACKWARD)) == (SRA_RESERVE_VALIDITY | SRA_RESERVE_BACKWARD)) {
    // compacted dO, dQ, dK, dV of the reference: needed only where a mask meets the backward
    const size_t rows = size_t(c.batch) * std::max(c.n_ref, 1);
    for (int slot = 4; slot <= 7; ++slot)
      if (e == cudaSuccess && !ctx->cbuf[slot]) e = cudaMalloc(&ctx->cbuf[slot], rows * row);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return ctx_fail(ctx, SRA_ERR_OOM, "validity compaction buffer allocation failed"); }
  }
  if (what & SRA_RESERVE_HOST) {
    constexpr int kChunks = 8;
    const size_t gen_bytes = size_t(c.batch) * c.n_gen * row, ref_bytes = size_t(c.batch) * std::max(c.n_ref, 1) * row;
    const size_t want[8] = {gen_bytes, gen_bytes, gen_bytes, gen_bytes, ref_bytes, ref_bytes,
                            size_t(c.batch) * c.heads * c.n_gen * 4, size_t(c.batch) * c.heads * std::max(c.n_ref, 1) * 4};
    for (int i = 0; i < 8 && e == cudaSuccess; ++i)
      if (!ctx->stage[i]) e = cudaMalloc(&ctx->stage[i], want[i]);
    // segment partials of the reference-first phase, per batch item
    const size_t prow = 3 * size_t(c.batch) * c.heads * c.n_gen;  // reference segment + up to two generation-key chunks
    if (e == cudaSuccess && !ctx->ws_seg_o) e = cudaMalloc(&ctx->ws_seg_o, prow * c.head_dim * sizeof(float));
    if (e == cudaSuccess && !ctx->ws_seg_lse) e = cudaMalloc(&ctx->ws_seg_lse, prow * sizeof(float));
    if (e == cudaSuccess) e = ensure_pair(ctx->d_seg_items, ctx->cap_seg, 3 * size_t(std::max(ctx->n_gen_items, 1)));  // [A ; B_0 ; B_1]
    if (e != cudaSuccess) { (void)cudaGetLastError(); return ctx_fail(ctx, SRA_ERR_OOM, "host staging allocation failed"); }
    if (!ctx->s_h2d) {
      e = cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking);
      if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking);
      ctx->pipe_ev.assign(2 * kChunks + 6, nullptr);
      for (cudaEvent_t& ev : ctx->pipe_ev)
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreate(&ctx->rate_ev[0]);
      if (e == cudaSuccess) e = cudaEventCreate(&ctx->rate_ev[1]);
      if (e != cudaSuccess) return ctx_fail_cuda(ctx, e, "pipeline stream / event creation");
      // host -> device copy bandwidth of this box, measured once (64 MB from pinned memory; the second copy is timed):
      // it sizes the reference-first phase of the pipelined step
      void* hbuf = nullptr;
      const size_t probe = std::min<size_t>(size_t(64) << 20, gen_bytes);
      if (cudaMallocHost(&hbuf, probe) == cudaSuccess) {
        std::memset(hbuf, 0, probe);
        cudaMemcpyAsync(ctx->stage[0], hbuf, probe, cudaMemcpyHostToDevice, ctx->s_h2d);
        cudaEventRecord(ctx->rate_ev[0], ctx->s_h2d);
        cudaMemcpyAsync(ctx->stage[0], hbuf, probe, cudaMemcpyHostToDevice, ctx->s_h2d);
        cudaEventRecord(ctx->rate_ev[1], ctx->s_h2d);
        float ms = 0.f;
        if (cudaEventSynchronize(ctx->rate_ev[1]) == cudaSuccess && cudaEventElapsedTime(&ms, ctx->rate_ev[0], ctx->rate_ev[1]) == cudaSuccess && ms > 0.f)
          ctx->h2d_gbs = double(probe) / (ms * 1e-3) / 1e9;
        cudaFreeHost(hbuf);
      }
      (void)cudaGetLastError();
    }
    ctx->reserved |= SRA_RESERVE_HOST;
  }
  return SRA_OK;
}

}  // namespace sra

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

const char* sra_status_string(int s) {
  switch (s) {
    case SRA_OK: return "SRA_OK";
    case SRA_ERR_INVALID_ARG: return "SRA_ERR_INVALID_ARG";
    case SRA_ERR_UNSUPPORTED: return "SRA_ERR_UNSUPPORTED";
    case SRA_ERR_CUDA: return "SRA_ERR_CUDA";
    case SRA_ERR_NO_REF_CACHE: return "SRA_ERR_NO_REF_CACHE";
    case SRA_ERR_OOM: return "SRA_ERR_OOM";
    default: return "SRA_ERR_UNKNOWN";
  }
}

const char* sra_last_error(const sra_ctx* ctx) { return ctx ? ctx->err.c_str() : ""; }

int sra_create(const sra_config* cfg, sra_ctx** out) {
  if (!out) return SRA_ERR_INVALID_ARG;
  *out = nullptr;
  if (!cfg) return SRA_ERR_INVALID_ARG;
  if (cfg->batch < 1 || cfg->heads < 1 || cfg->n_gen < 1 || cfg->n_ref < 0 || cfg->n_ref_blocks < 0)
    return SRA_ERR_INVALID_ARG;
  if (cfg->head_dim != 64 && cfg->head_dim != 128) return SRA_ERR_UNSUPPORTED;
  if ((cfg->n_ref == 0) != (cfg->n_ref_blocks == 0)) return SRA_ERR_INVALID_ARG;
  if (cfg->n_ref_blocks > 0) {
    if (!cfg->ref_block_offsets || cfg->ref_block_offsets[0] != 0) return SRA_ERR_INVALID_ARG;
    for (int j = 0; j < cfg->n_ref_blocks; ++j)
      if (cfg->ref_block_offsets[j + 1] <= cfg->ref_block_offsets[j]) return SRA_ERR_INVALID_ARG;
    if (cfg->ref_block_offsets[cfg->n_ref_blocks] != cfg->n_ref) return SRA_ERR_INVALID_ARG;
  }
  if (cfg->heads > 65535 || cfg->batch > 65535) return SRA_ERR_INVALID_ARG;
  sra_ctx* ctx = new (std::nothrow) sra_ctx();
  if (!ctx) return SRA_ERR_OOM;
  ctx->cfg = *cfg;
  ctx->off.assign(1, 0);
  for (int j = 0; j < cfg->n_ref_blocks; ++j) ctx->off.push_back(cfg->ref_block_offsets[j + 1]);
  ctx->cfg.ref_block_offsets = nullptr;
  ctx->scale = cfg->softmax_scale > 0.f ? cfg->softmax_scale : 1.0f / std::sqrt(float(cfg->head_dim));
  ctx->nr = cfg->n_ref;
  ctx->n_masks = 1;
  ctx->nr_b.assign(1, cfg->n_ref);
  ctx->offe_b.assign(1, ctx->off);

  // Device discovery.  Without a usable CUDA device the ctx is host-only: the schedule can be inspected, every
  // compute entry point fails with SRA_ERR_UNSUPPORTED (there is no CPU fallback).
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    (void)cudaGetLastError();
    ctx->device = -1;
    build_schedule(ctx);
    *out = ctx;
    return SRA_OK;
  }
  int dev = cfg->device;
  if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) dev = 0;
  if (dev >= ndev) { delete ctx; return SRA_ERR_INVALID_ARG; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { (void)cudaGetLastError(); delete ctx; return SRA_ERR_CUDA; }
  ctx->device = dev;
  // the library carries sm_100a code only ('a' targets are not forward compatible: an sm_103 part cannot run it)
  ctx->sm100 = prop.major == 10 && prop.minor == 0;
  if (ctx->sm100) ctx->num_sms = prop.multiProcessorCount;
  build_schedule(ctx);
  if (ctx->sm100) {
    // Everything sra_cache_reference_kv / sra_forward need is allocated here, sized from the config: the device
    // schedule buffers, the key-split workspace and the resident cache (2 * B * n_ref * H * d bf16).
    sra::DeviceGuard guard(dev);
    if (int rc = ensure_schedule_capacity(ctx)) { sra_destroy(ctx); return rc; }
    const size_t elems = size_t(cfg->batch) * cfg->n_ref * cfg->heads * cfg->head_dim;
    if (elems > 0) {
      cudaError_t e = cudaMalloc(&ctx->cache_k, elems * 2);
      if (e == cudaSuccess) e = cudaMalloc(&ctx->cache_v, elems * 2);
      if (e != cudaSuccess) { (void)cudaGetLastError(); sra_destroy(ctx); return SRA_ERR_OOM; }
    }
  }
  *out = ctx;
  return SRA_OK;
}

void sra_destroy(sra_ctx* ctx) {
  if (!ctx) return;
  if (ctx->device >= 0) {
    sra::DeviceGuard guard(ctx->device);
    for (int i = 0; i < 2; ++i) {
      cudaFree(ctx->d_fwd_items[i]); cudaFree(ctx->d_pair_items[i]); cudaFree(ctx->d_split_items[i]);
      cudaFree(ctx->d_bwd_items[i]); cudaFree(ctx->d_seg_items[i]);
      cudaFree(ctx->bnd_fwd.d_maps[i]); cudaFree(ctx->bnd_fwd.d_ends[i]);
      cudaFree(ctx->bnd_bwd.d_maps[i]); cudaFree(ctx->bnd_bwd.d_ends[i]);
    }
    cudaFree(ctx->ws_part_o);
    cudaFree(ctx->ws_part_lse);
    cudaFree(ctx->ws_seg_o);
    cudaFree(ctx->ws_seg_lse);
    cudaFree(ctx->d_gidx);
    cudaFree(ctx->d_cidx);
    for (void* q : ctx->cbuf) cudaFree(q);
    cudaFree(ctx->cache_k);
    cudaFree(ctx->cache_v);
    cudaFree(ctx->ws_dq);
    cudaFree(ctx->ws_delta);
    cudaFree(ctx->ws_lse2);
    for (void* s : ctx->stage) cudaFree(s);
    if (ctx->s_h2d) cudaStreamDestroy(ctx->s_h2d);
    if (ctx->s_d2h) cudaStreamDestroy(ctx->s_d2h);
    for (cudaEvent_t ev : ctx->pipe_ev)
      if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : ctx->rate_ev)
      if (ev) cudaEventDestroy(ev);
    for (auto& e : ctx->ev)
      for (cudaEvent_t x : e)
        if (x) cudaEventDestroy(x);
    (void)cudaGetLastError();
  }
  delete ctx;
}

static int check_device(sra_ctx* ctx) {
  if (ctx->device < 0) return fail(ctx, SRA_ERR_UNSUPPORTED, "no CUDA device: this library has no CPU path");
  if (!ctx->sm100) return fail(ctx, SRA_ERR_UNSUPPORTED, "device is not sm_100 (B200); kernels are sm_100a-only");
  return SRA_OK;
}

int sra_reserve(sra_ctx* ctx, uint32_t what) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (what & ~uint32_t(SRA_RESERVE_BACKWARD | SRA_RESERVE_HOST | SRA_RESERVE_VALIDITY)) return fail(ctx, SRA_ERR_INVALID_ARG, "unknown SRA_RESERVE_* bit");
  if (int rc = check_device(ctx)) return rc;
  sra::DeviceGuard guard(ctx->device);
  return sra::reserve(ctx, what);
}

static int cache_reference_kv(sra_ctx* ctx, const void* k_ref, const void* v_ref, const float* cos_ref, const float* sin_ref,
                              bool rope, void* cuda_stream) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (int rc = check_device(ctx)) return rc;
  if (ctx->cfg.n_ref == 0) return SRA_OK;
  if (!k_ref || !v_ref) return fail(ctx, SRA_ERR_INVALID_ARG, "k_ref / v_ref must be non-NULL");
  if (rope && (!cos_ref || !sin_ref)) return fail(ctx, SRA_ERR_INVALID_ARG, "cos_ref / sin_ref must be non-NULL");
  const sra_config& c = ctx->cfg;
  sra::DeviceGuard guard(ctx->device);
  if (int rc = sra::sync_schedule(ctx, cudaStream_t(cuda_stream))) return rc;
  if (ctx->nr == 0) { ctx->cache_valid = true; return SRA_OK; }  // every reference token is invalid: nothing to cache
  const size_t elems = size_t(c.batch) * ctx->nr * c.heads * c.head_dim;
  const int vec = c.head_dim / 8;
  const size_t total = elems / 8;
  const int threads = 256;
  const int blocks = sra::grid_for(ctx, total, threads);
  cudaError_t e;
  {
    sra::KernelTimer kt(ctx, SRA_KERNEL_CACHE_RELAYOUT, cudaStream_t(cuda_stream));
    const int32_t* gidx = ctx->has_valid ? ctx->d_gidx : nullptr;
    if (rope)
      sra::relayout_rope_head_major_kernel<<<blocks, threads, 0, cudaStream_t(cuda_stream)>>>(
          static_cast<const uint4*>(k_ref), static_cast<const uint4*>(v_ref), reinterpret_cast<uint4*>(ctx->cache_k),
          reinterpret_cast<uint4*>(ctx->cache_v), ctx->nr, c.heads, vec, total, gidx, c.n_ref,
          reinterpret_cast<const float4*>(cos_ref), reinterpret_cast<const float4*>(sin_ref));
    else
      sra::relayout_head_major_kernel<<<blocks, threads, 0, cudaStream_t(cuda_stream)>>>(
          static_cast<const uint4*>(k_ref), static_cast<const uint4*>(v_ref), reinterpret_cast<uint4*>(ctx->cache_k),
          reinterpret_cast<uint4*>(ctx->cache_v), ctx->nr, c.heads, vec, total, gidx, c.n_ref);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return fail_cuda(ctx, e, "cache relayout launch");
  ctx->launches += 1;
  ctx->cache_valid = true;
  return SRA_OK;
}

int sra_cache_reference_kv(sra_ctx* ctx, const void* k_ref, const void* v_ref, void* cuda_stream) {
  nvtx_range r("sra_cache_reference_kv");
  return cache_reference_kv(ctx, k_ref, v_ref, nullptr, nullptr, false, cuda_stream);
}

int sra_cache_reference_kv_rope(sra_ctx* ctx, const void* k_ref, const void* v_ref, const float* cos_ref,
                                const float* sin_ref, void* cuda_stream) {
  nvtx_range r("sra_cache_reference_kv_rope");
  return cache_reference_kv(ctx, k_ref, v_ref, cos_ref, sin_ref, true, cuda_stream);
}

int sra_apply_rope(sra_ctx* ctx, void* x0, void* x1, const float* cos, const float* sin, int32_t n_tokens,
                   void* cuda_stream) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (int rc = check_device(ctx)) return rc;
  if (n_tokens <= 0) return SRA_OK;
  if (!x0 || !cos || !sin) return fail(ctx, SRA_ERR_INVALID_ARG, "x0 / cos / sin must be non-NULL");
  const sra_config& c = ctx->cfg;
  sra::DeviceGuard guard(ctx->device);
  const int vec = c.head_dim / 8;
  const size_t total = size_t(c.batch) * n_tokens * c.heads * vec;
  cudaError_t e;
  {
    sra::KernelTimer kt(ctx, SRA_KERNEL_ROPE, cudaStream_t(cuda_stream));
    sra::rope_inplace_kernel<<<sra::grid_for(ctx, total), 256, 0, cudaStream_t(cuda_stream)>>>(
        static_cast<uint4*>(x0), static_cast<uint4*>(x1), n_tokens, c.heads, vec, total,
        reinterpret_cast<const float4*>(cos), reinterpret_cast<const float4*>(sin));
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return fail_cuda(ctx, e, "rope launch");
  ctx->launches += 1;
  return SRA_OK;
}

static int forward_core(sra_ctx* ctx, const sra_fwd_args* a, void* cuda_stream);
static int forward_checked(sra_ctx* ctx, const sra_fwd_args* a, void* cuda_stream);

int sra_forward(sra_ctx* ctx, const sra_fwd_args* a, void* cuda_stream) {
  nvtx_range r("sra_forward");
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (!a) return fail(ctx, SRA_ERR_INVALID_ARG, "args is NULL");
  if (int rc = check_device(ctx)) return rc;
  sra::DeviceGuard guard(ctx->device);
  return forward_checked(ctx, a, cuda_stream);
}

// sra_forward without the entry-point bookkeeping (also the device leg of sra_forward_host)
static int forward_checked(sra_ctx* ctx, const sra_fwd_args* a, void* cuda_stream) {
  const sra_config& c = ctx->cfg;
  if (!a->q_gen || !a->k_gen || !a->v_gen || !a->o_gen) return fail(ctx, SRA_ERR_INVALID_ARG, "q_gen/k_gen/v_gen/o_gen required");
  if ((a->k_ref == nullptr) != (a->v_ref == nullptr)) return fail(ctx, SRA_ERR_INVALID_ARG, "k_ref and v_ref must both be NULL or both non-NULL");
  const bool with_ref_rows = a->q_ref != nullptr && c.n_ref > 0;
  if (with_ref_rows && !a->o_ref) return fail(ctx, SRA_ERR_INVALID_ARG, "o_ref required when q_ref is given");
  const bool use_cache = c.n_ref > 0 && a->k_ref == nullptr;
  if (use_cache && !ctx->cache_valid) return fail(ctx, SRA_ERR_NO_REF_CACHE, "k_ref/v_ref NULL but sra_cache_reference_kv was never called");
  const void* ptrs[] = {a->q_gen, a->k_gen, a->v_gen, a->q_ref, a->k_ref, a->v_ref, a->o_gen, a->o_ref};
  for (const void* q : ptrs)
    if (q && (reinterpret_cast<uintptr_t>(q) & 15)) return fail(ctx, SRA_ERR_INVALID_ARG, "tensor pointers must be 16-byte aligned");
  cudaStream_t st = cudaStream_t(cuda_stream);
  if (int rc = sra::sync_schedule(ctx, st)) return rc;

  if (!ctx->has_valid || c.n_ref == 0) return forward_core(ctx, a, cuda_stream);
  // Validity path: the kernels run on the compacted reference; invalid reference rows get
  // O = 0, LSE = -inf.
  sra_fwd_args e = *a;
  int rc;
  if ((rc = sra::compact_rows(ctx, 0, a->q_ref, &e.q_ref, st))) return rc;
  if ((rc = sra::compact_rows(ctx, 1, a->k_ref, &e.k_ref, st))) return rc;
  if ((rc = sra::compact_rows(ctx, 2, a->v_ref, &e.v_ref, st))) return rc;
  e.o_ref = nullptr; e.lse_ref = nullptr;
  if (with_ref_rows) {
    void* q;
    if ((rc = sra::compact_out(ctx, 3, &q))) return rc;
    e.o_ref = q;
    if (a->lse_ref) { if ((rc = sra::compact_out(ctx, 8, &q))) return rc; e.lse_ref = static_cast<float*>(q); }
  }
  if ((rc = forward_core(ctx, &e, cuda_stream))) return rc;
  if (with_ref_rows) {
    if ((rc = sra::expand_rows(ctx, 3, a->o_ref, st))) return rc;
    if (a->lse_ref && (rc = sra::expand_lse(ctx, a->lse_ref, st))) return rc;
  }
  return SRA_OK;
}

// The launch itself, on the effective (validity-compacted) reference: `a` holds device pointers whose reference
// tensors have nr rows.
static int forward_core(sra_ctx* ctx, const sra_fwd_args* a, void* cuda_stream) {
  const sra_config& c = ctx->cfg;
  const int nr = ctx->nr;
  const bool with_ref_rows = a->q_ref != nullptr && nr > 0;
  const bool use_cache = nr > 0 && a->k_ref == nullptr;
  CUtensorMap maps[6];
  const int B = c.batch, H = c.heads, d = c.head_dim;
  int rc;
  // CTA pairs: each CTA loads 64 of a K tile's 128 keys (box of 64 rows); V shares are ordinary [128 x 64] boxes
  const bool pairs = ctx->use_pairs;
  const int k_box = pairs ? kTile / 2 : kTile;
  if ((rc = sra::make_tmap_bf16(ctx, &maps[0], a->q_gen, B, c.n_gen, H, d, false, kTile))) return rc;
  if ((rc = sra::make_tmap_bf16(ctx, &maps[1], a->k_gen, B, c.n_gen, H, d, false, k_box))) return rc;
  if ((rc = sra::make_tmap_bf16(ctx, &maps[2], a->v_gen, B, c.n_gen, H, d, false, kTile))) return rc;
  maps[3] = maps[0]; maps[4] = maps[1]; maps[5] = maps[2];  // placeholders when n_ref == 0 (never dereferenced)
  if (nr > 0) {
    if (with_ref_rows && (rc = sra::make_tmap_bf16(ctx, &maps[3], a->q_ref, B, nr, H, d, false, kTile))) return rc;
    const void* kr = use_cache ? ctx->cache_k : a->k_ref;
    const void* vr = use_cache ? ctx->cache_v : a->v_ref;
    if ((rc = sra::make_tmap_bf16(ctx, &maps[4], kr, B, nr, H, d, use_cache, k_box))) return rc;
    if ((rc = sra::make_tmap_bf16(ctx, &maps[5], vr, B, nr, H, d, use_cache, kTile))) return rc;
  }
  sra::FwdParams p{};
  const bool split = ctx->n_split > 1;
  const int sb = ctx->sched_buf;
  p.items = split ? ctx->d_split_items[sb] : pairs ? ctx->d_pair_items[sb] : ctx->d_fwd_items[sb];
  p.n_items = pairs ? ctx->n_gen_pairs + (with_ref_rows ? ctx->max_ref_pairs : 0)
                    : ctx->n_gen_items * ctx->n_split + (with_ref_rows ? ctx->max_ref_items : 0);
  p.item_batch_stride = ctx->n_masks > 1 ? (pairs ? ctx->pair_stride : ctx->fwd_stride) : 0;
  p.part_o = ctx->ws_part_o;
  p.part_lse = ctx->ws_part_lse;
  const bool seg = ctx->sub_seg;  // segment-split items of the pipelined host path (merged by its caller)
  if (seg) {
    p.items = ctx->d_seg_items[ctx->seg_buf];
    p.part_o = ctx->ws_seg_o;
    p.part_lse = ctx->ws_seg_lse;
  }
  if (ctx->sub_count >= 0) {  // sra_forward_host pipelines a step as several launches over item sub-ranges
    // the range is given in 256-row slabs (indices into fwd_items, or into the [A ; B] segment list of the generation
    // slabs); with pairs it starts and ends on pair boundaries (the caller snaps its chunks) and is converted
    int first = ctx->sub_first, end = ctx->sub_first + ctx->sub_count;
    if (pairs) {
      const int G = ctx->n_gen_items;
      auto pi = [&](int idx) {
        if (seg) return (idx / G) * ctx->n_gen_pairs + int(ctx->pair_of_item[idx % G]);  // list [A ; B_0 ; ...] of G slabs each
        if (idx >= G + ctx->n_ref_items) return ctx->pair_stride;  // end of the (padded) reference range
        return int(ctx->pair_of_item[idx]);
      };
      first = pi(first);
      end = pi(end);
    }
    p.items += first;
    p.n_items = end - first;
    if (p.n_items <= 0) return SRA_OK;
  }
  p.heads = H; p.batch = B; p.n_gen = c.n_gen; p.n_ref = nr;
  p.scale = ctx->scale;
  p.scale_log2 = ctx->scale * 1.4426950408889634f;
  p.o_gen = static_cast<__nv_bfloat16*>(a->o_gen);
  p.o_ref = static_cast<__nv_bfloat16*>(a->o_ref);
  p.lse_gen = a->lse_gen;
  p.lse_ref = a->lse_ref;
  p.ref_kv_head_major = use_cache ? 1 : 0;
  {
    const void* kr = nr > 0 ? (use_cache ? ctx->cache_k : a->k_ref) : nullptr;
    const void* vr = nr > 0 ? (use_cache ? ctx->cache_v : a->v_ref) : nullptr;
    const sra_ctx::BoundRole roles[6] = {{a->k_gen, c.n_gen, false, false, k_box}, {a->v_gen, c.n_gen, false, false, kTile},
                                         {kr, nr, true, use_cache, k_box}, {vr, nr, true, use_cache, kTile},
                                         {a->q_gen, c.n_gen, false, false, kTile},
                                         {with_ref_rows ? a->q_ref : nullptr, nr, true, false, kTile}};
    if ((rc = sra::bound_maps(ctx, ctx->bnd_fwd, roles, 6, cudaStream_t(cuda_stream), &p.bound))) return rc;
  }
  cudaError_t e;
  {
    sra::KernelTimer kt(ctx, SRA_KERNEL_FWD, cudaStream_t(cuda_stream));
    e = pairs ? sra::launch_fwd<128, 2>(maps, p, cudaStream_t(cuda_stream))
        : (d == 128) ? sra::launch_fwd<128, 1>(maps, p, cudaStream_t(cuda_stream))
                     : sra::launch_fwd<64, 1>(maps, p, cudaStream_t(cuda_stream));
  }
  if (e != cudaSuccess) return fail_cuda(ctx, e, "sra_fwd_kernel launch");
  ctx->launches += 1;
  if (split && !seg) {
    sra::KernelTimer kt(ctx, SRA_KERNEL_FWD_MERGE, cudaStream_t(cuda_stream));
    e = sra::launch_fwd_merge(p, d, ctx->n_split, cudaStream_t(cuda_stream), ctx->num_sms * 16);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "sra_fwd_merge_kernel launch");
    ctx->launches += 1;
  }
  return SRA_OK;
}

// Pipelined host path.  The generation rows go in kChunks slabs whose H2D copy (slab c+1) and D2H copy
// (slab c-1) run on their own streams under the forward launch of slab c (query slabs are independent work items,
// PCIe is full duplex).  The one transfer nothing could hide - K_g and V_g, which every generation row needs - is
// covered by "reference keys first" (the reference K/V are already resident): the first n_first slabs
// are uploaded ahead of K_g / V_g and attend the REFERENCE segment only while K_g / V_g are in flight (A items, fp32
// partials); once K_g / V_g have landed they attend the generation segment (B items) and the two partials of every
// row are merged by sra_fwd_merge_kernel (the key-split machinery of the short-query regime).  The remaining
// slabs run the ordinary single-pass items.  The reference rows go in before the last slab; launches cover several
// slabs where the copies allow.  With batch > 1 a slab is the same row range of every batch item (strided copies);
// with a validity mask the reference rows are gathered from / scattered into the staged tensors.  Everything is
// ordered after prior work on `st`, and `st` is made to wait for the last D2H copy, so the call stays asynchronous
// on the caller's stream.
static int forward_host_pipelined(sra_ctx* ctx, const sra_fwd_host_args* a, cudaStream_t st, bool with_ref_rows) {
  constexpr int kChunks = 8;
  const sra_config& c = ctx->cfg;
  const int Bn = c.batch;
  const size_t row = size_t(c.heads) * c.head_dim * 2;
  const size_t gen_pitch = size_t(c.n_gen) * row;            // one batch item of a generation tensor
  const size_t gen_bytes = size_t(Bn) * gen_pitch, ref_bytes = size_t(Bn) * c.n_ref * row;
  // How many slabs take the reference-first route: enough reference-segment work to cover the K_g / V_g upload, at
  // most kChunks - 2.  Both rates are measured: the copy bandwidth when the staging was reserved, the forward rate
  // from the previous call's launches (a first call assumes 1 PFLOP/s).
  int n_first = 0;
  bool copy_bound = false;  // even kChunks - 2 slabs of reference-segment work do not cover the K_g / V_g upload
  if (ctx->nr > 0 && ctx->n_masks == 1) {
    if (ctx->rate_pending && cudaEventQuery(ctx->rate_ev[1]) == cudaSuccess) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, ctx->rate_ev[0], ctx->rate_ev[1]) == cudaSuccess && ms > 0.f) ctx->fwd_flops_per_s = ctx->rate_flops / (ms * 1e-3);
      ctx->rate_pending = false;
    }
    (void)cudaGetLastError();
    const double t_up = 2.0 * double(gen_bytes) / (ctx->h2d_gbs * 1e9);
    const double t_chunk = 4.0 * c.head_dim * double(c.n_gen) * double(ctx->nr) * c.heads * Bn / ctx->fwd_flops_per_s / kChunks;
    const double need = std::ceil(t_up / t_chunk);
    n_first = int(std::min<double>(kChunks - 2, need));
    copy_bound = need > kChunks - 2;
  }
  const int G = ctx->n_gen_items;
  // Copy-bound shapes (480p, the training batch: the reference-segment work of the first slabs is shorter than the K_g /
  // V_g upload) also stream the generation keys: K_g / V_g go up in kc = 2 halves and the first slabs attend half c as
  // soon as it has landed (B_c items, partial 1 + c), instead of idling until the whole upload is in.
  const int k_mid = (c.n_gen / kTile / 2) * kTile;
  const int kc = (n_first > 0 && copy_bound && ctx->window < 0 && k_mid > 0) ? 2 : 1;
  if (n_first > 0 && (ctx->seg_dirty || ctx->seg_kc != kc)) {
    // (with CTA pairs the lists are built from the generation PAIR items)
    const std::vector<sra::FwdItem>& src = ctx->use_pairs ? ctx->pair_items : ctx->fwd_items;
    const int Gs = ctx->use_pairs ? ctx->n_gen_pairs : G;
    std::vector<sra::FwdItem> seg((1 + size_t(kc)) * Gs);
    for (int g = 0; g < Gs; ++g) {
      sra::FwdItem A = src[g];
      A.q_is_ref = 1 << 8; A.seg0_len = 0;                   // partial 0: reference keys only
      seg[g] = A;
      for (int kp = 0; kp < kc; ++kp) {                      // partial 1 + kp: generation keys (of half kp) only
        sra::FwdItem Bi = src[g];
        Bi.q_is_ref = (2 + kp) << 8; Bi.seg1_len = 0;
        if (kc == 2) {                                       // (no window: seg0 = [0, n_gen))
          Bi.seg0_start = kp == 0 ? 0 : k_mid;
          Bi.seg0_len = kp == 0 ? k_mid : c.n_gen - k_mid;
        }
        seg[(1 + size_t(kp)) * Gs + g] = Bi;
      }
    }
    // (sized for the three-list form at once: the measured rates may switch kc between calls, and no call after the
    //  first may allocate)
    cudaError_t e = ensure_pair(ctx->d_seg_items, ctx->cap_seg, 3 * size_t(Gs));
    const int nb = ctx->seg_buf ^ 1;
    if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->d_seg_items[nb], seg.data(), seg.size() * sizeof(sra::FwdItem), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(ctx, SRA_ERR_OOM, "reference-first item list upload failed"); }
    ctx->seg_buf = nb;
    ctx->seg_dirty = false;
    ctx->seg_kc = kc;
  }
  cudaEvent_t* ev_q = ctx->pipe_ev.data();            // [kChunks] slab c of Q is on the device
  cudaEvent_t* ev_c = ev_q + kChunks;                 // [kChunks] slab c of O is computed
  cudaEvent_t ev_start = ev_c[kChunks], ev_kv = ev_c[kChunks + 1], ev_qr = ev_c[kChunks + 2], ev_cr = ev_c[kChunks + 3],
              ev_done = ev_c[kChunks + 4], ev_kv0 = ev_c[kChunks + 5];
  char* dq = static_cast<char*>(ctx->stage[0]);
  char* dout = static_cast<char*>(ctx->stage[3]);
  const char* hq = static_cast<const char*>(a->q_gen);
  char* hout = static_cast<char*>(a->o_gen);
  sra_fwd_args d{};
  d.q_gen = ctx->stage[0]; d.k_gen = ctx->stage[1]; d.v_gen = ctx->stage[2]; d.o_gen = ctx->stage[3];
  d.lse_gen = a->lse_gen ? static_cast<float*>(ctx->stage[6]) : nullptr;
  const int per = (G + kChunks - 1) / kChunks;
  auto chunk_start = [&](int ch) {  // first slab of chunk ch; never the second slab of a CTA pair
    int i = std::min(ch * per, G);
    if (ctx->use_pairs && i > 0 && i < G && ctx->pair_of_item[i] == ctx->pair_of_item[i - 1]) ++i;
    return i;
  };
  auto rows_of = [&](int ch, int& i0, int& i1, size_t& r0, size_t& r1) {
    i0 = chunk_start(ch);
    i1 = chunk_start(ch + 1);
    // G items are ordered by row and tile [0, n_gen) (with a temporal window they are cut at frame boundaries, so
    // an item is not always kQRowsPerCta rows)
    r0 = i0 < G ? size_t(ctx->fwd_items[i0].q_row0) : size_t(c.n_gen);
    r1 = i1 < G ? size_t(ctx->fwd_items[i1].q_row0) : size_t(c.n_gen);
  };
  // rows [r0, r1) of every batch item (one strided copy)
  auto copy_rows = [&](char* dst, const char* src, size_t r0, size_t r1, cudaMemcpyKind kind, cudaStream_t s) {
    if (r1 <= r0) return cudaSuccess;
    if (Bn == 1) return cudaMemcpyAsync(dst + r0 * row, src + r0 * row, (r1 - r0) * row, kind, s);
    return cudaMemcpy2DAsync(dst + r0 * row, gen_pitch, src + r0 * row, gen_pitch, (r1 - r0) * row, Bn, kind, s);
  };
  cudaError_t e = cudaEventRecord(ev_start, st);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->s_h2d, ev_start, 0);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->s_d2h, ev_start, 0);
  // every H2D copy is enqueued (and its event recorded) before the first launch waits on one:
  // Q slabs [0, n_first), K_g, V_g, Q slabs [n_first, kChunks), q_ref
  auto copy_q = [&](int ch) {
    int i0, i1; size_t r0, r1;
    rows_of(ch, i0, i1, r0, r1);
    if (e == cudaSuccess && i1 > i0) e = copy_rows(dq, hq, r0, r1, cudaMemcpyHostToDevice, ctx->s_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(ev_q[ch], ctx->s_h2d);
  };
  for (int ch = 0; ch < n_first; ++ch) copy_q(ch);
  for (int kp = 0; kp < kc; ++kp) {  // K_g / V_g, whole or in two key halves (rows [k0, k1) of every batch item)
    const size_t k0 = kp == 0 ? 0 : size_t(k_mid), k1 = kp == kc - 1 ? size_t(c.n_gen) : size_t(k_mid);
    if (e == cudaSuccess) e = copy_rows(static_cast<char*>(ctx->stage[1]), static_cast<const char*>(a->k_gen), k0, k1, cudaMemcpyHostToDevice, ctx->s_h2d);
    if (e == cudaSuccess) e = copy_rows(static_cast<char*>(ctx->stage[2]), static_cast<const char*>(a->v_gen), k0, k1, cudaMemcpyHostToDevice, ctx->s_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(kp == kc - 1 ? ev_kv : ev_kv0, ctx->s_h2d);
  }
  for (int ch = n_first; ch < kChunks; ++ch) copy_q(ch);
  if (e == cudaSuccess && with_ref_rows) {
    e = cudaMemcpyAsync(ctx->stage[4], a->q_ref, ref_bytes, cudaMemcpyHostToDevice, ctx->s_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(ev_qr, ctx->s_h2d);
  }
  if (e != cudaSuccess) return fail_cuda(ctx, e, "host->device copy");
  auto launch = [&](bool seg, int first, int count, const sra_fwd_args& args, bool checked) -> int {
    ctx->sub_seg = seg; ctx->sub_first = first; ctx->sub_count = count;
    const int rc = checked ? forward_checked(ctx, &args, st) : forward_core(ctx, &args, st);
    ctx->sub_seg = false; ctx->sub_count = -1;
    return rc;
  };
  // Launches are grouped over several slabs wherever the copies allow it: every kernel boundary drains the GPU
  // through a partially filled last wave (~0.6 ms at 720p), so fewer, larger launches.
  auto span = [&](int c0, int c1, int& i0, int& i1, size_t& r0, size_t& r1) {  // slabs [c0, c1)
    int x; size_t y;
    rows_of(c0, i0, x, r0, y);
    rows_of(c1 - 1, x, i1, y, r1);
  };
  auto copy_out = [&](int c0, int c1) {  // rows of slabs [c0, c1) are final in the staging buffer: send them home
    int i0, i1; size_t r0, r1;
    span(c0, c1, i0, i1, r0, r1);
    if (e == cudaSuccess) e = cudaEventRecord(ev_c[c0], st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->s_d2h, ev_c[c0], 0);
    if (e == cudaSuccess) e = copy_rows(hout, dout, r0, r1, cudaMemcpyDeviceToHost, ctx->s_d2h);
  };
  // phase 1: reference segment of the first slabs, under the K_g / V_g upload (slab 0 as soon as it has landed, the
  // others together: their copies are long done when slab 0's launch ends)
  for (int g = 0; g < 2 && e == cudaSuccess; ++g) {
    const int c0 = g == 0 ? 0 : 1, c1 = g == 0 ? std::min(1, n_first) : n_first;
    if (c1 <= c0) continue;
    int i0, i1; size_t r0, r1;
    span(c0, c1, i0, i1, r0, r1);
    e = cudaStreamWaitEvent(st, ev_q[c1 - 1], 0);
    if (e != cudaSuccess) break;
    if (int rc = launch(true, i0, i1 - i0, d, false)) return rc;
  }
  if (e == cudaSuccess) e = cudaStreamWaitEvent(st, kc == 2 ? ev_kv0 : ev_kv, 0);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "pipelined host copy");
  auto run_ref_rows = [&]() -> int {
    // reference rows: their q_ref copy has had the first slabs' compute time to land; their output copy is
    // hidden under the last slab.  (Under a validity mask forward_checked gathers the valid rows of the staged Q_r
    // and scatters O_r / LSE_r back into the staged outputs.)
    cudaError_t er = cudaStreamWaitEvent(st, ev_qr, 0);
    if (er != cudaSuccess) return fail_cuda(ctx, er, "pipelined host copy");
    sra_fwd_args dr = d;
    dr.q_ref = ctx->stage[4]; dr.o_ref = ctx->stage[5];
    dr.lse_ref = a->lse_ref ? static_cast<float*>(ctx->stage[7]) : nullptr;
    if (int rc = launch(false, G, ctx->max_ref_items, dr, true)) return rc;
    er = cudaEventRecord(ev_cr, st);
    if (er == cudaSuccess) er = cudaStreamWaitEvent(ctx->s_d2h, ev_cr, 0);
    if (er == cudaSuccess) er = cudaMemcpyAsync(a->o_ref, ctx->stage[5], ref_bytes, cudaMemcpyDeviceToHost, ctx->s_d2h);
    if (er == cudaSuccess && dr.lse_ref) er = cudaMemcpyAsync(a->lse_ref, dr.lse_ref, size_t(Bn) * c.heads * c.n_ref * 4, cudaMemcpyDeviceToHost, ctx->s_d2h);
    return er == cudaSuccess ? SRA_OK : fail_cuda(ctx, er, "pipelined host copy");
  };
  // phase 2: generation segment of the first slabs in one launch, one merge of their partials
  if (n_first > 0) {
    int i0, i1; size_t r0, r1;
    span(0, n_first, i0, i1, r0, r1);
    for (int kp = 0; kp < kc; ++kp) {
      if (kp == 1) {  // the second half of K_g / V_g
        e = cudaStreamWaitEvent(st, ev_kv, 0);
        if (e != cudaSuccess) return fail_cuda(ctx, e, "pipelined host copy");
      }
      if (int rc = launch(true, (1 + kp) * G + i0, i1 - i0, d, false)) return rc;
    }
    sra::FwdParams mp{};
    mp.part_o = ctx->ws_seg_o; mp.part_lse = ctx->ws_seg_lse;
    mp.o_gen = static_cast<__nv_bfloat16*>(d.o_gen); mp.lse_gen = d.lse_gen;
    mp.batch = Bn; mp.heads = c.heads; mp.n_gen = c.n_gen;
    {
      sra::KernelTimer kt(ctx, SRA_KERNEL_FWD_MERGE, st);
      e = sra::launch_fwd_merge(mp, c.head_dim, 1 + kc, st, ctx->num_sms * 16, int(r0), int(r1 - r0));
    }
    if (e != cudaSuccess) return fail_cuda(ctx, e, "sra_fwd_merge_kernel launch");
    if (r1 > r0) ctx->launches += 1;
    copy_out(0, n_first);
  }
  // phase 3: the ordinary slabs - all but the last in one launch (without a reference-first phase slab 0 goes alone,
  // as soon as it has landed), the reference rows, then the last slab, under which the other outputs go home
  {
    const int mid0 = n_first > 0 ? n_first : 1;
    const int groups[3][2] = {{n_first, n_first > 0 ? n_first : 1}, {mid0, kChunks - 1}, {kChunks - 1, kChunks}};
    for (int g = 0; g < 3 && e == cudaSuccess; ++g) {
      const int c0 = groups[g][0], c1 = groups[g][1];
      if (g == 2 && with_ref_rows)
        if (int rc = run_ref_rows()) return rc;
      if (c1 <= c0) continue;
      int i0, i1; size_t r0, r1;
      span(c0, c1, i0, i1, r0, r1);
      e = cudaStreamWaitEvent(st, ev_q[c1 - 1], 0);
      if (e != cudaSuccess) break;
      const bool time_it = g == 1 && i1 > i0 && !ctx->rate_pending;  // the big middle launch calibrates the forward rate
      if (time_it) cudaEventRecord(ctx->rate_ev[0], st);
      if (int rc = launch(false, i0, i1 - i0, d, false)) return rc;
      if (time_it) {
        cudaEventRecord(ctx->rate_ev[1], st);
        ctx->rate_flops = 4.0 * c.head_dim * double(r1 - r0) * (double(c.n_gen) + double(ctx->nr)) * c.heads * Bn;
        if (ctx->window >= 0) ctx->rate_flops = 0.0;  // (a windowed slab sees fewer keys: no calibration from it)
        ctx->rate_pending = ctx->rate_flops > 0.0;
      }
      copy_out(c0, c1);
    }
  }
  if (e == cudaSuccess && d.lse_gen)
    e = cudaMemcpyAsync(a->lse_gen, d.lse_gen, size_t(Bn) * c.heads * c.n_gen * 4, cudaMemcpyDeviceToHost, ctx->s_d2h);
  if (e == cudaSuccess) e = cudaEventRecord(ev_done, ctx->s_d2h);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_done, 0);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "pipelined host copy");
  return SRA_OK;
}

int sra_forward_host(sra_ctx* ctx, const sra_fwd_host_args* a, void* cuda_stream) {
  nvtx_range r("sra_forward_host");
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (!a) return fail(ctx, SRA_ERR_INVALID_ARG, "args is NULL");
  if (int rc = check_device(ctx)) return rc;
  const sra_config& c = ctx->cfg;
  if (!a->q_gen || !a->k_gen || !a->v_gen || !a->o_gen) return fail(ctx, SRA_ERR_INVALID_ARG, "q_gen/k_gen/v_gen/o_gen required");
  const bool with_ref_rows = a->q_ref != nullptr && c.n_ref > 0;
  if (with_ref_rows && !a->o_ref) return fail(ctx, SRA_ERR_INVALID_ARG, "o_ref required when q_ref is given");
  if (c.n_ref > 0 && !ctx->cache_valid) return fail(ctx, SRA_ERR_NO_REF_CACHE, "sra_forward_host reads reference K/V from the resident cache");
  sra::DeviceGuard guard(ctx->device);
  if (int rc = sra::reserve(ctx, SRA_RESERVE_HOST)) return rc;
  const size_t row = size_t(c.heads) * c.head_dim * 2;
  const size_t gen_bytes = size_t(c.batch) * c.n_gen * row, ref_bytes = size_t(c.batch) * c.n_ref * row;
  const size_t lse_gen_bytes = size_t(c.batch) * c.heads * c.n_gen * 4, lse_ref_bytes = size_t(c.batch) * c.heads * c.n_ref * 4;
  cudaStream_t st = cudaStream_t(cuda_stream);
  if (int rc = sra::sync_schedule(ctx, st)) return rc;
  if (ctx->n_split == 1 && ctx->n_gen_items >= 16)
    return forward_host_pipelined(ctx, a, st, with_ref_rows);
  // few generation slabs (the short-query regime): the step is a handful of milliseconds of copies around a
  // sub-millisecond launch - nothing to pipeline
  cudaError_t e = cudaMemcpyAsync(ctx->stage[0], a->q_gen, gen_bytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->stage[1], a->k_gen, gen_bytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->stage[2], a->v_gen, gen_bytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess && with_ref_rows) e = cudaMemcpyAsync(ctx->stage[4], a->q_ref, ref_bytes, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "host->device copy");
  sra_fwd_args d{};
  d.q_gen = ctx->stage[0]; d.k_gen = ctx->stage[1]; d.v_gen = ctx->stage[2]; d.o_gen = ctx->stage[3];
  if (with_ref_rows) { d.q_ref = ctx->stage[4]; d.o_ref = ctx->stage[5]; }
  d.lse_gen = a->lse_gen ? static_cast<float*>(ctx->stage[6]) : nullptr;
  d.lse_ref = (with_ref_rows && a->lse_ref) ? static_cast<float*>(ctx->stage[7]) : nullptr;
  if (int rc = forward_checked(ctx, &d, cuda_stream)) return rc;
  e = cudaMemcpyAsync(a->o_gen, ctx->stage[3], gen_bytes, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && with_ref_rows) e = cudaMemcpyAsync(a->o_ref, ctx->stage[5], ref_bytes, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && d.lse_gen) e = cudaMemcpyAsync(a->lse_gen, d.lse_gen, lse_gen_bytes, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && d.lse_ref) e = cudaMemcpyAsync(a->lse_ref, d.lse_ref, lse_ref_bytes, cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "device->host copy");
  return SRA_OK;
}

int sra_backward(sra_ctx* ctx, const sra_bwd_args* a, void* cuda_stream) {
  nvtx_range r("sra_backward");
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (!a) return fail(ctx, SRA_ERR_INVALID_ARG, "args is NULL");
  if (int rc = check_device(ctx)) return rc;
  sra::DeviceGuard guard(ctx->device);
  return sra::run_backward(ctx, a, cudaStream_t(cuda_stream));
}

int sra_useful_flops(const sra_ctx* ctx, int include_ref_rows, int backward, double* out) {
  if (!ctx || !out) return SRA_ERR_INVALID_ARG;
  const sra_config& c = ctx->cfg;
  double pairs = 0.0;
  for (int b = 0; b < c.batch; ++b) {
    const int m = ctx->mask_of(b);
    const double nr = ctx->nr_b[m];  // invalid reference tokens are not useful work
    if (ctx->window >= 0 && ctx->gen_frames.size() >= 2) {  // temporal window: generation keys of frames [f - w, f + w] only
      const std::vector<int32_t>& fr = ctx->gen_frames;
      const int F = int(fr.size()) - 1;
      for (int f = 0; f < F; ++f)
        pairs += double(fr[f + 1] - fr[f]) *
                 (double(fr[std::min(F, f + ctx->window + 1)] - fr[std::max(0, f - ctx->window)]) + nr);
    } else {
      pairs += double(c.n_gen) * (double(c.n_gen) + nr);
    }
    if (include_ref_rows)
      for (size_t j = 0; j + 1 < ctx->offe_b[m].size(); ++j) {
        const double bsz = double(ctx->offe_b[m][j + 1] - ctx->offe_b[m][j]);
        pairs += bsz * bsz;
      }
  }
  *out = 4.0 * c.head_dim * pairs * c.heads * (backward ? 2.5 : 1.0);
  return SRA_OK;
}

int sra_schedule_info(const sra_ctx* ctx, int32_t* n_gen_items, int32_t* n_ref_items, int64_t* key_tiles_gen,
                      int64_t* key_tiles_ref) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  int64_t tg = 0, tr = 0;
  for (size_t i = 0; i < ctx->fwd_items.size(); ++i) {
    const FwdItem& it = ctx->fwd_items[i];
    const int64_t qt = (it.q_rows + kTile - 1) / kTile;
    const int64_t t = qt * ((it.seg0_len + kTile - 1) / kTile + (it.seg1_len + kTile - 1) / kTile);
    (it.q_is_ref ? tr : tg) += t;
  }
  if (n_gen_items) *n_gen_items = ctx->n_gen_items;
  if (n_ref_items) *n_ref_items = ctx->n_ref_items;
  if (key_tiles_gen) *key_tiles_gen = tg;
  if (key_tiles_ref) *key_tiles_ref = tr;
  return SRA_OK;
}

static int copy_items(const std::vector<FwdItem>& v, int32_t* items, int32_t capacity, int32_t* n_items) {
  static_assert(sizeof(FwdItem) == 8 * sizeof(int32_t), "FwdItem layout is part of the ABI");
  if (n_items) *n_items = int32_t(v.size());
  if (items) {
    const int n = std::min<int>(capacity, int(v.size()));
    std::memcpy(items, v.data(), size_t(std::max(n, 0)) * sizeof(FwdItem));
  }
  return SRA_OK;
}

int sra_schedule_copy(const sra_ctx* ctx, int32_t* items, int32_t capacity, int32_t* n_items) {
  if (!ctx || !n_items) return SRA_ERR_INVALID_ARG;
  return copy_items(ctx->fwd_items, items, capacity, n_items);
}

int sra_batch_schedule_copy(const sra_ctx* ctx, int32_t batch_item, int32_t* items, int32_t capacity, int32_t* n_items) {
  if (!ctx || !n_items || batch_item < 0 || batch_item >= ctx->cfg.batch) return SRA_ERR_INVALID_ARG;
  const int m = ctx->mask_of(batch_item);
  std::vector<FwdItem> v;
  for (int i = 0; i < ctx->fwd_stride; ++i) {
    const FwdItem& it = ctx->st_fwd[size_t(m) * ctx->fwd_stride + i];
    if (it.q_rows > 0) v.push_back(it);  // (padding items are not part of the schedule)
  }
  return copy_items(v, items, capacity, n_items);
}

int sra_pair_schedule_copy(const sra_ctx* ctx, int32_t* use_pairs, int32_t* items, int32_t capacity, int32_t* n_items) {
  if (!ctx || !use_pairs) return SRA_ERR_INVALID_ARG;
  *use_pairs = ctx->use_pairs ? 1 : 0;
  return copy_items(ctx->pair_items, items, capacity, n_items);
}

int sra_bound_ends_copy(const sra_ctx* ctx, int32_t* ends, int32_t capacity, int32_t* n_gen_ends, int32_t* ref_stride,
                        int32_t* n_ends) {
  if (!ctx || !n_ends) return SRA_ERR_INVALID_ARG;
  *n_ends = int32_t(ctx->bound_ends.size());
  if (n_gen_ends) *n_gen_ends = ctx->n_gen_ends;
  if (ref_stride) *ref_stride = ctx->ref_end_stride;
  if (ends) {
    if (capacity < *n_ends) return SRA_ERR_INVALID_ARG;
    std::copy(ctx->bound_ends.begin(), ctx->bound_ends.end(), ends);
  }
  return SRA_OK;
}

int sra_split_schedule_copy(const sra_ctx* ctx, int32_t* n_split, int32_t* items, int32_t capacity, int32_t* n_items) {
  if (!ctx || !n_split) return SRA_ERR_INVALID_ARG;
  *n_split = ctx->n_split;
  return copy_items(ctx->n_split > 1 ? ctx->split_items : ctx->fwd_items, items, capacity, n_items);
}

int sra_set_temporal_window(sra_ctx* ctx, int32_t n_frames, const int32_t* gen_frame_offsets, int32_t window) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (window >= 0) {
    if (n_frames < 1 || !gen_frame_offsets || gen_frame_offsets[0] != 0 || gen_frame_offsets[n_frames] != ctx->cfg.n_gen)
      return fail(ctx, SRA_ERR_INVALID_ARG, "gen_frame_offsets must run from 0 to n_gen");
    for (int f = 0; f < n_frames; ++f)
      if (gen_frame_offsets[f + 1] <= gen_frame_offsets[f]) return fail(ctx, SRA_ERR_INVALID_ARG, "gen_frame_offsets must be strictly increasing");
    ctx->gen_frames.assign(gen_frame_offsets, gen_frame_offsets + n_frames + 1);
    ctx->window = window;
  } else {
    ctx->gen_frames.clear();
    ctx->window = -1;
  }
  build_schedule(ctx);  // host lists only: the next launch uploads them on its own stream (sra::sync_schedule)
  return SRA_OK;
}

int sra_set_reference_validity_batched(sra_ctx* ctx, const uint8_t* valid, int32_t n_masks) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  const sra_config& c = ctx->cfg;
  if (valid && n_masks != 1 && n_masks != c.batch) return fail(ctx, SRA_ERR_INVALID_ARG, "n_masks must be 1 or batch");
  const int M = valid ? n_masks : 1;
  const int n_ref = std::max(c.n_ref, 0);
  std::vector<std::vector<int32_t>> gidx(M), offe(M);
  bool all = true;
  int nr_max = 0;
  for (int m = 0; m < M; ++m) {
    const uint8_t* v = valid ? valid + size_t(m) * n_ref : nullptr;
    offe[m].assign(1, 0);
    for (size_t j = 0; j + 1 < ctx->off.size(); ++j) {
      int cnt = 0;
      for (int t = ctx->off[j]; t < ctx->off[j + 1]; ++t) {
        if (!v || v[t]) { gidx[m].push_back(t); ++cnt; } else all = false;
      }
      if (cnt > 0) offe[m].push_back(offe[m].back() + cnt);  // a block with no valid token disappears
    }
    nr_max = std::max(nr_max, int(gidx[m].size()));
  }
  ctx->has_valid = !all;
  ctx->n_masks = all ? 1 : M;
  ctx->nr = all ? c.n_ref : nr_max;
  ctx->nr_b.clear(); ctx->offe_b.clear();
  for (int m = 0; m < ctx->n_masks; ++m) {
    ctx->nr_b.push_back(all ? c.n_ref : int(gidx[m].size()));
    ctx->offe_b.push_back(all ? ctx->off : offe[m]);
  }
  // index arrays per BATCH ITEM (a shared mask is replicated): compact row -> token (-1 = padding), token -> compact row
  ctx->h_gidx.clear(); ctx->h_cidx.clear();
  if (ctx->has_valid) {
    ctx->h_gidx.assign(size_t(c.batch) * std::max(ctx->nr, 0), -1);
    ctx->h_cidx.assign(size_t(c.batch) * n_ref, -1);
    for (int b = 0; b < c.batch; ++b) {
      const std::vector<int32_t>& g = gidx[M == 1 ? 0 : b];
      for (size_t i = 0; i < g.size(); ++i) {
        ctx->h_gidx[size_t(b) * ctx->nr + i] = g[i];
        ctx->h_cidx[size_t(b) * n_ref + g[i]] = int32_t(i);
      }
    }
  }
  ctx->idx_dirty = true;
  ctx->cache_valid = false;  // the resident cache holds the previous compaction
  ctx->tmaps.clear();        // (maps over ctx-owned compacted buffers describe the previous row count)
  build_schedule(ctx);       // host lists only: uploaded by the next launch, on its stream
  return SRA_OK;
}

int sra_set_reference_validity(sra_ctx* ctx, const uint8_t* valid) { return sra_set_reference_validity_batched(ctx, valid, 1); }

int64_t sra_cache_bytes(const sra_ctx* ctx) {
  if (!ctx || !ctx->cache_k || !ctx->cache_valid) return 0;
  const sra_config& c = ctx->cfg;
  int64_t rows = 0;
  for (int b = 0; b < c.batch; ++b) rows += ctx->nr_b[ctx->mask_of(b)];
  return int64_t(2) * rows * c.heads * c.head_dim * 2;
}

int sra_set_kernel_timing(sra_ctx* ctx, int enable) {
  if (!ctx) return SRA_ERR_INVALID_ARG;
  ctx->err.clear();
  if (int rc = check_device(ctx)) return rc;
  sra::DeviceGuard guard(ctx->device);
  if (enable && !ctx->ev[0][0]) {
    for (auto& e : ctx->ev)
      for (cudaEvent_t& x : e)
        if (cudaEventCreate(&x) != cudaSuccess) return fail(ctx, SRA_ERR_CUDA, "cudaEventCreate failed");
  }
  ctx->timing = enable != 0;
  for (bool& r : ctx->ev_recorded) r = false;
  return SRA_OK;
}

int sra_kernel_time_ms(sra_ctx* ctx, int which, float* ms) {
  if (!ctx || !ms || which < 0 || which >= SRA_NUM_KERNELS) return SRA_ERR_INVALID_ARG;
  if (!ctx->timing || !ctx->ev_recorded[which]) return fail(ctx, SRA_ERR_INVALID_ARG, "kernel timing is off or the kernel was not launched");
  sra::DeviceGuard guard(ctx->device);
  cudaError_t e = cudaEventSynchronize(ctx->ev[which][1]);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms, ctx->ev[which][0], ctx->ev[which][1]);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaEventElapsedTime");
  return SRA_OK;
}

int64_t sra_launch_count(const sra_ctx* ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"
