// sra_forward_gen_static: the generation rows' attention for callers that
// cannot call cudaMalloc - code under CUDA graph capture, tight serving loops, harnesses that forbid it.
//
// It is the key-split short-query path of sra_forward (sra_fwd_kernel writing fp32 partials, then a merge) with NO
// context: every byte of scratch - the work-item list and the partials (O_s, LSE_s) - lives in ONE file-scope
// `static __device__` array of SRA_STATIC_SCRATCH_BYTES, which every GPU that loads the library holds until exit.
// The entry point calls no cudaMalloc / cudaFree / allocating routine and copies nothing from the host: the work items
// are written by a one-block kernel, the tensor maps travel as kernel parameters.
//
// In HOST code the array's name is a host-side stand-in, not a device address: the device address is taken once per
// device, with that device current, by cudaGetSymbolAddress (scratch_of below) and handed to sra_fwd_kernel (defined
// in sra_fwd.cu) as a pointer; the two kernels of THIS file name the array directly.
//
// Every call shares the array and finds the last call's contents in it.  Nothing has to start at zero: the item list
// and every partial row that the merge reads are rewritten by the call itself.  Calls that overlap on the GPU (two
// streams, two host threads) race on it - callers serialise.
#include <algorithm>
#include <cstdio>
#include <cstring>

#include "ptx.cuh"
#include "sra_common.h"
#include "sra_ctx.h"

namespace {

using sra::FwdItem;
using sra::kQRowsPerCta;
using sra::kTile;

constexpr size_t kScratchBytes = SRA_STATIC_SCRATCH_BYTES;
constexpr size_t kItemBytes = 64 * 1024;                       // work items first: up to 2048 of them
constexpr int kMaxItems = int(kItemBytes / sizeof(FwdItem));
static_assert(sizeof(FwdItem) == 32, "work item layout");

static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

thread_local char t_err[256] = "";

int fail(int code, const char* fmt, double a = 0, double b = 0) {
  std::snprintf(t_err, sizeof(t_err), fmt, a, b);
  return code;
}
int fail_cuda(cudaError_t e, const char* what) {
  std::snprintf(t_err, sizeof(t_err), "%s: %s", what, cudaGetErrorString(e));
  (void)cudaGetLastError();
  return SRA_ERR_CUDA;
}

// ---- set-up, once per device: the array's DEVICE address and what the device is
struct DeviceInfo {
  void* scratch = nullptr;
  int num_sms = 0;
  bool sm100 = false;
  bool ready = false;
};
DeviceInfo g_dev[64];

int scratch_of(int dev, DeviceInfo** out) {  // (the caller has made `dev` current)
  if (dev < 0 || dev >= 64) return fail(SRA_ERR_INVALID_ARG, "device ordinal out of range");
  DeviceInfo& d = g_dev[dev];
  if (!d.ready) {
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (e != cudaSuccess || ptr == nullptr) {
      (void)cudaGetLastError();
      std::snprintf(t_err, sizeof(t_err), "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
      return SRA_ERR_CUDA;
    }
    int major = 0, minor = 0, sms = 0;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    d.scratch = ptr;
    d.num_sms = sms > 0 ? sms : 148;
    d.sm100 = major == 10 && minor == 0;
    d.ready = true;
  }
  *out = &d;
  return SRA_OK;
}

}  // namespace

namespace sra {
// ---- the work items, written on the device straight into the array (named directly: device code may).
// Slab g = rows [256 g, 256 g + 256) of Q_g; split sp of n_split takes key tiles [tiles sp / n_split, tiles (sp + 1) /
// n_split) of the t0 generation + t1 reference key tiles (whole 128-key tiles; the same cut as the library's key-split
// schedule) and writes partial sp.
__global__ void sra_static_items_kernel(int n_gen, int n_ref, int n_slabs, int n_split) {
  FwdItem* items = reinterpret_cast<FwdItem*>(g_static_scratch);
  const int t0 = (n_gen + kTile - 1) / kTile, t1 = (n_ref + kTile - 1) / kTile;
  const long long tiles = t0 + t1;
  for (int i = threadIdx.x; i < n_slabs * n_split; i += blockDim.x) {
    const int g = i / n_split, sp = i % n_split;
    const int a = int(tiles * sp / n_split), b = int(tiles * (sp + 1) / n_split);
    const int g0 = min(a, t0), g1 = min(b, t0);
    const int r0 = max(a, t0) - t0, r1 = max(b, t0) - t0;
    FwdItem it;
    it.q_is_ref = (sp + 1) << 8;
    it.q_row0 = g * kQRowsPerCta;
    it.q_rows = min(kQRowsPerCta, n_gen - g * kQRowsPerCta);
    it.seg0_is_ref = 0;
    it.seg0_start = g0 * kTile;
    it.seg0_len = g1 > g0 ? min(n_gen, g1 * kTile) - g0 * kTile : 0;
    it.seg1_start = r0 * kTile;
    it.seg1_len = r1 > r0 ? min(n_ref, r1 * kTile) - r0 * kTile : 0;
    items[i] = it;
  }
}

// ---- merge (the variant of sra_fwd_merge_kernel whose partials sit in the static array, named directly):
// O = sum_s exp(LSE_s - LSE) O_s, LSE = log sum_s exp(LSE_s); one warp per (batch, token, head) output row.
template <int D>
__global__ void sra_static_merge_kernel(size_t off_lse, size_t off_o, __nv_bfloat16* __restrict__ o_gen,
                                        float* __restrict__ lse_gen, int n_split, int B, int H, int n_gen) {
  const float* part_lse = reinterpret_cast<const float*>(g_static_scratch + off_lse);
  const float* part_o = reinterpret_cast<const float*>(g_static_scratch + off_o);
  const int lane = threadIdx.x & 31;
  const size_t warp_id = (blockIdx.x * size_t(blockDim.x) + threadIdx.x) >> 5;
  const size_t n_warps = (gridDim.x * size_t(blockDim.x)) >> 5;
  const size_t rows = size_t(B) * n_gen * H;
  const size_t split_stride = size_t(B) * H * n_gen;
  constexpr int V = D / 32;  // floats per lane
  for (size_t r = warp_id; r < rows; r += n_warps) {
    const int h = int(r % H);
    const size_t t = r / H;
    const int n = int(t % n_gen);
    const int b = int(t / n_gen);
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
#pragma unroll
      for (int k = 0; k < V; ++k) acc[k] = fmaf(w, src[k], acc[k]);
    }
    const float inv = 1.0f / wsum;
    __nv_bfloat16* dst = o_gen + ((size_t(b) * n_gen + n) * H + h) * D + lane * V;
#pragma unroll
    for (int k = 0; k < V; k += 2) *reinterpret_cast<uint32_t*>(dst + k) = sra::pack_bf16(acc[k] * inv, acc[k + 1] * inv);
    if (lse_gen != nullptr && lane == 0) lse_gen[prow] = m + __logf(wsum);
  }
}

}  // namespace sra

namespace {
// Smallest split count (>= 8 key tiles per split) that fills whole waves of CTAs to >= 92 %, else the one that fills
// them best; 1 when the keys are too few to cut.
int auto_split(long base_ctas, int tiles, int num_sms) {
  const int n_max = std::min(64, tiles / 8);
  if (n_max < 2) return 1;
  int best = n_max;
  if (base_ctas * n_max >= num_sms) {
    double best_eff = 0.0;
    for (int n = 1; n <= n_max; ++n) {
      const long ctas = base_ctas * n;
      if (ctas < num_sms) continue;
      const long waves = (ctas + num_sms - 1) / num_sms;
      const double eff = double(ctas) / double(waves * num_sms);
      if (eff >= 0.92) return n;
      if (eff > best_eff) { best_eff = eff; best = n; }
    }
  }
  return best;
}

size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

}  // namespace

extern "C" {

const char* sra_static_last_error(void) { return t_err; }

int sra_static_scratch_bytes(const sra_static_fwd_args* a, int32_t n_split, int64_t* bytes) {
  if (!a || !bytes || n_split < 1) return SRA_ERR_INVALID_ARG;
  const size_t rows = size_t(n_split) * a->batch * a->heads * a->n_gen;
  *bytes = int64_t(kItemBytes + align256(rows * 4) + rows * a->head_dim * 4);
  return SRA_OK;
}

int sra_forward_gen_static(const sra_static_fwd_args* a, void* cuda_stream) {
  t_err[0] = 0;
  if (!a) return fail(SRA_ERR_INVALID_ARG, "args is NULL");
  const int B = a->batch, H = a->heads, d = a->head_dim, Ng = a->n_gen, Nr = a->n_ref;
  if (B < 1 || H < 1 || Ng < 1 || Nr < 0) return fail(SRA_ERR_INVALID_ARG, "batch, heads, n_gen >= 1 and n_ref >= 0 required");
  if (d != 64 && d != 128) return fail(SRA_ERR_UNSUPPORTED, "head_dim must be 64 or 128");
  if (!a->q_gen || !a->k_gen || !a->v_gen || !a->o_gen) return fail(SRA_ERR_INVALID_ARG, "q_gen / k_gen / v_gen / o_gen required");
  if (Nr > 0 && (!a->k_ref || !a->v_ref)) return fail(SRA_ERR_INVALID_ARG, "k_ref / v_ref required when n_ref > 0");
  const void* ptrs[] = {a->q_gen, a->k_gen, a->v_gen, a->k_ref, a->v_ref, a->o_gen};
  for (const void* q : ptrs)
    if (q && (reinterpret_cast<uintptr_t>(q) & 15)) return fail(SRA_ERR_INVALID_ARG, "tensor pointers must be 16-byte aligned");
  int dev = a->device;
  if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return fail(SRA_ERR_UNSUPPORTED, "no CUDA device: this library has no CPU path"); }
  sra::DeviceGuard guard(dev);
  DeviceInfo* di = nullptr;
  if (int rc = scratch_of(dev, &di)) return rc;
  if (!di->sm100) return fail(SRA_ERR_UNSUPPORTED, "device is not sm_100 (B200); kernels are sm_100a-only");

  const int n_slabs = (Ng + kQRowsPerCta - 1) / kQRowsPerCta;
  const int tiles = (Ng + kTile - 1) / kTile + (Nr + kTile - 1) / kTile;
  int n_split = a->n_split > 0 ? a->n_split : auto_split(long(n_slabs) * H * B, tiles, di->num_sms);
  if (n_split > tiles || n_split > 64) return fail(SRA_ERR_INVALID_ARG, "n_split %.0f exceeds the key tiles (%.0f) or 64", n_split, tiles);
  if (size_t(n_slabs) * n_split > size_t(kMaxItems))
    return fail(SRA_ERR_INVALID_ARG, "%.0f work items exceed the static maximum of %.0f", double(n_slabs) * n_split, kMaxItems);
  int64_t need = 0;
  sra_static_scratch_bytes(a, n_split, &need);
  if (size_t(need) > kScratchBytes)
    return fail(SRA_ERR_INVALID_ARG, "problem needs %.0f bytes of scratch, the static array holds %.0f (SRA_STATIC_SCRATCH_BYTES): use sra_create / sra_forward",
                double(need), double(kScratchBytes));
  const size_t rows = size_t(n_split) * B * H * Ng;
  const size_t off_lse = kItemBytes, off_o = kItemBytes + align256(rows * 4);
  unsigned char* scratch = static_cast<unsigned char*>(di->scratch);  // the DEVICE address (cudaGetSymbolAddress)
  cudaStream_t st = cudaStream_t(cuda_stream);

  CUtensorMap maps[6];
  int rc;
  if ((rc = sra::make_tmap_bf16(nullptr, &maps[0], a->q_gen, B, Ng, H, d, false, kTile))) return fail(rc, "cuTensorMapEncodeTiled failed");
  if ((rc = sra::make_tmap_bf16(nullptr, &maps[1], a->k_gen, B, Ng, H, d, false, kTile))) return fail(rc, "cuTensorMapEncodeTiled failed");
  if ((rc = sra::make_tmap_bf16(nullptr, &maps[2], a->v_gen, B, Ng, H, d, false, kTile))) return fail(rc, "cuTensorMapEncodeTiled failed");
  maps[3] = maps[0]; maps[4] = maps[1]; maps[5] = maps[2];
  if (Nr > 0) {
    if ((rc = sra::make_tmap_bf16(nullptr, &maps[4], a->k_ref, B, Nr, H, d, false, kTile))) return fail(rc, "cuTensorMapEncodeTiled failed");
    if ((rc = sra::make_tmap_bf16(nullptr, &maps[5], a->v_ref, B, Nr, H, d, false, kTile))) return fail(rc, "cuTensorMapEncodeTiled failed");
  }
  sra::sra_static_items_kernel<<<1, 256, 0, st>>>(Ng, Nr, n_slabs, n_split);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(e, "sra_static_items_kernel launch");

  sra::FwdParams p{};
  p.items = reinterpret_cast<const FwdItem*>(scratch);
  p.n_items = n_slabs * n_split;
  p.item_batch_stride = 0;
  p.heads = H; p.batch = B; p.n_gen = Ng; p.n_ref = Nr;
  p.scale = a->softmax_scale > 0.f ? a->softmax_scale : 1.0f / sqrtf(float(d));
  p.scale_log2 = p.scale * 1.4426950408889634f;
  p.o_gen = static_cast<__nv_bfloat16*>(a->o_gen);
  p.lse_gen = a->lse_gen;
  p.ref_kv_head_major = 0;
  p.part_lse = reinterpret_cast<float*>(scratch + off_lse);
  p.part_o = reinterpret_cast<float*>(scratch + off_o);
  e = d == 128 ? sra::launch_fwd<128, 1>(maps, p, st) : sra::launch_fwd<64, 1>(maps, p, st);
  if (e != cudaSuccess) return fail_cuda(e, "sra_fwd_kernel launch");

  const size_t out_rows = size_t(B) * Ng * H;
  const int threads = 256;
  const int blocks = int(std::min<size_t>((out_rows * 32 + threads - 1) / threads, size_t(di->num_sms) * 16));
  if (d == 128)
    sra::sra_static_merge_kernel<128><<<blocks, threads, 0, st>>>(off_lse, off_o, p.o_gen, p.lse_gen, n_split, B, H, Ng);
  else
    sra::sra_static_merge_kernel<64><<<blocks, threads, 0, st>>>(off_lse, off_o, p.o_gen, p.lse_gen, n_split, B, H, Ng);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(e, "sra_static_merge_kernel launch");
  return SRA_OK;
}

}  // extern "C"
