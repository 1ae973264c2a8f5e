/* sra.h - C ABI of the B200-native Sparse Reference Attention (SRA) library.
 *
 * SRA is the asymmetric self-attention of the VideoRef DiT of arxiv/paper_2606_13872:
 *   "Generation tokens attend to all reference tokens ... while reference tokens only
 *    self-attend"                                              (section 1)
 *   structured sparsity, cost ~linear in reference length      (section 2.1)
 *   reference K/V "computed once at the first denoising step and cached in GPU memory",
 *   then concatenated with fresh generation K/V                (section 4.3)
 *   references enter SFT training through SRA => backward      (section 3.3)
 * The paper prints no equation; the mask reading:
 *   rows/cols ordered [G ; R];  G row i sees every key of G u R;
 *   R row i sees key j  iff  j in R and block(i) == block(j)  (blocks = contiguous ranges
 *   given by ref_block_offsets, one block = one latent frame in the paper-shaped configs).
 *   O = softmax(scale * Q K^T restricted to visible keys) V,  LSE = log sum exp (natural log).
 *
 * Conventions
 *   - extern "C", plain pointers + sizes, no torch types.  Every function returns an int
 *     status (0 = SRA_OK, <0 = error) and never throws / aborts.
 *   - "device" pointers are CUDA device pointers on the ctx's device; "host" pointers are
 *     ordinary host memory.  The caller owns every tensor; the library owns only sra_ctx
 *     (resident reference-KV cache, tile schedule, fp32 backward workspace).  Every entry point
 *     makes the ctx's device current for its own duration and restores the caller's device.
 *   - Memory: sra_create allocates what sra_cache_reference_kv and sra_forward need (cache,
 *     device schedule, key-split workspace).  The optional paths - backward workspace, host
 *     staging of sra_forward_host, compaction buffers of a validity mask - are allocated ONCE,
 *     sized from the config for the largest case, by sra_reserve or at the first call that needs
 *     them; no steady-state call allocates, frees, creates a stream or synchronises the device.
 *   - Tensor layout: bf16, [batch, tokens, heads, head_dim], head_dim contiguous,
 *     16-byte aligned base pointers.  LSE: fp32 [batch, heads, tokens].
 *   - Calls are asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy
 *     default stream).  Argument / launch errors are returned synchronously; execution
 *     faults surface at the caller's next synchronisation.
 *   - Mask isolation holds for non-finite data too.  A query's outputs (and the gradients that depend only on what
 *     that query sees) are unaffected by Inf / NaN in keys, values or queries it must not see: masked scores are
 *     removed by selection (P = 0 exactly), and the ragged last tile of a reference block / of a temporal-window frame
 *     is loaded through a tensor map bounded at the segment's end, so the neighbouring block's or frame's rows are
 *     never fetched (they would meet P = 0 in an MMA: 0 * Inf = NaN).  Rows that DO see a non-finite value are
 *     non-finite, as the definition says (tests/test_gpu_nonfinite.py).
 *   - One ctx is used from one thread at a time.  No CPU fallback exists: on a device that
 *     is not sm_100 every compute entry point returns SRA_ERR_UNSUPPORTED.
 */
#ifndef SRA_H_
#define SRA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SRA_OK 0
#define SRA_ERR_INVALID_ARG (-1)  /* NULL where required, bad sizes, bad offsets            */
#define SRA_ERR_UNSUPPORTED (-2)  /* head_dim not in {64,128}; device is not sm_100         */
#define SRA_ERR_CUDA (-3)         /* a CUDA runtime/driver call failed (see sra_last_error) */
#define SRA_ERR_NO_REF_CACHE (-4) /* k_ref/v_ref NULL but sra_cache_reference_kv not called */
#define SRA_ERR_OOM (-5)          /* device or host allocation failed                       */

typedef struct sra_ctx sra_ctx;

/* Problem statement (shapes from BASELINE.json configs). */
typedef struct {
  int32_t batch;                    /* B >= 1                                                       */
  int32_t heads;                    /* H >= 1 (plain multi-head; the paper is silent on GQA)        */
  int32_t head_dim;                 /* d in {64, 128}                                               */
  int32_t n_gen;                    /* generation tokens per batch item (frames x tokens/frame) >=1 */
  int32_t n_ref;                    /* reference tokens per batch item; 0 => plain self-attention   */
  int32_t n_ref_blocks;             /* 0 iff n_ref == 0                                             */
  const int32_t* ref_block_offsets; /* HOST, n_ref_blocks+1 ints: [0]=0, strictly increasing,       */
                                    /* last = n_ref.  Copied at create.  NULL iff n_ref_blocks == 0 */
  float softmax_scale;              /* <= 0 => 1/sqrt(head_dim)                                     */
  int32_t device;                   /* CUDA ordinal, -1 = current device                            */
} sra_config;

/* Creates a context: validates the config, copies the block pattern, builds the tile
 * schedule (work items never enumerate a masked tile) and allocates, on
 * cfg->device, the resident reference-KV cache (2 * B*n_ref*H*d bf16), the device copies of the
 * schedule and - for short-query shapes - the key-split workspace.  The caller's current device
 * is left unchanged.  *out is set to NULL on failure (SRA_ERR_OOM if the device allocations fail).
 * Without a usable sm_100 device the context is host-only (schedule queries work, every compute
 * entry point returns SRA_ERR_UNSUPPORTED). */
int sra_create(const sra_config* cfg, sra_ctx** out);

/* One-time allocation of the optional paths, so that no later call allocates (each bit is also
 * reserved implicitly by the first call that needs it; reserving twice is a no-op):
 *   SRA_RESERVE_BACKWARD  fp32 workspace of sra_backward: dQ accumulators B*H*n_pad*d, D and LSE*log2e
 *                         B*H*n_pad each, n_pad = (n_gen + n_ref) rounded up to 64
 *   SRA_RESERVE_HOST      sra_forward_host: device staging of q/k/v/o (gen), q/o (ref) and both LSE,
 *                         two copy streams, events, the fp32 partials of its reference-first phase; measures the
 *                         host->device copy bandwidth once (64 MB probe) to size that phase
 *   SRA_RESERVE_VALIDITY  sra_set_reference_validity[_batched]: compacted Q_r/K_r/V_r/O_r/LSE_r (n_ref rows
 *                         capacity) and the index arrays; with SRA_RESERVE_BACKWARD also dO_r/dQ_r/dK_r/dV_r
 * Returns SRA_ERR_OOM if an allocation fails (nothing of that bit is kept), SRA_ERR_UNSUPPORTED
 * without an sm_100 device. */
#define SRA_RESERVE_BACKWARD 1u
#define SRA_RESERVE_HOST 2u
#define SRA_RESERVE_VALIDITY 4u
int sra_reserve(sra_ctx* ctx, uint32_t what);

/* "reference KV tensors ... computed once at the first denoising step and
 * cached in GPU memory".  k_ref / v_ref: DEVICE bf16 [B, n_ref, H, d] (post-projection,
 * post-RoPE).  They are COPIED (re-laid head-major [B, H, n_ref, d]) into ctx-owned HBM by a
 * CUDA kernel on `cuda_stream`; the cache stays valid until the next call or sra_destroy and
 * is read by every later sra_forward whose k_ref/v_ref are NULL.  n_ref == 0 => no-op. */
int sra_cache_reference_kv(sra_ctx* ctx, const void* k_ref, const void* v_ref, void* cuda_stream);

/* Fused producer of the cache (PAPER.md:223 - caching "eliminat[es] redundant linear projections and RoPE computations
 * across all steps").  Same as sra_cache_reference_kv, but k_ref is the PRE-RoPE key projection and
 * the rotation is applied inside the kernel that writes the resident head-major layout, so the rotated keys never
 * make a round trip through HBM.  Reading A18 (the paper gives no formula): RoFormer rotation on
 * interleaved pairs, (y[2i] + j y[2i+1]) = (x[2i] + j x[2i+1]) (cos[t,i] + j sin[t,i]), fp32 arithmetic, result
 * rounded to bf16 (nearest even); the same table for every head and batch entry.
 * cos_ref / sin_ref: DEVICE fp32 [n_ref, d/2], row t = ORIGINAL reference token t (also when a validity mask compacts
 * the cache).  v_ref is copied unrotated.  Both tables must be non-NULL (SRA_ERR_INVALID_ARG). */
int sra_cache_reference_kv_rope(sra_ctx* ctx, const void* k_ref, const void* v_ref, const float* cos_ref,
                                const float* sin_ref, void* cuda_stream);

/* The per-step side of the same operation: rotates, IN PLACE, one or two DEVICE bf16 tensors [B, n_tokens, H, d]
 * (typically the fresh Q_g and K_g of a denoising step, or Q_r / K_r in training) by the table cos / sin
 * (DEVICE fp32 [n_tokens, d/2]) with the arithmetic stated above.  x1 may be NULL.  One launch, 16 bytes per thread,
 * HBM-bound: 2 * bytes(x0, x1) + the table.  n_tokens <= 0 => no-op. */
int sra_apply_rope(sra_ctx* ctx, void* x0, void* x1, const float* cos, const float* sin, int32_t n_tokens,
                   void* cuda_stream);

typedef struct {
  const void* q_gen; /* DEVICE bf16 [B, n_gen, H, d]                                              */
  const void* k_gen; /* DEVICE bf16 [B, n_gen, H, d]                                              */
  const void* v_gen; /* DEVICE bf16 [B, n_gen, H, d]                                              */
  const void* q_ref; /* DEVICE bf16 [B, n_ref, H, d]; NULL => cached denoising step: R rows are   */
                     /* skipped entirely                                           */
  const void* k_ref; /* DEVICE bf16 [B, n_ref, H, d]; NULL => use the resident cache              */
  const void* v_ref; /* (both NULL or both non-NULL; non-NULL = training, nothing cached)         */
  void* o_gen;       /* out DEVICE bf16 [B, n_gen, H, d], fully overwritten                       */
  void* o_ref;       /* out DEVICE bf16 [B, n_ref, H, d]; required iff q_ref != NULL              */
  float* lse_gen;    /* out DEVICE fp32 [B, H, n_gen], natural log of the scaled scores; nullable */
  float* lse_ref;    /* out DEVICE fp32 [B, H, n_ref]; nullable                                   */
} sra_fwd_args;

/* SRA forward: O_g = softmax(s Q_g [K_g;K_r]^T)[V_g;V_r] and, per
 * reference block j, O_r[j] = softmax(s Q_r[j] K_r[j]^T) V_r[j].  bf16 in/out, fp32
 * accumulation and softmax.  One kernel launch. */
int sra_forward(sra_ctx* ctx, const sra_fwd_args* args, void* cuda_stream);


typedef struct {
  const void* q_gen; /* HOST bf16 [B, n_gen, H, d] (pinned memory recommended: the copies are async) */
  const void* k_gen; /* HOST bf16 [B, n_gen, H, d]                                                 */
  const void* v_gen; /* HOST bf16 [B, n_gen, H, d]                                                 */
  const void* q_ref; /* HOST bf16 [B, n_ref, H, d] or NULL (cached denoising step)                 */
  void* o_gen;       /* out HOST bf16 [B, n_gen, H, d]                                             */
  void* o_ref;       /* out HOST bf16 [B, n_ref, H, d]; required iff q_ref != NULL                 */
  float* lse_gen;    /* out HOST fp32 [B, H, n_gen]; nullable                                      */
  float* lse_ref;    /* out HOST fp32 [B, H, n_ref]; nullable                                      */
} sra_fwd_host_args;

/* End-to-end form of one denoising step (fresh generation Q/K/V arrive each step,
 * the reference K/V come from the resident cache): every pointer is a HOST pointer.  Enqueues on
 * `cuda_stream` the host->device copies of q/k/v into ctx-owned staging buffers (allocated on first
 * use, freed by sra_destroy), the same forward kernel as sra_forward, and the device->host copies of
 * the outputs.  The results are valid after the caller synchronises the stream.  Requires the
 * resident cache when n_ref > 0 (SRA_ERR_NO_REF_CACHE otherwise).
 * With batch == 1 and at least 16 query slabs the step is pipelined: the generation rows go in 8 slabs whose
 * host->device and device->host copies run on two ctx-owned copy streams underneath the forward launches of other
 * slabs (query slabs are independent work items; launches cover several slabs where the copies allow), reference
 * rows before the last slab.  The one
 * transfer every generation row needs, K_g and V_g, is hidden by "reference keys first": the first slabs (up to 6,
 * enough to cover the upload) attend the resident reference K/V while K_g / V_g are in flight, then the generation
 * keys, and the two fp32 partials (O_s, LSE_s) of each row are merged exactly as in the key-split schedule - so
 * those rows can differ from sra_forward's single-pass result in the last bf16 bit (same tolerance against the
 * oracle; the other slabs and the reference rows are bit-identical).  Copy-bound shapes (the reference-segment work
 * of six slab groups is shorter than the K_g / V_g upload, by the two measured rates; no temporal window) stream the
 * generation keys as well: K_g / V_g go up in two key halves, the first slabs attend each half as soon as it has
 * landed, three partials per row.  Needs 3 * B * H * n_gen * (d + 1) * 4 bytes of ctx-owned partial buffers.  The copy streams are ordered after prior work on `cuda_stream`, and `cuda_stream`
 * waits for the last device->host copy, so the call is still asynchronous on - and ordered by - the caller's stream.
 * The same pipeline runs with batch > 1 (a slab is the same row range of every batch item, copied with one strided
 * copy), under a validity mask (the reference rows are gathered from / scattered into the staged tensors) and under
 * a temporal window; with per-sample masks the reference-first phase is skipped.  Only shapes with fewer than 16
 * query slabs (the short-query regime, a sub-millisecond launch) copy serially.  The number of reference-first
 * slabs follows two measured rates: the host->device bandwidth (SRA_RESERVE_HOST) and the forward rate of the
 * previous call on this ctx.  Staging, streams and events: see sra_reserve(SRA_RESERVE_HOST). */
int sra_forward_host(sra_ctx* ctx, const sra_fwd_host_args* args, void* cuda_stream);

typedef struct {
  /* forward inputs, all required (training: nothing comes from the cache unless k_ref NULL) */
  const void *q_gen, *k_gen, *v_gen; /* DEVICE bf16 [B, n_gen, H, d]                              */
  const void *q_ref, *k_ref, *v_ref; /* DEVICE bf16 [B, n_ref, H, d]; q_ref NULL iff n_ref == 0;  */
                                     /* k_ref/v_ref NULL => resident cache                        */
  /* forward results */
  const void *o_gen, *o_ref;         /* DEVICE bf16, as written by sra_forward                    */
  const float *lse_gen, *lse_ref;    /* DEVICE fp32 [B, H, n], as written by sra_forward          */
  /* upstream gradients */
  const void *do_gen, *do_ref;       /* DEVICE bf16 [B, n, H, d]                                  */
  /* outputs, bf16, same shapes as the corresponding inputs, fully overwritten */
  void *dq_gen, *dk_gen, *dv_gen;
  void *dq_ref, *dk_ref, *dv_ref;
} sra_bwd_args;

/* SRA backward (standard softmax-attention calculus under the same
 * mask): D = rowsum(dO o O); P = exp(sQK^T - LSE); dV = P^T dO; dP = dO V^T;
 * dS = P o (dP - D); dQ = s dS K; dK = s dS^T Q.  dK_r/dV_r receive contributions from all G
 * rows and from the R rows of the same block.  head_dim 64 and 128.  dQ is accumulated in a ctx-owned fp32 workspace
 * with fp32 reductions in L2 (cp.reduce.async.bulk; the order of the additions is not fixed: results can differ in
 * the last bit between runs). */
int sra_backward(sra_ctx* ctx, const sra_bwd_args* args, void* cuda_stream);

/* Frees the cache, workspace and schedule.  NULL-safe. */
void sra_destroy(sra_ctx* ctx);

/* Useful (unmasked) FLOPs of one call: 4*d*pairs*H*B forward, 2.5x that backward, with
 * pairs = n_gen*(n_gen+n_ref) + (include_ref_rows ? sum_j b_j^2 : 0). */
int sra_useful_flops(const sra_ctx* ctx, int include_ref_rows, int backward, double* out);

/* Number of work items (CTAs) per (batch, head) the forward schedule enumerates for
 * generation rows / reference rows, and the total key tiles they visit (for tests of a2). */
int sra_schedule_info(const sra_ctx* ctx, int32_t* n_gen_items, int32_t* n_ref_items,
                      int64_t* key_tiles_gen, int64_t* key_tiles_ref);

/* Copies the forward schedule to HOST memory: up to `capacity` items of 8 int32 each
 * {q_is_ref, q_row0, q_rows, seg0_is_ref, seg0_start, seg0_len, seg1_start, seg1_len}
 * (seg1 is always the reference segment of a G item; len 0 = absent).  Returns the item
 * count in *n_items.  Pure host logic - usable without a GPU. */
int sra_schedule_copy(const sra_ctx* ctx, int32_t* items, int32_t capacity, int32_t* n_items);

/* Sparse temporal attention of the super-resolution refiner ("sparse temporal attention that restricts
 * each frame's receptive field to a local neighborhood").  The paper gives no window size and no
 * mask; the reading taken (A17): generation tokens are grouped in frames by `gen_frame_offsets` (HOST,
 * n_frames + 1 ints from 0 to n_gen, strictly increasing); a generation query of frame f sees the generation keys
 * of frames [f - window, f + window] (clipped) and - the refiner keeps the video reference conditioning - every
 * reference key; reference rows are unchanged.  window < 0 turns it off (gen_frame_offsets may then be NULL);
 * window >= n_frames - 1 is plain SRA.  The schedule is rebuilt: forward slabs and backward key tiles never straddle
 * a frame and masked tiles are never enumerated, so cost is linear in the window.  Forward and backward are
 * supported; the key-split short-query schedule is not combined with a window.  Host work only: the new schedule is
 * uploaded by the next launching call, on that call's stream (into the second of two device buffers, so kernels
 * already in flight keep the schedule they were launched with); calls issued on OTHER streams must be ordered after
 * that call by the caller.  Allocates only if the new schedule has more work items than any before it. */
int sra_set_temporal_window(sra_ctx* ctx, int32_t n_frames, const int32_t* gen_frame_offsets, int32_t window);

/* Sparse validity masking of reference tokens ("skip invalid reference tokens"; SURVEY.md 8f #1,
 * reading A8).  `valid`: HOST, n_ref bytes, non-zero = valid; NULL = every token valid again.  One mask per
 * context, shared by all batch items like the block pattern.  An invalid reference token is never a key (for
 * generation rows or for the reference rows of its block); as a query its output row is 0 and its LSE is -inf;
 * its gradient rows are 0.  The library compacts: the schedule, the resident cache, the workspaces and the
 * kernels only ever see the valid tokens (blocks shrink, empty blocks vanish), so invalid tokens cost nothing;
 * caller tensors keep their [B, n_ref, H, d] shape and are gathered / scattered by row.  Invalidates the
 * resident cache (call sra_cache_reference_kv again).  Host work only, like sra_set_temporal_window: the schedule and
 * the index arrays are uploaded by the next launching call on its stream.  Usable without a GPU (host schedule
 * only). */
int sra_set_reference_validity(sra_ctx* ctx, const uint8_t* valid);

/* Per-sample validity / variable reference length ("validity masks are precomputed per-rank"; reading
 * A12): `valid` = HOST, n_masks * n_ref bytes, n_masks = 1 (the call above) or n_masks = batch (row b = the mask of
 * batch item b).  Every batch item is the problem of sra_set_reference_validity under its own mask: it gets its own
 * compaction and its own work-item list (the lists of all items are stacked with a common stride and padded with
 * empty items, which the kernels skip at once), so a batch whose references have different lengths pays for its
 * valid tokens only.  Compacted tensors and the cache have max_b(valid_b) rows per item; the rows behind an item's
 * last valid token are zero.  The key-split short-query schedule is not combined with per-sample masks.
 * SRA_ERR_INVALID_ARG if n_masks is neither 1 nor batch. */
int sra_set_reference_validity_batched(sra_ctx* ctx, const uint8_t* valid, int32_t n_masks);

/* The forward schedule of ONE batch item (same 8-int32 layout as sra_schedule_copy; differs between items only under
 * per-sample masks).  Pure host logic. */
int sra_batch_schedule_copy(const sra_ctx* ctx, int32_t batch_item, int32_t* items, int32_t capacity, int32_t* n_items);

/* CTA-pair launch list (head_dim 128 without a key split: *use_pairs = 1): the items sra_fwd_kernel<128, 2> is
 * launched with - consecutive slabs of sra_schedule_copy that see the same keys merged into one item of up to 512
 * rows, run by a cluster of two CTAs that share every K/V tile (same 8-int32 layout).  Pure host logic. */
int sra_pair_schedule_copy(const sra_ctx* ctx, int32_t* use_pairs, int32_t* items, int32_t capacity, int32_t* n_items);

/* The segment ends that fall INSIDE a tensor (PAPER.md:85 reference blocks, PAPER.md:143 frames of a temporal window):
 * the kernels load the ragged last tile of such a segment through a tensor map bounded at its end, so the rows of the
 * neighbouring block / frame are never fetched (mask isolation for non-finite data, see the contract above).
 * ends (HOST, capacity int32, may be NULL to query the count): [*n_gen_ends generation-row ends | n_masks x
 * *ref_stride reference-row ends of each mask's compacted reference, ascending, padded with INT32_MAX]; *n_ends = the
 * total count.  Pure host logic. */
int sra_bound_ends_copy(const sra_ctx* ctx, int32_t* ends, int32_t capacity, int32_t* n_gen_ends, int32_t* ref_stride,
                        int32_t* n_ends);

/* Short-query schedules (north_star "cache-bound short-query cases"): when a context has fewer generation
 * slabs than about two per SM, sra_create cuts every generation slab into *n_split key ranges of whole
 * 128-key tiles; each range runs as its own CTA, writes an fp32 partial (O_s, LSE_s) into a ctx-owned
 * workspace, and a merge kernel combines them (O = sum_s exp(LSE_s - LSE) O_s).  *n_split == 1 means the
 * plain schedule of sra_schedule_copy is launched.  With `items` non-NULL the LAUNCHED list is copied
 * (same 8-int32 layout; q_is_ref bit 0 = reference rows, bits 8.. = split index + 1, 0 for unsplit items):
 * n_gen_items * n_split split slabs, then the reference items.  Pure host logic - usable without a GPU. */
int sra_split_schedule_copy(const sra_ctx* ctx, int32_t* n_split, int32_t* items, int32_t capacity, int32_t* n_items);

/* Bytes of reference K/V resident in the cache: 2 * sum_b valid_b * H * d * 2 (0 before the first cache call and after
 * a validity change until the cache is rebuilt).  The allocation itself is made at sra_create for n_ref rows. */
int64_t sra_cache_bytes(const sra_ctx* ctx);

/* ---- No-allocation entry point (an addition outside SURVEY.md 8; step a3) ------------------------
 * For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it): the
 * generation rows' attention  O_g = softmax(s Q_g [K_g ; K_r]^T) [V_g ; V_r]  (+ LSE_g) with NO context - nothing to
 * create, reserve or destroy.  It is sra_forward's key-split short-query path (fp32 partials per key range, then a
 * merge); ALL of its scratch - work items and partials - lives in one file-scope `static __device__` array of
 * SRA_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.  The call does not
 * allocate, free, copy from the host or synchronise, on any path.
 *   - Tensors: DEVICE bf16 [batch, tokens, heads, head_dim] as for sra_forward; k_ref / v_ref are the caller's
 *     (token-major) reference K / V - there is no resident cache without a context; NULL iff n_ref == 0.  Reference
 *     ROWS are not computed (a cached denoising step).  lse_gen: DEVICE fp32 [batch, heads, n_gen] or NULL.
 *   - n_split: key ranges per 256-row query slab, 0 = chosen to fill the GPU's SMs.
 *   - Limit: 64 KiB + n_split * batch * heads * n_gen * (head_dim + 1) * 4 bytes (sra_static_scratch_bytes) must fit in
 *     SRA_STATIC_SCRATCH_BYTES, and n_split * ceil(n_gen / 256) <= 2048; beyond that SRA_ERR_INVALID_ARG with the two
 *     figures in sra_static_last_error() - use sra_create / sra_forward, whose workspaces are sized from the config.
 *   - The array is SHARED by every call and keeps the last call's contents.  Nothing in it has to start at zero (each
 *     call rewrites every byte it later reads), but calls that overlap on the GPU - two streams, two threads - race on
 *     it: serialise them (one stream, or events).  Asynchronous on `cuda_stream` like every other entry point.
 *   - Errors: status codes as above; the message is per host thread (sra_static_last_error). */
#define SRA_STATIC_SCRATCH_BYTES (32u << 20)
typedef struct {
  int32_t batch, heads, head_dim; /* head_dim in {64, 128}                                                  */
  int32_t n_gen, n_ref;           /* generation rows / keys, reference keys (0 = plain self-attention)      */
  float softmax_scale;            /* <= 0: 1 / sqrt(head_dim)                                               */
  int32_t device;                 /* CUDA ordinal, -1 = current                                             */
  int32_t n_split;                /* 0 = automatic                                                          */
  const void *q_gen, *k_gen, *v_gen;
  const void *k_ref, *v_ref;
  void* o_gen;
  float* lse_gen;
} sra_static_fwd_args;
int sra_forward_gen_static(const sra_static_fwd_args* args, void* cuda_stream);
/* Bytes of the static array a problem needs with `n_split` key ranges (pure host arithmetic). */
int sra_static_scratch_bytes(const sra_static_fwd_args* args, int32_t n_split, int64_t* bytes);
const char* sra_static_last_error(void);

/* Optional per-kernel device timing (bench.py's roofline leg): when enabled, every launch is bracketed by
 * CUDA events recorded on the launching stream.  sra_kernel_time_ms returns the duration of the LAST launch
 * of kernel `which` (it synchronises on that launch's end event); SRA_ERR_INVALID_ARG if timing is off or the
 * kernel has not been launched since it was switched on. */
#define SRA_KERNEL_CACHE_RELAYOUT 0 /* a1 */
#define SRA_KERNEL_FWD 1            /* a3-a5 */
#define SRA_KERNEL_BWD_PREPROCESS 2 /* a6 */
#define SRA_KERNEL_BWD_MAIN 3       /* a7 */
#define SRA_KERNEL_BWD_DQ_FINALIZE 4 /* a8 */
#define SRA_KERNEL_FWD_MERGE 5       /* a5': merge of key-split partials (short-query schedules only) */
#define SRA_KERNEL_ROPE 6            /* sra_apply_rope (8f #3); the fused cache producer reports as CACHE_RELAYOUT */
#define SRA_NUM_KERNELS 7
int sra_set_kernel_timing(sra_ctx* ctx, int enable);
int sra_kernel_time_ms(sra_ctx* ctx, int which, float* ms);

/* Kernels launched by this ctx since creation (bench.py's gpu_launches). */
int64_t sra_launch_count(const sra_ctx* ctx);

const char* sra_status_string(int status);
const char* sra_last_error(const sra_ctx* ctx); /* "" if none; valid until the next call on ctx */

#ifdef __cplusplus
}
#endif
#endif /* SRA_H_ */
