/*
 * kv_pool.h — C-ABI of the D-instance (consumer) KV data path for sm_100a (B200).
 *
 * What this library is.  DOPD (arxiv 2511.20982) models PD-disaggregated serving as a
 * producer/consumer pair: "P-instances produce prefill-completed requests (together with
 * KV-cache), and D-instances consume those prefill-completed requests to perform token
 * generation" (§IV-B-1).  The consumer keeps each request's KV in "KV-cache
 * blocks" (§V-C), re-reads all of it from HBM on every decode step
 * (§IV-B-2: "the entire decoding inference latency ... is dedicated to
 * reading the KV-cache and model weights") and evaluates softmax(QK^T)V (PAPER.md:146,
 * Eq. 1) for the one new query token of every in-flight request.  The calls below are
 * that path and nothing else:
 *
 *   kv_pool_create          paged KV block pool + host block allocator
 *   kv_ingest               prefill-completed request's contiguous K/V -> paged blocks
 *                           (a2); with n_tokens = 1 it is the decode-step append (a3)
 *   paged_decode_attention  split-KV paged attention (a4) + log-sum-exp combine (a5)
 *   kv_free                 completed request's blocks back to the free list (a6)
 *
 * Conventions.
 *   - extern "C"; every entry point returns an int32_t status (KV_OK = 0, errors < 0)
 *     unless stated otherwise.  No exceptions, no aborts, nothing is printed.
 *   - "device" pointers are CUDA device pointers valid in the current context; "host"
 *     pointers are ordinary process memory.  The CALLER owns all device memory (slab, q,
 *     out, sources) and the stream; the library owns only its host metadata and pinned
 *     staging buffers.  Device pointers must be 16-byte aligned.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All
 *     GPU work of a call is enqueued on it and the call returns without synchronising;
 *     source buffers may be released once the stream has passed the call.
 *   - bf16 = IEEE bfloat16 bit patterns (uint16_t).  Sources, queries and outputs are always bf16;
 *     the pool is bf16 or, with kv_dtype = KV_DTYPE_FP8_E4M3, e4m3 codes + scales (see below).
 *   - One host thread per pool.  Pools are independent.
 *   - One attention stream per pool at a time: paged_decode_attention / paged_decode_step(_layers) /
 *     paged_varlen_attention launches of ONE pool share a device workspace (work and arrival counters,
 *     split-KV partials, the staged plan), so they must execute one after the other.  Calls on one stream
 *     do; when a call arrives on a different stream than the pool's previous attention launch the library
 *     orders it behind that launch itself (cudaStreamWaitEvent), so the result is still correct but the two
 *     do not overlap.  kv_ingest / kv_transfer / kv_gather have no such workspace and may run on any stream.
 *   - A pool belongs to the device its slab is on; calls made while another device is current switch to the
 *     pool's device for their duration.
 *
 * Slab layout (caller-visible so that an independent checker can read the pool).
 *   The caller allocates `kv_pool_required_bytes(cfg)` bytes at `device_base`.  The first
 *   `kv_pool_kv_bytes(cfg)` bytes are the KV region, bf16, indexed as
 *
 *       kv[layer][block][kv_head][c][slot][j]      c = 0: K, c = 1: V
 *         layer   in [0, num_layers)      block in [0, num_blocks)
 *         kv_head in [0, num_kv_heads)    slot  in [0, block_size)    j in [0, head_dim)
 *
 *   i.e. element offset ((((layer*num_blocks + block)*num_kv_heads + kv_head)*2 + c)
 *   *block_size + slot)*head_dim + j.  Token t of a request lives in block
 *   block_table[t / block_size] at slot t % block_size.  Bytes after the KV region are
 *   library-private metadata (device block_table mirror, work lists, split-KV partials).
 *   Slots at or beyond a request's length and blocks that are not allocated are never
 *   written by the library and never influence any output.
 */
#ifndef KV_POOL_H_
#define KV_POOL_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes -------------------------------------------------------------------- */
#define KV_OK                      0
#define KV_ERR_INVALID            -1  /* null / misaligned pointer, bad shape, bad argument  */
#define KV_ERR_NO_BLOCKS          -2  /* pool exhausted; the call changed nothing (atomic)   */
#define KV_ERR_UNKNOWN_REQUEST    -3  /* req_id not live                                     */
#define KV_ERR_TOO_LONG           -4  /* request would exceed max_blocks_per_request         */
#define KV_ERR_TOO_MANY_REQUESTS  -5  /* more than max_requests live requests                */
#define KV_ERR_CUDA               -6  /* a CUDA runtime call failed; see kv_last_cuda_error  */
#define KV_ERR_NO_DEVICE          -7  /* pool was created without a device slab (host-only)  */
#define KV_ERR_UNSUPPORTED        -8  /* call not available for this pool's kv_dtype         */
#define KV_ERR_SCRATCH_LIMIT      -9  /* paged_decode_attention_static: the plan needs more split-KV
                                         partial slots than KV_STATIC_MAX_PARTIALS; nothing changed */

/* ---- KV element types ---------------------------------------------------------------- */
#define KV_DTYPE_BF16              0  /* bf16 pool (the BASELINE.json configs)               */
#define KV_DTYPE_FP8_E4M3          1  /* NEXT-2: e4m3 codes + per-token fp32 scales          */

typedef struct kv_pool kv_pool_t; /* opaque, library-owned host object */

/*
 * Pool geometry.  Supported: head_dim in {64, 128}; block_size = 16;
 * num_q_heads % num_kv_heads == 0 with group size G = num_q_heads / num_kv_heads <= 8
 * (GQA mapping: query head h reads KV head h / G).
 */
typedef struct kv_pool_config {
  int32_t  num_layers;
  int32_t  num_q_heads;
  int32_t  num_kv_heads;
  int32_t  head_dim;
  int32_t  block_size;
  int64_t  num_blocks;              /* physical blocks per layer                            */
  int32_t  max_requests;            /* live requests (rows of the device block_table)       */
  int32_t  max_blocks_per_request;  /* columns of the device block_table                    */
  uint64_t alloc_seed;              /* 0: free list hands out 0,1,2,... (LIFO on reuse);
                                       !=0: initial free list is a Fisher-Yates permutation
                                       driven by splitmix64(alloc_seed) — fragmented pool   */
  void*    device_base;             /* device, >= kv_pool_required_bytes(cfg), 256-B aligned;
                                       NULL => host-only pool: allocator and planner work,
                                       calls that launch kernels return KV_ERR_NO_DEVICE    */
  int64_t  device_bytes;            /* size of the slab at device_base                      */
  int32_t  kv_dtype;                /* KV_DTYPE_BF16 (0) or KV_DTYPE_FP8_E4M3                */
} kv_pool_config_t;

/*
 * NEXT-2 — FP8 pool (kv_dtype = KV_DTYPE_FP8_E4M3).  The paper's models are FP8 and
 * M_token, the KV bytes per token, is the denominator of Eq. 13: an FP8 pool holds and
 * streams about twice the tokens per byte (cc_d x 1.94 at head_dim 128).  The paper fixes no KV
 * quantisation; the one used (C1-C4), per token row x[0..head_dim) of one
 * (layer, kv head, K|V), with every rounding in fp32:
 *     amax = max_j |x_j|;  scale = amax / 448;  inv = 448 / amax   (scale = inv = 1 if amax = 0)
 *     code_j = e4m3_rne_saturating(x_j * inv);        dequantised x^_j = e4m3(code_j) * scale
 * (e4m3 = OCP FP8 E4M3 "fn": 1-4-3 bits, bias 7, no infinities, max 448).  Sources and queries stay
 * bf16; kv_ingest quantises on the way in; paged_decode_attention evaluates Eq. 1 on the dequantised
 * values.  KV region layout, one tile of 32*head_dim + 128 bytes per (layer, block, kv_head), tiles
 * ordered [layer][block][kv_head]:
 *     K8[16][head_dim] codes | V8[16][head_dim] codes | sc[16][2] fp32 = (k scale, v scale) of slot t
 * Available on an FP8 pool: kv_reserve, kv_ingest(_host), paged_decode_attention(_host),
 * paged_decode_step(_host) (the fused append quantises the new row exactly as kv_ingest does: same
 * bytes), paged_varlen_attention, kv_free, kv_transfer (FP8 -> FP8), kv_gather (codes + scales, see there)
 * and the introspection / profiling calls.
 */

/* Bytes of the KV region / of the whole slab (KV region + private metadata) for `cfg`
 * (device_base / device_bytes ignored).  Return < 0 (a KV_ERR_*) on an invalid config.    */
int64_t kv_pool_kv_bytes(const kv_pool_config_t* cfg);
int64_t kv_pool_required_bytes(const kv_pool_config_t* cfg);

/* Create / destroy.  Create validates cfg, builds the free list, allocates pinned staging
 * (skipped for a host-only pool) and does NOT touch the KV region (prior bytes retained).
 * Destroy synchronises nothing: the caller must have drained streams using the pool.       */
int32_t kv_pool_create(const kv_pool_config_t* cfg, kv_pool_t** out_pool);
int32_t kv_pool_destroy(kv_pool_t* pool);

/*
 * a1 — block allocation + block_table build, host only ("KV-cache blocks";
 * PAPER.md:82 "block fragmentation and count").  Grows each request from len to
 * len + n_tokens[i] tokens: takes ceil((len+n)/bs) - ceil(len/bs) block ids from the free
 * list and appends them to the request's block list.  Unknown req_id => created with
 * length 0.  Atomic over the batch: on any error nothing changes.  Duplicate ids in one
 * call => KV_ERR_INVALID.  n_tokens[i] = 0 is allowed (creates an empty request).
 * kv_ingest calls this internally; it is exported for host-side planning and tests.
 */
int32_t kv_reserve(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids /*host*/,
                   const int32_t* n_tokens /*host*/);

/*
 * a2 / a3 — KV ingest ("prefill-completed requests (together with KV-cache)";
 * PAPER.md:360 transfer into the consumer's KV-cache blocks; PAPER.md:219 decode steps).
 * For request i, layers [layer_begin, layer_begin + layer_count):
 *     kv[l][block_table_i[(p+t)/bs]][h][c][(p+t)%bs][:] = src_c[i][l-layer_begin][h][t][:]
 * for t in [0, n_tokens[i]), where p is the request's length before the reservation.
 *   k_src[i], v_src[i]: device, bf16, contiguous [layer_count][num_kv_heads][n_tokens[i]][head_dim].
 *   layer_begin == 0 : performs kv_reserve(n_tokens) first (p = current length), then copies.
 *   layer_begin  > 0 : layer-sliced continuation: copies into the LAST reservation of each
 *                      request (p = length - n_tokens[i]); n_tokens[i] must equal that
 *                      reservation's size, else KV_ERR_INVALID.  This lets a producer stream
 *                      KV layer by layer, and a decode loop append per layer.
 * A pure bit copy: no arithmetic, no conversion.  Bytes outside the written slots keep
 * their previous contents.  Errors as kv_reserve, plus KV_ERR_NO_DEVICE / KV_ERR_CUDA.
 * Atomic: if the call fails for any reason — including a CUDA error while enqueuing — the
 * reservation it made is rolled back and no request is modified.
 */
int32_t kv_ingest(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids /*host*/,
                  const int32_t* n_tokens /*host*/,
                  const void* const* k_src /*host array of device ptrs*/,
                  const void* const* v_src /*host array of device ptrs*/,
                  int32_t layer_begin, int32_t layer_count, void* cuda_stream);

/*
 * a4 + a5 — one decode step's attention for one layer (Eq. 1 restricted to
 * the decode case of PAPER.md:200/:219: one query token per request over that request's
 * stored KV, all n tokens visible, no mask; scale reading SURVEY §8(c) A1):
 *     out[i][h][:] = sum_t softmax_t( sm_scale * <q[i][h], K_t> ) * V_t ,
 *     K_t, V_t = token t of request req_ids[i], KV head h / G, layer `layer`, t < len_i.
 *   q, out: device, bf16, [batch][num_q_heads][head_dim]; out is written RNE-rounded from
 *   fp32 accumulation.  sm_scale <= 0 selects 1/sqrt(head_dim).
 * One launch on `cuda_stream`: a split-KV kernel (per (request, kv_head, chunk) online softmax -> partial
 * (m, l, O)) whose last-arriving chunk merges the partials (LSE combine); with option fuse_combine = 0 the
 * merge is a second launch.
 * Errors: KV_ERR_UNKNOWN_REQUEST; a request of length 0 or a duplicate id => KV_ERR_INVALID;
 * batch > max_requests => KV_ERR_INVALID; KV_ERR_NO_DEVICE; KV_ERR_CUDA.
 */
int32_t paged_decode_attention(kv_pool_t* pool, int32_t layer, int32_t batch,
                               const int64_t* req_ids /*host*/, const void* q /*device*/,
                               void* out /*device*/, float sm_scale, void* cuda_stream);

/*
 * a3 + a4 + a5 fused — one launch per layer and decode step.  Same result as
 *     kv_ingest(n_tokens = 1 per request, layer_begin = layer, layer_count = 1)   then
 *     paged_decode_attention(layer)
 * but the new token's K/V row is appended by the attention kernel itself: the work unit that
 * owns a request's last block reads that row from k_new / v_new, uses it, and writes it into
 * the pool (every decode iteration adds one token to each in-flight request and
 * re-reads its KV).  Protocol per decode step:
 *     kv_reserve(pool, batch, req_ids, ones)           once, host only (a1)
 *     for layer in 0 .. num_layers-1:
 *         paged_decode_step(pool, layer, batch, req_ids, q, k_new, v_new, out, ...)
 *   k_new, v_new: device, bf16, [batch][num_kv_heads][head_dim] — row i belongs to req_ids[i]
 *   and lands at that request's last position (length - 1).
 * Errors: as paged_decode_attention; additionally KV_ERR_INVALID unless every request's last
 * reservation is exactly one token (no reservation since, no multi-token reservation).
 * Calling it twice for the same layer and step rewrites the same row (idempotent).
 */
int32_t paged_decode_step(kv_pool_t* pool, int32_t layer, int32_t batch,
                          const int64_t* req_ids /*host*/, const void* q /*device*/,
                          const void* k_new /*device*/, const void* v_new /*device*/,
                          void* out /*device*/, float sm_scale, void* cuda_stream);

/*
 * One decode step's attention for layers [layer_begin, layer_begin + layer_count) in ONE host call
 * (PAPER.md:204 names the "CUDA graph inference configuration" as the deployed form of the decode step:
 * the step is enqueued as a unit, not layer by layer from the host).  Equivalent to
 *     if (flags & KV_STEP_RESERVE) kv_reserve(pool, batch, req_ids, ones);          (layer_begin must be 0)
 *     for l in layer_begin .. layer_begin + layer_count - 1:
 *         k_new ? paged_decode_step(pool, l, batch, req_ids, q_l, k_new_l, v_new_l, out_l, sm_scale, stream)
 *               : paged_decode_attention(pool, l, batch, req_ids, q_l, out_l, sm_scale, stream)
 * with q_l = q + (l - layer_begin) * q_layer_stride_bytes (out_l likewise) and k_new_l = k_new +
 * (l - layer_begin) * kv_layer_stride_bytes (v_new_l likewise); strides in bytes, multiples of 16.
 * One plan, one upload; the layer launches are issued back to back with the programmatic-dependent-launch
 * attribute (option "pdl", default 1), so the CTAs of layer l+1 take over SMs as layer l drains and their
 * work-item and block-id reads overlap its tail; every read of q, k_new, v_new and every write happens
 * after layer l (and whatever produced q) has completed (griddepcontrol.wait).  It is for callers that hold
 * the queries of several layers at once (bench, replay, a captured graph whose other kernels sit in
 * between); a model that computes q_l from out_(l-1) calls it with layer_count = 1 per layer and still gets
 * the one-plan-per-step and PDL behaviour.  k_new = v_new = NULL selects attention without append.
 * Errors: as paged_decode_step / paged_decode_attention / kv_reserve; KV_STEP_RESERVE with layer_begin != 0 or
 * without k_new => KV_ERR_INVALID.  On error nothing changes (a reservation made by this call is rolled back).
 */
#define KV_STEP_RESERVE 1
int32_t paged_decode_step_layers(kv_pool_t* pool, int32_t layer_begin, int32_t layer_count, int32_t batch,
                                 const int64_t* req_ids /*host*/, const void* q /*device*/,
                                 const void* k_new /*device or NULL*/, const void* v_new /*device or NULL*/,
                                 void* out /*device*/, int64_t q_layer_stride_bytes, int64_t kv_layer_stride_bytes,
                                 float sm_scale, int32_t flags, void* cuda_stream);

/*
 * a4 + a5 for callers that must not allocate — code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc.  Same operation, arguments, result and errors as paged_decode_attention (Eq. 1 in
 * the decode form of PAPER.md:200/:219; same plan, same kernel, same merge), but the split-KV workspace — arrival
 * counters and the (m, l, O) partials — is NOT taken from the pool's slab: it lives in a file-scope
 * `static __device__` array of the library, KV_STATIC_MAX_PARTIALS partial slots at the widest geometry
 * (G = 8, head_dim 128), kv_static_scratch_bytes() = 17 055 744 bytes (16.3 MiB), which every GPU that loads the
 * library holds until the process exits.  The call itself performs no cudaMalloc, no cudaFree and no allocating
 * library routine: it looks the array's device address up once per device (cudaGetSymbolAddress, with the pool's
 * device current), stages the plan through the pinned slots kv_pool_create set up, clears the arrival counters it
 * is going to use (cudaMemsetAsync on `cuda_stream`; the array keeps the last call's contents) and launches.
 *   Limit: a batch whose split-KV plan needs more than KV_STATIC_MAX_PARTIALS partial slots (one per (split request,
 *   kv head, chunk); kv_plan_decode shows the plan) => KV_ERR_SCRATCH_LIMIT, nothing changed.  Larger
 *   "min_chunk_blocks" / smaller "items_per_slot" options shrink the count; paged_decode_attention has no such limit.
 *   Sharing: ALL calls of ALL pools on a device share the one array.  Calls that may overlap on the GPU (different
 *   streams without an ordering between them, or two pools driven from two threads) race on it and return garbage;
 *   the caller orders them.  Calls on one stream are ordered by the stream.  Relative to the pool's other attention
 *   calls the one-attention-stream rule above applies unchanged.
 */
#define KV_STATIC_MAX_PARTIALS 4096
int64_t kv_static_scratch_bytes(void);
int32_t paged_decode_attention_static(kv_pool_t* pool, int32_t layer, int32_t batch,
                                      const int64_t* req_ids /*host*/, const void* q /*device*/,
                                      void* out /*device*/, float sm_scale, void* cuda_stream);

/*
 * NEXT-1 — variable-q-length causal paged attention: in-place prefill of ultra-short requests
 * merged with decoding (§V-E: "For ultra-short requests we employ PD-aggregation:
 * merging their prefill with other requests' decoding on D-instances avoids unnecessary
 * KV-cache transfers"; such requests run "in-place (i.e., without remote
 * prefill)").  One call serves a batch that mixes decode rows (q_lens[i] = 1) and prefill rows
 * (q_lens[i] = number of prompt tokens computed in this step).  Request i's query tokens are
 * its LAST q_lens[i] stored tokens — their K/V must already be in the pool (kv_ingest, possibly
 * layer-sliced) — and query token t of request i, at absolute position P = len_i - q_lens[i] + t,
 * attends stored tokens 0..P inclusive (Eq. 1, with a causal mask; readings
 * DESIGN.md B1-B3):
 *     out[row][h][:] = sum_{s <= P} softmax_s( sm_scale * <q[row][h], K_s> ) * V_s ,
 *     row = sum_{k < i} q_lens[k] + t,   K_s, V_s of KV head h / G, layer `layer`.
 *   q_lens: host int32[batch], 1 <= q_lens[i] <= len_i.
 *   q, out: device, bf16, [sum_i q_lens[i]][num_q_heads][head_dim]; out RNE from fp32.
 * With every q_lens[i] = 1 the result equals paged_decode_attention's.  One launch; split-KV
 * partials are merged inside the kernel.  Errors: KV_ERR_UNKNOWN_REQUEST; q_lens[i] outside
 * [1, len_i] or a duplicate id => KV_ERR_INVALID; more query tiles than the plan staging holds
 * => KV_ERR_TOO_LONG; KV_ERR_NO_DEVICE; KV_ERR_CUDA.  Nothing changes on error.
 */
int32_t paged_varlen_attention(kv_pool_t* pool, int32_t layer, int32_t batch,
                               const int64_t* req_ids /*host*/, const int32_t* q_lens /*host*/,
                               const void* q /*device*/, void* out /*device*/, float sm_scale,
                               void* cuda_stream);

/*
 * NEXT-1, the new tokens' K/V written into the pool as the step goes (§V-E: the ultra-short
 * request's prefill runs in place on the D-instance, so its K/V are produced there, layer by layer, beside the decode
 * rows' one new token each).  One host call per layer, equivalent to
 *     if (flags & KV_STEP_RESERVE) kv_reserve(pool, batch, req_ids, q_lens);              (layer must be 0)
 *     kv_ingest(pool, batch, req_ids, q_lens, k_new, v_new, layer, 1, stream)             as a continuation of that
 *                                                                                          reservation (also for layer 0)
 *     paged_varlen_attention(pool, layer, batch, req_ids, q_lens, q, out, sm_scale, stream)
 *   k_new[i], v_new[i]: device, bf16, contiguous [num_kv_heads][q_lens[i]][head_dim] — THIS layer's K / V of request i's
 *   q_lens[i] new tokens (a decode row: one token; an in-place prefill row: its prompt, or the next chunk of it);
 *   host arrays of `batch` device pointers.  q, out: as paged_varlen_attention.  An FP8 pool quantises the rows exactly
 *   as kv_ingest does.  Two launches on `cuda_stream` (scatter, attention); the attention's plan is made once per step
 *   and reused by the following layers.
 * Without KV_STEP_RESERVE every request's last reservation must be exactly q_lens[i] tokens (kv_reserve by the caller,
 * or this call for layer 0), else KV_ERR_INVALID.  Errors: as kv_reserve / kv_ingest / paged_varlen_attention;
 * q_lens[i] < 1 => KV_ERR_INVALID.  If the call fails before anything is enqueued — allocation, validation, a plan that
 * does not fit — nothing changes (a reservation it made is rolled back).
 */
int32_t paged_varlen_step(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids /*host*/,
                          const int32_t* q_lens /*host*/, const void* q /*device*/,
                          const void* const* k_new /*host array of device ptrs*/,
                          const void* const* v_new /*host array of device ptrs*/, void* out /*device*/,
                          float sm_scale, int32_t flags, void* cuda_stream);

/*
 * a6 — free (a completed request releases consumer capacity).  Host only
 * and immediate: blocks return to the free list (LIFO) and the table row is dropped.  The
 * caller must not ingest into recycled blocks on a different stream before the attention
 * that last read them has finished.  Atomic: an unknown or duplicate id => nothing freed.
 */
int32_t kv_free(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids /*host*/);

/* ---- introspection ------------------------------------------------------------------- */

/* Block list and length of a live request (host).  Writes min(cap, n_blocks) ids.         */
int32_t kv_block_table(const kv_pool_t* pool, int64_t req_id, int32_t* out_blocks /*host*/,
                       int32_t cap, int32_t* out_n_blocks, int32_t* out_len);

/* Occupancy — the `load_kv` signal of PAPER.md:352 / :419.  Any out pointer may be NULL.  */
int32_t kv_pool_stats(const kv_pool_t* pool, int64_t* blocks_total, int64_t* blocks_free,
                      int32_t* live_requests, int64_t* blocks_high_water);

/* Inverse of ingest's relocation for one request, all layers (test support; also the producer-side
 * paged->contiguous step of SURVEY §8(f) NEXT-4).
 *   bf16 pool: k_dst / v_dst device bf16 [num_layers][num_kv_heads][len][head_dim].
 *   FP8 pool:  the STORED codes and row scales, not re-quantised and not dequantised.  k_dst (v_dst likewise):
 *              e4m3 codes u8 [num_layers][num_kv_heads][len][head_dim], then, at the next 16-byte boundary,
 *              fp32 scales [num_layers][num_kv_heads][len]; kv_gather_bytes() is the size of each of the two.
 * With option src_kv_heads = H the contiguous side is H heads wide (this pool's heads at src_head_begin).   */
int32_t kv_gather(kv_pool_t* pool, int64_t req_id, void* k_dst /*device*/,
                  void* v_dst /*device*/, void* cuda_stream);
/* Bytes kv_gather writes to EACH of k_dst and v_dst for a request of n_tokens tokens; < 0 on an invalid config. */
int64_t kv_gather_bytes(const kv_pool_config_t* cfg, int32_t n_tokens);

/*
 * NEXT-4 — producer -> consumer transfer, paged -> paged (§II: "KV-cache transmission can add on
 * the order of 15-80ms depending on block fragmentation and count"; §V-C: the KV-cache
 * transmitter moves a prefill-completed request's KV into KV-cache blocks registered on the consumer).
 * For i in [0, n_req): request src_req_ids[i] of `src` (the producer's pool), all its len_i tokens, becomes
 * request dst_req_ids[i] of `dst` (this D-instance's pool), layers [layer_begin, layer_begin + layer_count):
 *     dst.kv[l][dst_table_i[t / bs]][h][c][t % bs][:] = src.kv[l][src_table_i[t / bs]][h][c][t % bs][:]
 * — each side addressed through its own block list, block to block, no contiguous staging buffer, ONE launch
 * for all requests (on `dst`'s device, pulling: a src slab that is peer-mapped memory of the producer GPU makes
 * this the NVLink hop and the scatter in one kernel).  src is read-only.  The pools must agree in num_layers,
 * num_kv_heads, head_dim, block_size and kv_dtype (FP8 pools move codes and row scales verbatim); num_blocks,
 * alloc_seed and the block lists are independent.
 *   layer_begin == 0 : dst_req_ids[i] must not be live in dst; it is created with length len_i (kv_reserve).
 *   layer_begin  > 0 : continuation (a producer streaming layer by layer): dst_req_ids[i] must be live with
 *                      length len_i and a last reservation of len_i tokens.
 * Bytes of dst outside the written token slots keep their contents.  Atomic: on any error nothing changes in
 * either pool.  Errors: KV_ERR_UNKNOWN_REQUEST (src id not live), KV_ERR_INVALID (geometry mismatch, src == dst,
 * duplicate ids, dst id live at layer_begin 0), KV_ERR_NO_BLOCKS, KV_ERR_TOO_LONG, KV_ERR_TOO_MANY_REQUESTS,
 * KV_ERR_NO_DEVICE, KV_ERR_CUDA.  The caller orders the call after whatever wrote the src blocks.
 */
int32_t kv_transfer(kv_pool_t* dst, const kv_pool_t* src, int32_t n_req, const int64_t* dst_req_ids /*host*/,
                    const int64_t* src_req_ids /*host*/, int32_t layer_begin, int32_t layer_count,
                    void* cuda_stream);

/*
 * Host-only view of the split-KV plan paged_decode_attention would use for this batch
 * (no GPU work).  A work item is (batch index, kv_head, first block, block count,
 * partial slot or -1 when the item is its request's only chunk and writes `out` directly).
 * out_items: host int32[cap_items][5]; *out_n_items = total item count (may exceed cap);
 * *out_chunk_blocks = chunk size in blocks.  Items are ordered longest-first.
 */
int32_t kv_plan_decode(kv_pool_t* pool, int32_t batch, const int64_t* req_ids /*host*/,
                       int32_t* out_items /*host*/, int32_t cap_items, int32_t* out_n_items,
                       int32_t* out_chunk_blocks);

/*
 * Host-buffer forms of a2/a3 and a4+a5 — the producer's KV (the request
 * "together with KV-cache" handed from P to D) and the step's queries arriving in HOST
 * memory.  Same semantics and errors as kv_ingest / paged_decode_attention, except that
 * k_src[i] / v_src[i] / q / out are HOST pointers (pinned memory for true asynchrony;
 * pageable memory works but the copy is synchronous for the host).  kv_ingest_host reads sources
 * that are pinned, device-addressable (cudaHostAlloc / cudaHostRegister) and 16-byte aligned IN PLACE:
 * the scatter kernel pulls them over PCIe straight into their blocks and `staging` is not touched
 * (option "host_zero_copy", default 1).  Otherwise (pageable sources, or option 0) the sources go
 * through the caller-owned device staging buffer `staging` (device, 256-byte aligned): the copy engine
 * fills it on a stream the pool owns, in groups of requests (pieces of 8 MiB), and each group's scatter
 * is enqueued on `cuda_stream` behind its copies, so a group is scattered while the next one crosses the
 * bus; the copies are ordered behind what precedes the call on `cuda_stream` and behind the scatters of
 * the pool's previous staged call.  Ingest needs sum_i 2 * layer_count*Hkv*n_tokens[i]*d*2 bytes (each
 * tensor rounded up to 256 B), attention needs 2 * batch*Hq*d*2 bytes (rounded likewise);
 * a smaller `staging_bytes` => KV_ERR_INVALID before anything changes.  The staging buffer may be reused
 * by the pool's next call; the host buffers may be reused once the stream has passed the call.
 * (Measured on PCIe 5 x16, one 3.1 GB call alone: 51.5 GB/s in place, 54.0 GB/s staged, 55.5 GB/s a plain copy.)
 */
int32_t kv_ingest_host(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids /*host*/,
                       const int32_t* n_tokens /*host*/,
                       const void* const* k_src /*host array of HOST ptrs*/,
                       const void* const* v_src /*host array of HOST ptrs*/,
                       int32_t layer_begin, int32_t layer_count, void* staging /*device*/,
                       int64_t staging_bytes, void* cuda_stream);
int32_t paged_decode_attention_host(kv_pool_t* pool, int32_t layer, int32_t batch,
                                    const int64_t* req_ids /*host*/, const void* q /*HOST*/,
                                    void* out /*HOST*/, float sm_scale, void* staging /*device*/,
                                    int64_t staging_bytes, void* cuda_stream);
/* paged_decode_step with q, k_new, v_new, out in HOST memory; staging needs
 * 2 * batch*Hq*d*2 + 2 * batch*Hkv*d*2 bytes (each of the four rounded up to 256 B).       */
int32_t paged_decode_step_host(kv_pool_t* pool, int32_t layer, int32_t batch,
                               const int64_t* req_ids /*host*/, const void* q /*HOST*/,
                               const void* k_new /*HOST*/, const void* v_new /*HOST*/,
                               void* out /*HOST*/, float sm_scale, void* staging /*device*/,
                               int64_t staging_bytes, void* cuda_stream);

/* ---- NEXT-3: D-instance capacity model (host only, closed forms) ------------------------ */

/*
 * What the measured bandwidth of this path is FOR in DOPD (§IV-B-2): sizing a
 * D-instance.  Plain fp64 evaluation of
 *     V_mem = (M_gpu - M') x TP - M_model                                  (Eq. 11)
 *     V_BW  = t_d^SLO x alpha x TP x BW                                    (Eq. 12)
 *     cc_d  = min(V_mem, V_BW) / ((ISL + OSL/2) x M_token)                 (Eq. 13)
 * Readings (A10): alpha, undefined in the text, is the achieved fraction of the HBM
 * bandwidth BW (what bench.py measures for the KV part); M_token, undefined in the text, is the KV
 * bytes of one token over the whole model, 2 x layers x kv_heads x head_dim x bytes/element
 * (kv_token_bytes); M_gpu, M', BW are per GPU, M_model and M_token for the whole model.
 * All byte quantities in bytes, times in seconds, lengths in tokens.
 */
typedef struct kv_capacity_model {
  double  m_gpu;       /* HBM bytes per GPU (M_gpu)                                         */
  double  m_reserved;  /* M': peak activation + ancillary bytes per GPU                     */
  double  m_model;     /* model weight bytes, whole model (M_model)                         */
  int32_t tp;          /* tensor-parallel size of the D-instance (TP >= 1)                  */
  double  bw;          /* HBM bytes/s per GPU (BW)                                          */
  double  alpha;       /* achieved fraction of BW, in (0, 1.5]                              */
  double  t_d_slo;     /* TPOT SLO limit, seconds                                           */
  double  isl, osl;    /* input / output sequence length, tokens (isl >= 0, osl > 0)        */
  double  m_token;     /* KV bytes per token, whole model (M_token > 0)                     */
} kv_capacity_model_t;

typedef struct kv_capacity {
  double  v_mem;            /* Eq. 11 (may be <= 0: the model does not fit)                 */
  double  v_bw;             /* Eq. 12                                                       */
  double  cc_d;             /* Eq. 13, not rounded; 0 when v_mem <= 0                       */
  int32_t bandwidth_bound;  /* 1 if v_bw < v_mem (the TPOT SLO, not capacity, limits cc_d)  */
} kv_capacity_t;

/* KV_ERR_INVALID on a null pointer or an argument outside the ranges above; nothing written then. */
int32_t kv_capacity(const kv_capacity_model_t* model, kv_capacity_t* out);

/*
 * Optimal P/D ratio (Eq. 14: n_p x (t_d x OSL / t_p) = n_d x cc_d; the closed form the
 * text announces at PAPER.md:225 is missing from the extraction and is read as)
 *     R_opt = n_p / n_d = cc_d x t_p / (t_d x OSL),
 * t_p = time of one prefill, t_d = time of one decode step at concurrency cc_d, both seconds.
 * All arguments must be > 0, else KV_ERR_INVALID.
 */
int32_t kv_optimal_pd_ratio(double cc_d, double t_p, double t_d, double osl, double* out_ratio);

/* M_token of a pool geometry, the KV bytes one token occupies over the whole model: bf16 pool
 * 2 x num_layers x num_kv_heads x head_dim x 2; FP8 pool num_layers x num_kv_heads x (2 x head_dim + 8)
 * (codes + the two fp32 row scales); < 0 on an invalid config.                               */
int64_t kv_token_bytes(const kv_pool_config_t* cfg);

/* Number of kernels this pool has launched since creation (bench `gpu_launches`).         */
int64_t kv_launch_count(const kv_pool_t* pool);

/* Event counters of this pool since creation, by name (>= 0; KV_ERR_INVALID for an unknown name):
 *   "launches" (= kv_launch_count), "plans_uploaded" (split-KV plans staged; a step's layers share one),
 *   "attn_chained_launches" (attention launches whose predecessor on the stream was an attention launch of the same
 *   plan: their CTAs read work items and block ids before griddepcontrol.wait), "attn_stream_switches" (attention
 *   calls that arrived on another stream and were ordered behind the previous one), "host_ingest_zero_copy" /
 *   "host_ingest_staged" (kv_ingest_host calls that read pinned sources in place / went through `staging`).  */
int64_t kv_pool_counter(const kv_pool_t* pool, const char* name);

/*
 * Per-kernel device timing (bench `roofline`).  With option "profile" = 1 every kernel
 * launch (paged_decode_step_layers: every group of layer_count launches, counted as layer_count) is
 * bracketed by a pair of CUDA events on its own stream (a ring of
 * KV_PROFILE_RING pairs per kind; older samples are folded into the running sums when their
 * slot is reused, which synchronises on that sample).  kv_profile_read synchronises on the
 * outstanding samples of `kind`, returns the number of launches and their summed duration in
 * milliseconds since the last kv_profile_reset, and leaves the sums in place.
 */
#define KV_KERNEL_ATTN     0   /* the decode attention kernel (a4)  */
#define KV_KERNEL_COMBINE  1   /* combine_kernel (a5)               */
#define KV_KERNEL_INGEST   2   /* ingest_kernel, scatter (a2 / a3)  */
#define KV_KERNEL_GATHER   3   /* ingest_kernel, gather direction   */
#define KV_KERNEL_VARQ     4   /* the attention kernel, variable-q  */
#define KV_KERNEL_TRANSFER 5   /* transfer_kernel (NEXT-4)          */
#define KV_KERNEL_KINDS    6
#define KV_PROFILE_RING    1024
int32_t kv_profile_read(kv_pool_t* pool, int32_t kind, int64_t* out_launches, double* out_ms);
int32_t kv_profile_reset(kv_pool_t* pool);

/* Tuning knobs (all optional; defaults chosen for B200).  key: "min_chunk_blocks" (smallest
 * split-KV chunk, in blocks), "ctas_per_sm" (resident attention CTAs per SM the planner
 * sizes the work list for), "items_per_slot" (work items per resident warp), "fuse_combine"
 * (1, default: the split-KV merge runs inside the attention kernel; 0: separate combine
 * kernel), "ring" (bf16 pools: 3, default, or 2 = shared-memory tile ring with that many slots per warp and
 * 2 / 3 CTAs per SM), "pdl" (1, default: attention launches carry the programmatic-dependent-launch attribute;
 * 0: plain launches), "tma" (0, default; 1: pools with head_dim 128 fetch full KV tiles with one
 * cp.async.bulk.tensor per tile (FP8: plus one bulk copy of the tile's scales) instead of 16-byte cp.async — the
 * measured alternative of DESIGN.md §5; KV_ERR_UNSUPPORTED for head_dim 64), "tc" (FP8 pools with head_dim 128: which kernel runs
 * decode attention (paged_decode_attention / _step / _step_layers).  1: attn_tc_kernel on the tcgen05 tensor cores —
 * 128-token tiles staged by TMA, e4m3 operands fed to tcgen05.mma straight from shared memory, accumulators in TMEM;
 * 0: the mma.sync kernel, which also serves paged_varlen_attention, head_dim 64 and bf16 pools whatever the option says;
 * 2 (default): attn_tc_kernel unless more than half of the batch's requests are at most 256 tokens long (it runs one
 * work unit per CTA at a time and pays a pipeline fill per unit; counter "attn_tc_launches" says what ran).  Same
 * results within the stated tolerance, same bytes appended; 1 on a pool that cannot run it => KV_ERR_UNSUPPORTED), "side_upload" (1, default: plan uploads run on a stream the pool owns, beside whatever the
 * caller's stream is executing, and the caller's stream waits for them by event; 0: uploads on the caller's stream), "host_zero_copy" (1, default: see kv_ingest_host), "profile" (0/1, see kv_profile_read);
 * KV-head sharding of a TP-sharded D-instance: "src_kv_heads" = H (0 = off) then
 * "src_head_begin" = h0 declare that the contiguous side of kv_ingest(_host) / kv_gather is the FULL-width tensor
 * [layer_count][H][n_tokens][head_dim] of which this pool holds heads [h0, h0 + num_kv_heads): every GPU of the
 * instance ingests its slice from the same producer buffer, runs attention on its own query heads, and no
 * collective is needed inside this path (q, k_new, v_new, out stay local-width).
 * Unknown key or out-of-range value => KV_ERR_INVALID.                                                          */
int32_t kv_pool_set_option(kv_pool_t* pool, const char* key, int64_t value);

/* Last CUDA error code seen by this pool (cudaError_t as int; 0 = none).                  */
int32_t kv_last_cuda_error(const kv_pool_t* pool);

/* Static string for a status code.                                                        */
const char* kv_strerror(int32_t status);

/* Library version, "major.minor.patch".                                                   */
const char* kv_version(void);

#ifdef __cplusplus
} /* extern "C" */
#endif
#endif /* KV_POOL_H_ */
