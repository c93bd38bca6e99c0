// kv_pool.cu — the C-ABI of include/kv_pool.h: argument checking, host bookkeeping (kv_host.h), staging of small
// descriptor blobs, and kernel launches (kv_copy.cuh, kv_attn.cuh).  Every step of the data path runs in the
// kernels; nothing here touches KV bytes on the host.
#include <cuda.h>           // CUtensorMap and its enums only; the encoder is fetched through the runtime (no -lcuda)
#include <cuda_runtime.h>

#include <cmath>
#include <cstring>
#include <deque>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/kv_pool.h"
#include "kv_host.h"
#include "kv_common.cuh"
#include "kv_copy.cuh"
#include "kv_attn.cuh"
#include "kv_attn_tc.cuh"

namespace {

using namespace kvp;

constexpr int64_t kAlign = 256;
constexpr int kRing = 16;                      // plan staging slots: the host may run this many plan uploads ahead of the GPU
constexpr int64_t kIngestBlobBytes = 2 << 20;  // per ingest launch; larger calls are sub-batched.  One request's
                                               // descriptor (48 B + <= 8 B x kMaxBlocksPerRequest) always fits.
constexpr int64_t kIngestRingBytes = 16 << 20; // descriptor staging ring: ~1000 decode appends in flight
constexpr int32_t kMaxPartials = 32768;        // split-KV partial slots in the workspace
static_assert(sizeof(CUtensorMap) == 128, "AttnParams::tmap carries a CUtensorMap");
static_assert(48 + 8LL * kvp::kMaxBlocksPerRequest <= kIngestBlobBytes, "a request's descriptor must fit one blob");

inline int64_t align_up(int64_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

// ---- static scratch of paged_decode_attention_static (the entry point that allocates nothing) -------------------
// Split-KV workspace for at most KV_STATIC_MAX_PARTIALS partial slots at the widest geometry (G = 8, head_dim 128):
//     arrive  int32 [P]            chunks finished per split (request, kv head) — must be zero when a launch starts
//     part_ml float [P][8][2]      (m, l) of a partial
//     part_o  float [P][8][128]    un-normalised partial outputs
// One array per device that loads the library, held until the process exits; shared by every pool and every call.
constexpr int64_t kStaticArriveBytes = static_cast<int64_t>(KV_STATIC_MAX_PARTIALS) * 4;
constexpr int64_t kStaticMlBytes = static_cast<int64_t>(KV_STATIC_MAX_PARTIALS) * 8 * 2 * 4;
constexpr int64_t kStaticOBytes = static_cast<int64_t>(KV_STATIC_MAX_PARTIALS) * 8 * 128 * 4;
constexpr int64_t kStaticScratchBytes = kStaticArriveBytes + kStaticMlBytes + kStaticOBytes;
static_assert(kStaticArriveBytes % kAlign == 0 && kStaticMlBytes % kAlign == 0, "sections stay 256-byte aligned");
}  // namespace

static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {
// Device address of g_static_scratch on `device`, which must be current.  In host code the array's name is only a
// handle for the runtime, not an address a kernel can use: the address is looked up once per device and cached.
constexpr int kMaxStaticDevices = 64;
cudaError_t static_scratch_address(int device, unsigned char** out) {
  static std::mutex mu;
  static unsigned char* ptrs[kMaxStaticDevices] = {};
  if (device < 0 || device >= kMaxStaticDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!ptrs[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    ptrs[device] = static_cast<unsigned char*>(p);
  }
  *out = ptrs[device];
  return cudaSuccess;
}

struct Layout {  // byte offsets inside the caller's slab
  int64_t kv_bytes, block_table, counters, arrive, ingest_blobs, plan_blobs, part_o, part_ml, total;
  int64_t plan_blob_bytes;
};

int64_t tile_bytes(const kv_pool_config_t& c) {
  return c.kv_dtype == KV_DTYPE_FP8_E4M3 ? 32LL * c.head_dim + 128 : 2LL * c.block_size * c.head_dim * 2;
}

Layout make_layout(const kv_pool_config_t& c) {
  Layout L{};
  const int64_t G = c.num_q_heads / c.num_kv_heads;
  L.kv_bytes = static_cast<int64_t>(c.num_layers) * c.num_blocks * c.num_kv_heads * tile_bytes(c);
  int64_t off = align_up(L.kv_bytes);
  L.block_table = off;
  off = align_up(off + static_cast<int64_t>(c.max_requests) * c.max_blocks_per_request * 4);
  L.counters = off;
  off = align_up(off + 256);
  L.arrive = off;
  off = align_up(off + static_cast<int64_t>(kMaxPartials) * 4);
  L.ingest_blobs = off;
  off = align_up(off + kIngestRingBytes);
  const int64_t items_cap = static_cast<int64_t>(c.max_requests) + kMaxPartials;
  const int64_t comb_cap = static_cast<int64_t>(c.max_requests);
  L.plan_blob_bytes = align_up(items_cap * static_cast<int64_t>(sizeof(WorkItem)) + comb_cap * static_cast<int64_t>(sizeof(CombineEntry)));
  L.plan_blobs = off;
  off = align_up(off + kRing * L.plan_blob_bytes);
  L.part_o = off;
  off = align_up(off + static_cast<int64_t>(kMaxPartials) * G * c.head_dim * 4);
  L.part_ml = off;
  off = align_up(off + static_cast<int64_t>(kMaxPartials) * G * 2 * 4);
  L.total = off;
  return L;
}

struct StageSlot {
  char* host = nullptr;   // pinned
  char* host_dev = nullptr;  // the same pinned buffer as the device addresses it (zero-copy reads by plan_upload_kernel)
  char* dev = nullptr;    // inside the slab
  cudaEvent_t ev = nullptr;
  cudaEvent_t up_ev = nullptr;  // side-stream upload of this slot's plan has completed
  bool in_flight = false;
};

// Descriptor staging for ingest launches: a byte ring in pinned host memory mirrored by a device
// ring in the slab.  Segments are handed out in ring order; a segment is reused only after the
// event recorded behind the launch that read it has completed, so the host never waits on
// unrelated work (a decode append on stream A does not wait for a bulk ingest on stream B unless
// the ring has wrapped all the way round to it).
struct ByteRing {
  struct Seg { int64_t begin, end; cudaEvent_t ev; };
  char* host = nullptr;
  char* dev = nullptr;
  int64_t cap = 0, head = 0;
  std::deque<Seg> inflight;
  std::vector<cudaEvent_t> spare;

  cudaError_t retire_front(bool wait) {
    Seg& f = inflight.front();
    cudaError_t e = wait ? cudaEventSynchronize(f.ev) : cudaEventQuery(f.ev);
    if (e != cudaSuccess) return e;  // cudaErrorNotReady when !wait and still running
    spare.push_back(f.ev);
    inflight.pop_front();
    return cudaSuccess;
  }
  // Reserve `bytes` (<= cap); *off receives the offset valid in both host and dev.
  cudaError_t alloc(int64_t bytes, int64_t* off) {
    bytes = align_up(bytes);
    if (head + bytes > cap) head = 0;
    const int64_t b = head, e = head + bytes;
    for (;;) {
      bool clash = false;
      for (const Seg& s : inflight) if (s.begin < e && b < s.end) { clash = true; break; }
      if (!clash) break;
      cudaError_t err = retire_front(true);
      if (err != cudaSuccess) return err;
    }
    while (!inflight.empty()) {  // opportunistic clean-up keeps the overlap scan short
      cudaError_t err = retire_front(false);
      if (err == cudaErrorNotReady) break;
      if (err != cudaSuccess) return err;
    }
    head = e;
    *off = b;
    return cudaSuccess;
  }
  cudaError_t commit(int64_t off, int64_t bytes, cudaStream_t st) {
    cudaEvent_t ev = nullptr;
    if (!spare.empty()) { ev = spare.back(); spare.pop_back(); }
    else {
      cudaError_t e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
      if (e != cudaSuccess) return e;
    }
    cudaError_t e = cudaEventRecord(ev, st);
    inflight.push_back({off, off + align_up(bytes), ev});
    return e;
  }
  void destroy() {
    for (Seg& s : inflight) cudaEventDestroy(s.ev);
    for (cudaEvent_t e : spare) cudaEventDestroy(e);
    inflight.clear(); spare.clear();
    if (host) cudaFreeHost(host);
    host = nullptr;
  }
};

// Event pairs around the launches of one kernel kind (kv_profile_read).  A pair may bracket a group of
// back-to-back launches (paged_decode_step_layers): the group's time is attributed to `count` launches.
struct ProfRing {
  std::vector<cudaEvent_t> a, b;
  std::vector<int32_t> live;        // launches bracketed by pair i (0: free)
  int next = 0;
  int64_t launches = 0;
  double ms = 0.0;

  cudaError_t fold(int i) {
    if (!live[static_cast<size_t>(i)]) return cudaSuccess;
    cudaError_t e = cudaEventSynchronize(b[static_cast<size_t>(i)]);
    float t = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, a[static_cast<size_t>(i)], b[static_cast<size_t>(i)]);
    if (e == cudaSuccess) { ms += t; launches += live[static_cast<size_t>(i)]; }
    live[static_cast<size_t>(i)] = 0;
    return e;
  }
  cudaError_t begin(cudaStream_t st) {
    if (a.empty()) {
      a.resize(KV_PROFILE_RING); b.resize(KV_PROFILE_RING); live.assign(KV_PROFILE_RING, 0);
      for (int i = 0; i < KV_PROFILE_RING; ++i) {
        cudaError_t e = cudaEventCreate(&a[static_cast<size_t>(i)]);
        if (e == cudaSuccess) e = cudaEventCreate(&b[static_cast<size_t>(i)]);
        if (e != cudaSuccess) return e;
      }
    }
    cudaError_t e = fold(next);
    if (e != cudaSuccess) return e;
    return cudaEventRecord(a[static_cast<size_t>(next)], st);
  }
  cudaError_t end(cudaStream_t st, int32_t count = 1) {
    cudaError_t e = cudaEventRecord(b[static_cast<size_t>(next)], st);
    live[static_cast<size_t>(next)] = count;
    next = (next + 1) % KV_PROFILE_RING;
    return e;
  }
  cudaError_t drain() {
    for (int i = 0; i < static_cast<int>(live.size()); ++i) {
      cudaError_t e = fold(i);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  }
  void destroy() {
    for (cudaEvent_t e : a) if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : b) if (e) cudaEventDestroy(e);
    a.clear(); b.clear(); live.clear();
  }
};

}  // namespace

struct kv_pool {
  kvp::HostState hs;
  Layout lay{};
  bool has_device = false;
  char* base = nullptr;
  int device = 0;                  // the device the slab lives on (cudaPointerGetAttributes at create)
  int num_sms = 148;
  int32_t last_cuda = 0;
  int64_t launches = 0;
  // tuning
  int32_t min_chunk_blocks = 64;   // smallest split-KV chunk: 64 blocks = 512 KiB of KV per unit at d = 128 (bf16);
  bool min_chunk_set = false;      //   FP8 pools default to 32 blocks (tiles are half the bytes) unless the caller chose
  int32_t ctas_per_sm = 0;         // 0: what the kernel variant runs with (2 or 3); else the planner sizes for this many
  int32_t items_per_slot = 2;     // guided chunking: first chunk = remaining work / (2 x resident warps)
  bool items_per_slot_set = false;  // FP8 kernel (12 warps per SM): 1 measured best unless the caller chose
  bool fuse_combine = true;
  int32_t src_kv_heads = 0;       // KV-head sharding: heads of the contiguous side of ingest / gather (0: this pool's own)
  int32_t src_head_begin = 0;     //                   this pool's head 0 is that side's head src_head_begin
  int32_t ring = 3;               // bf16 pool: ring slots per warp, 3 (2 CTAs per SM, default) or 2 (3 CTAs per SM)
  bool pdl = true;                // attention launches carry the programmatic-dependent-launch attribute
  bool side_upload = true;        // plan uploads on the pool's own stream (overlapping the caller's stream), joined by an event
  cudaStream_t up_stream = nullptr;
  // kv_ingest_host, staged form: the copy engine fills the caller's staging buffer on this stream, group of requests
  // by group, while the scatter of the previous group runs on the caller's stream
  cudaStream_t copy_stream = nullptr;
  static constexpr int kStageGroups = 16;
  cudaEvent_t grp_ev[kStageGroups] = {};
  cudaEvent_t stage_ev = nullptr;   // behind the last scatter that read the staging buffer
  bool stage_busy = false;
  bool tma = false;               // bf16 pools, head_dim 128: full tiles by cp.async.bulk.tensor (UTMALDG) instead of LDGSTS
  bool tmap_ok = false;
  int32_t tc = 2;                 // FP8 pools, head_dim 128: decode attention on tcgen05 / TMEM (attn_tc_kernel): 0 never (mma.sync
                                  //   kernel), 1 always, 2 (default) unless most of the batch's requests are one or two tiles long
  bool tmap16_ok = false;
  alignas(64) CUtensorMap tmap16; // the same region, box 16 rows: the K codes or the V codes of one (block, kv head) tile
  alignas(64) CUtensorMap tmap;   // the KV region as [rows][128 B], box 64 rows, 128-byte swizzle
  // event counters (kv_pool_counter)
  int64_t n_zero_copy = 0, n_staged = 0, n_chained = 0, n_stream_switch = 0, n_plans = 0, n_tc_launches = 0;
  bool host_zero_copy = true;     // kv_ingest_host reads device-addressable pinned sources in place (no staging pass)
  bool profile = false;
  ProfRing prof[KV_KERNEL_KINDS];
  // staging
  ByteRing ingest_ring;
  StageSlot plan_ring[kRing];
  int plan_next = 0;
  // cached decode plan (reused across the layers of one step)
  uint64_t plan_epoch = 0;
  std::vector<int64_t> plan_ids;
  int plan_slot = -1;
  int32_t plan_n_items = 0, plan_n_combines = 0;
  int32_t plan_kind = 0;        // 0: decode plan, 1: variable-q plan (48-byte items)
  bool plan_tc = false;         // the decode plan was sized for (and runs on) attn_tc_kernel
  std::vector<int32_t> plan_qlens;
  std::vector<kvp::HostState::QueryTile> plan_tiles;
  int32_t plan_append_ok = -1;  // -1 unknown, 0 / 1: every request's last reservation is one token
  int64_t plan_combine_off = 0;
  kvp::DecodePlan plan;
  std::vector<int32_t> ones;
  // ordering of attention launches (they share the pool's device workspace): the stream of the last one and an
  // event behind it (the staged plan slot's), and what a following launch may assume about its predecessor
  bool attn_any = false;
  cudaStream_t attn_stream = nullptr;
  cudaEvent_t attn_ev = nullptr;
  int chain_slot = -1;          // plan slot of the pool's LAST launch if that was an attention launch, else -1
  int chain_kind = 0;           // 0 decode, 1 decode + append, 2 variable-q

  int32_t cuda_fail(cudaError_t e) {
    last_cuda = static_cast<int32_t>(e);
    return KV_ERR_CUDA;
  }
  bool fp8() const { return hs.cfg.kv_dtype == KV_DTYPE_FP8_E4M3; }
  int32_t kernel_ctas() const { return fp8() ? 3 : (ring == 2 ? 3 : 2); }
  bool tc_capable() const { return tc != 0 && tmap16_ok; }
  // tcgen05 kernel for this decode batch?  It runs ONE unit at a time per CTA (two per SM): a batch made mostly of requests
  // of one or two 128-token tiles (config 5: 80 % of the requests, 3280 of 4392 units) is better served by the mma.sync
  // kernel's twelve independent warps per SM (measured: 1.02 vs 0.995 of the copy ceiling there; 1.05 vs 1.07 on config 4)
  bool tc_for(int32_t batch, const int64_t* req_ids) const {
    if (!tc_capable()) return false;
    if (tc == 1) return true;
    int32_t small = 0;
    for (int32_t i = 0; i < batch; ++i) {
      auto it = hs.reqs.find(req_ids[i]);
      if (it != hs.reqs.end() && it->second.len <= 2 * kvp::kTcTileTokens) ++small;
    }
    return 2 * small <= batch;
  }
  // work units the attention kernel of a decode (or variable-q) launch processes at a time: resident warps of the
  // mma.sync kernels, resident CTAs of the tcgen05 kernel
  int32_t slots(bool varq = false, bool use_tc = false) const {
    if (!varq && use_tc) return num_sms * (ctas_per_sm > 0 ? ctas_per_sm : 2);
    return num_sms * (ctas_per_sm > 0 ? ctas_per_sm : kernel_ctas()) * kvp::kAttnWarps;
  }
  int32_t src_heads() const { return src_kv_heads > 0 ? src_kv_heads : hs.cfg.num_kv_heads; }
  int32_t min_chunk() const { return (fp8() && !min_chunk_set) ? 32 : min_chunk_blocks; }
  int32_t ips() const { return (fp8() && !items_per_slot_set) ? 1 : items_per_slot; }
};

namespace {

#define KV_CUDA(pool, expr)                                   \
  do {                                                        \
    cudaError_t e_ = (expr);                                  \
    if (e_ != cudaSuccess) return (pool)->cuda_fail(e_);      \
  } while (0)

// Calls run on the pool's device whatever device is current, and leave the caller's current device as it was.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(const kv_pool* pool) {
    if (!pool->has_device) return;
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != pool->device) {
      err = cudaSetDevice(pool->device);
      switched = err == cudaSuccess;
    }
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define KV_ON_DEVICE(pool)                                    \
  DeviceGuard guard_(pool);                                   \
  if (guard_.err != cudaSuccess) return (pool)->cuda_fail(guard_.err)

int32_t acquire(kv_pool* pool, StageSlot* ring, int* next, StageSlot** out) {
  const int idx = *next;
  *next = (idx + 1) % kRing;
  StageSlot& s = ring[idx];
  if (s.in_flight) {
    KV_CUDA(pool, cudaEventSynchronize(s.ev));
    s.in_flight = false;
  }
  *out = &s;
  return idx;
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

enum class CopyKind { kScatter, kGather, kTransfer };

// One launch of a relocation kernel over the serialised requests `reqs` / block ids `ids`.
int32_t launch_copy(kv_pool* pool, CopyKind kind, const kv_pool* src_pool, const std::vector<IngestReq>& reqs,
                    const std::vector<int32_t>& ids, int64_t total_units, int32_t layer_begin, int32_t layer_count,
                    cudaStream_t stream) {
  if (total_units == 0) return KV_OK;
  const size_t req_bytes = reqs.size() * sizeof(IngestReq);
  const size_t id_bytes = ids.size() * sizeof(int32_t);
  ByteRing& ring = pool->ingest_ring;
  int64_t off = 0;
  KV_CUDA(pool, ring.alloc(static_cast<int64_t>(req_bytes + id_bytes), &off));
  char* hbuf = ring.host + off;
  char* dbuf = ring.dev + off;
  std::memcpy(hbuf, reqs.data(), req_bytes);
  std::memcpy(hbuf + req_bytes, ids.data(), id_bytes);
  KV_CUDA(pool, cudaMemcpyAsync(dbuf, hbuf, req_bytes + id_bytes, cudaMemcpyHostToDevice, stream));
  const kv_pool_config_t& c = pool->hs.cfg;
  IngestParams p{};
  p.reqs = reinterpret_cast<const IngestReq*>(dbuf);
  p.blk_ids = reinterpret_cast<const int32_t*>(dbuf + req_bytes);
  p.n_req = static_cast<int32_t>(reqs.size());
  p.total_units = total_units;
  p.kv = reinterpret_cast<uint16_t*>(pool->base);
  p.block_table = reinterpret_cast<int32_t*>(pool->base + pool->lay.block_table);
  p.bt_stride = c.max_blocks_per_request;
  p.layer_begin = layer_begin;
  p.layer_count = layer_count;
  p.num_kv_heads = c.num_kv_heads;
  p.num_blocks = c.num_blocks;
  p.src_kv_heads = pool->src_heads();
  p.src_head_begin = pool->src_head_begin;
  if (src_pool) {
    p.src_kv = reinterpret_cast<const uint16_t*>(src_pool->base);
    p.src_num_blocks = src_pool->hs.cfg.num_blocks;
  }
  const bool fp8 = pool->fp8(), d128 = c.head_dim == 128;
  const unsigned grid = static_cast<unsigned>((total_units + kIngestWarps - 1) / kIngestWarps);
  const int prof_kind = kind == CopyKind::kScatter ? KV_KERNEL_INGEST : kind == CopyKind::kGather ? KV_KERNEL_GATHER : KV_KERNEL_TRANSFER;
  ProfRing& pr = pool->prof[prof_kind];
  if (pool->profile) KV_CUDA(pool, pr.begin(stream));
  if (kind == CopyKind::kTransfer) {
    if (fp8) { if (d128) transfer_kernel<128, true><<<grid, kIngestThreads, 0, stream>>>(p); else transfer_kernel<64, true><<<grid, kIngestThreads, 0, stream>>>(p); }
    else     { if (d128) transfer_kernel<128, false><<<grid, kIngestThreads, 0, stream>>>(p); else transfer_kernel<64, false><<<grid, kIngestThreads, 0, stream>>>(p); }
  } else if (kind == CopyKind::kGather) {
    if (fp8) { if (d128) gather_fp8_kernel<128><<<grid, kIngestThreads, 0, stream>>>(p); else gather_fp8_kernel<64><<<grid, kIngestThreads, 0, stream>>>(p); }
    else     { if (d128) ingest_kernel<128, true><<<grid, kIngestThreads, 0, stream>>>(p); else ingest_kernel<64, true><<<grid, kIngestThreads, 0, stream>>>(p); }
  } else if (fp8) {
    const unsigned grid8 = static_cast<unsigned>((2 * total_units + kIngest8Warps - 1) / kIngest8Warps);   // a warp per (unit, K|V)
    if (d128) ingest_fp8_kernel<128><<<grid8, kIngest8Threads, 0, stream>>>(p); else ingest_fp8_kernel<64><<<grid8, kIngest8Threads, 0, stream>>>(p);
  } else {
    if (d128) ingest_kernel<128, false><<<grid, kIngestThreads, 0, stream>>>(p); else ingest_kernel<64, false><<<grid, kIngestThreads, 0, stream>>>(p);
  }
  KV_CUDA(pool, cudaGetLastError());
  if (pool->profile) KV_CUDA(pool, pr.end(stream));
  ++pool->launches;
  pool->chain_slot = -1;   // the pool's last launch is no longer an attention launch
  KV_CUDA(pool, ring.commit(off, static_cast<int64_t>(req_bytes + id_bytes), stream));
  return KV_OK;
}

// Serialise requests into copy launches, sub-batching so each blob fits its staging segment.  For a transfer
// src_pool / src_ids name the producer's pool and request ids; its block ids follow the consumer's per request.
int32_t run_copy(kv_pool* pool, CopyKind kind, const kv_pool* src_pool, const int64_t* src_ids, int32_t n_req,
                 const int64_t* req_ids, const int32_t* n_tokens, const void* const* k_ptrs, const void* const* v_ptrs,
                 const int32_t* start_pos, int32_t layer_begin, int32_t layer_count, cudaStream_t stream) {
  const kv_pool_config_t& c = pool->hs.cfg;
  // blocks per unit: the quantising scatter gives a warp a run of consecutive blocks, the plain copies one block
  // (a run of two FP8 tiles per warp in the transfer was measured: 0.951 -> 0.928 of the copy ceiling, not kept)
  const int32_t run = (kind == CopyKind::kScatter && pool->fp8()) ? kIngest8Run : 1;
  std::vector<IngestReq> reqs;
  std::vector<int32_t> ids;
  int64_t units = 0;
  auto flush = [&]() -> int32_t {
    int32_t rc = launch_copy(pool, kind, src_pool, reqs, ids, units, layer_begin, layer_count, stream);
    reqs.clear();
    ids.clear();
    units = 0;
    return rc;
  };
  for (int32_t i = 0; i < n_req; ++i) {
    if (n_tokens[i] == 0) continue;
    const Request& r = pool->hs.reqs.find(req_ids[i])->second;
    const int32_t sp = start_pos[i];
    const int32_t b0 = sp / c.block_size;
    const int32_t b1 = (sp + n_tokens[i] - 1) / c.block_size;
    const int32_t touched = b1 - b0 + 1;
    const int64_t need = static_cast<int64_t>(sizeof(IngestReq)) + (src_pool ? 8LL : 4LL) * touched;
    const int64_t used = static_cast<int64_t>(reqs.size() * sizeof(IngestReq) + ids.size() * 4);
    if (used + need > kIngestBlobBytes) {   // need alone always fits (kMaxBlocksPerRequest)
      int32_t rc = flush();
      if (rc != KV_OK) return rc;
    }
    IngestReq q{};
    q.k_src = k_ptrs ? reinterpret_cast<uint64_t>(k_ptrs[i]) : 0;
    q.v_src = v_ptrs ? reinterpret_cast<uint64_t>(v_ptrs[i]) : 0;
    q.unit_begin = units;
    q.n_tokens = n_tokens[i];
    q.start_pos = sp;
    q.slot = r.slot;
    q.blk0 = b0;
    q.n_touched = touched;
    q.blk_off = static_cast<int32_t>(ids.size());
    reqs.push_back(q);
    ids.insert(ids.end(), r.blocks.begin() + b0, r.blocks.begin() + b1 + 1);
    if (src_pool) {
      const Request& sr = src_pool->hs.reqs.find(src_ids[i])->second;
      ids.insert(ids.end(), sr.blocks.begin() + b0, sr.blocks.begin() + b1 + 1);
    }
    units += static_cast<int64_t>((touched + run - 1) / run) * layer_count * c.num_kv_heads;
  }
  return flush();
}

// ---- attention kernel variants ---------------------------------------------------------------

using AttnFn = void (*)(const AttnParams);
struct AttnVariant {
  AttnFn fn;
  size_t smem;
  int ctas;
  int threads = kAttnThreads;
  int units_per_cta = kAttnWarps;   // work units a CTA processes at a time
};

constexpr int kFp8RingSlots = 4;   // FP8 pools: 4 ring slots per warp, 3 CTAs per SM

template <class TP, bool kAppend, bool kVarQ, int R, int kCtas>
AttnVariant variant() {
  // TMA variants: + 1 KiB so the rings can start on a 1 KiB boundary, + one mbarrier per slot and warp
  const size_t extra = TP::kTma ? 1024 + static_cast<size_t>(kAttnWarps) * R * 8 : 0;
  return {attn_kernel<TP, kAppend, kVarQ, R, kCtas>, static_cast<size_t>(kAttnWarps) * TP::template warp_ring_bytes<R>() + extra, kCtas};
}
template <class TP, int R, int kCtas>
AttnVariant variant_of(bool append, bool varq) {
  if (varq) return variant<TP, false, true, R, kCtas>();
  return append ? variant<TP, true, false, R, kCtas>() : variant<TP, false, false, R, kCtas>();
}
AttnVariant pick_variant(const kv_pool* pool, bool append, bool varq, bool use_tc = false) {
  const bool d128 = pool->hs.cfg.head_dim == 128;
  if (!varq && use_tc)
    return {append ? attn_tc_kernel<true> : attn_tc_kernel<false>, kTcSmemBytes, 2, kTcThreads, 1};
  if (pool->fp8() && pool->tma && pool->tmap_ok && d128) return variant_of<Fp8Tiles<128, true>, kFp8RingSlots, 3>(append, varq);
  if (pool->fp8())
    return d128 ? variant_of<Fp8Tiles<128>, kFp8RingSlots, 3>(append, varq) : variant_of<Fp8Tiles<64>, kFp8RingSlots, 3>(append, varq);
  if (pool->tma && pool->tmap_ok && d128) return variant_of<Bf16Tiles<128, true>, 3, 2>(append, varq);
  if (pool->ring == 2)
    return d128 ? variant_of<Bf16Tiles<128>, 2, 3>(append, varq) : variant_of<Bf16Tiles<64>, 2, 3>(append, varq);
  return d128 ? variant_of<Bf16Tiles<128>, 3, 2>(append, varq) : variant_of<Bf16Tiles<64>, 3, 2>(append, varq);
}

// The KV region as a 2-D tensor of 128-byte rows (head_dim 128): a bf16 (block, kv head) tile is 64 consecutive rows,
// an FP8 tile 33 (32 code rows + the scales row).  CU_TENSOR_MAP_SWIZZLE_128B is the layout the <.., true> providers read.
bool make_tensor_map(kv_pool* pool, CUtensorMap* out, uint32_t box_rows) {
  const kv_pool_config_t& c = pool->hs.cfg;
  if (c.head_dim != 128 || pool->lay.kv_bytes % 128 != 0) return false;
  using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres{};
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return false;
  }
  const cuuint64_t rows = static_cast<cuuint64_t>(pool->lay.kv_bytes / 128);
  if (rows >= (1ull << 31)) return false;                       // tile coordinates are int32
  const cuuint64_t gdim[2] = {128, rows};
  const cuuint64_t gstride[1] = {128};                           // bytes between rows (dimension 1)
  const cuuint32_t box[2] = {128, box_rows};
  const cuuint32_t estride[2] = {1, 1};
  const CUresult r = reinterpret_cast<EncodeFn>(fn)(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, pool->base, gdim, gstride, box,
                                                    estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// Dynamic shared memory above 48 KiB needs an opt-in per (kernel, device).
cudaError_t ensure_smem_optin(const AttnVariant& v, int device) {
  struct Key { AttnFn fn; int dev; };
  static std::vector<Key> done;
  for (const Key& k : done) if (k.fn == v.fn && k.dev == device) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void*>(v.fn), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       static_cast<int>(v.smem));
  if (e == cudaSuccess) done.push_back({v.fn, device});
  return e;
}

cudaError_t launch_attn_kernel(const kv_pool* pool, const AttnVariant& v, const AttnParams& p, cudaStream_t stream) {
  cudaError_t e = ensure_smem_optin(v, pool->device);
  if (e != cudaSuccess) return e;
  const int32_t want = (p.n_units + v.units_per_cta - 1) / v.units_per_cta;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(std::max(1, std::min(want, pool->num_sms * v.ctas))));
  cfg.blockDim = dim3(static_cast<unsigned>(v.threads));
  cfg.dynamicSmemBytes = v.smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pool->pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, v.fn, p);
}

// Stage a plan blob: with PDL a kernel reads the pinned staging buffer in place (the stream stays kernel-only, so
// the programmatic chain is not cut by a copy); without it a plain cudaMemcpyAsync.
cudaError_t upload_plan(kv_pool* pool, const StageSlot& s, size_t bytes, cudaStream_t stream) {
  ++pool->n_plans;
  if (!pool->pdl || bytes == 0) return bytes ? cudaMemcpyAsync(s.dev, s.host, bytes, cudaMemcpyHostToDevice, stream) : cudaSuccess;
  const int n16 = static_cast<int>((bytes + 15) / 16);
  const unsigned grid = static_cast<unsigned>(std::max(1, std::min((n16 + 255) / 256, 32)));
  if (pool->side_upload && pool->up_stream) {
    // The slot is free (acquire waited for its last reader) and nothing else touches it: the copy may run beside
    // whatever the caller's stream is executing; the caller's stream only waits for its completion.
    plan_upload_kernel<<<grid, 256, 0, pool->up_stream>>>(reinterpret_cast<const uint4*>(s.host_dev), reinterpret_cast<uint4*>(s.dev), n16);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventRecord(s.up_ev, pool->up_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, s.up_ev, 0);
    return e;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(256);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, plan_upload_kernel, reinterpret_cast<const uint4*>(s.host_dev), reinterpret_cast<uint4*>(s.dev), n16);
}

// Attention launches of one pool must not overlap (shared workspace): a call on another stream than the
// previous one is ordered behind it.
int32_t order_attention(kv_pool* pool, cudaStream_t stream) {
  if (pool->attn_any && stream != pool->attn_stream) {
    KV_CUDA(pool, cudaStreamWaitEvent(stream, pool->attn_ev, 0));
    pool->chain_slot = -1;
    ++pool->n_stream_switch;
  }
  return KV_OK;
}

void attention_launched(kv_pool* pool, cudaStream_t stream, const StageSlot& s, int kind) {
  pool->attn_any = true;
  pool->attn_stream = stream;
  pool->attn_ev = s.ev;
  pool->chain_slot = pool->plan_slot;
  pool->chain_kind = kind;
}

}  // namespace

extern "C" {

int64_t kv_pool_kv_bytes(const kv_pool_config_t* cfg) {
  if (!cfg) return KV_ERR_INVALID;
  int32_t rc = HostState::validate(*cfg);
  if (rc != KV_OK) return rc;
  return make_layout(*cfg).kv_bytes;
}

int64_t kv_pool_required_bytes(const kv_pool_config_t* cfg) {
  if (!cfg) return KV_ERR_INVALID;
  int32_t rc = HostState::validate(*cfg);
  if (rc != KV_OK) return rc;
  return make_layout(*cfg).total;
}

int32_t kv_pool_create(const kv_pool_config_t* cfg, kv_pool_t** out_pool) {
  if (!cfg || !out_pool) return KV_ERR_INVALID;
  *out_pool = nullptr;
  int32_t rc = HostState::validate(*cfg);
  if (rc != KV_OK) return rc;
  const Layout lay = make_layout(*cfg);
  if (cfg->device_base) {
    if ((reinterpret_cast<uintptr_t>(cfg->device_base) & (kAlign - 1)) != 0) return KV_ERR_INVALID;
    if (cfg->device_bytes < lay.total) return KV_ERR_INVALID;
  }
  kv_pool* pool = new (std::nothrow) kv_pool();
  if (!pool) return KV_ERR_INVALID;
  pool->hs.init(*cfg);
  pool->lay = lay;
  if (cfg->device_base) {
    pool->base = static_cast<char*>(cfg->device_base);
    // the pool lives where its slab lives, whatever device happens to be current
    cudaPointerAttributes pa{};
    cudaError_t e = cudaPointerGetAttributes(&pa, cfg->device_base);
    if (e == cudaSuccess && pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) {
      delete pool;
      return KV_ERR_INVALID;
    }
    if (e == cudaSuccess) pool->device = pa.device;
    pool->has_device = true;
    DeviceGuard guard(pool);
    if (e == cudaSuccess) e = guard.err;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&pool->num_sms, cudaDevAttrMultiProcessorCount, pool->device);
    if (e == cudaSuccess) e = cudaHostAlloc(reinterpret_cast<void**>(&pool->ingest_ring.host), kIngestRingBytes, cudaHostAllocDefault);
    pool->ingest_ring.dev = pool->base + lay.ingest_blobs;
    pool->ingest_ring.cap = kIngestRingBytes;
    for (int i = 0; e == cudaSuccess && i < kRing; ++i) {
      e = cudaHostAlloc(reinterpret_cast<void**>(&pool->plan_ring[i].host), lay.plan_blob_bytes, cudaHostAllocMapped);
      if (e == cudaSuccess) e = cudaHostGetDevicePointer(reinterpret_cast<void**>(&pool->plan_ring[i].host_dev), pool->plan_ring[i].host, 0);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pool->plan_ring[i].ev, cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pool->plan_ring[i].up_ev, cudaEventDisableTiming);
      pool->plan_ring[i].dev = pool->base + lay.plan_blobs + i * lay.plan_blob_bytes;
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&pool->up_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&pool->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; e == cudaSuccess && i < kv_pool::kStageGroups; ++i) e = cudaEventCreateWithFlags(&pool->grp_ev[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pool->stage_ev, cudaEventDisableTiming);
    // work counters start at zero; the attention kernel rewinds them itself afterwards
    // FP8: the 32 code rows of a tile in one box (its scales row follows them); bf16: the tile's 64 rows
    if (e == cudaSuccess) pool->tmap_ok = make_tensor_map(pool, &pool->tmap, pool->fp8() ? 32u : 64u);
    if (e == cudaSuccess && pool->fp8()) pool->tmap16_ok = make_tensor_map(pool, &pool->tmap16, 16u);
    if (e == cudaSuccess) e = cudaMemset(pool->base + lay.counters, 0, 256);
    if (e == cudaSuccess) e = cudaMemset(pool->base + lay.arrive, 0, static_cast<size_t>(kMaxPartials) * 4);
    if (e != cudaSuccess) {
      kv_pool_destroy(pool);
      return KV_ERR_CUDA;
    }
  }
  *out_pool = pool;
  return KV_OK;
}

int32_t kv_pool_destroy(kv_pool_t* pool) {
  if (!pool) return KV_ERR_INVALID;
  {
    DeviceGuard guard(pool);
    pool->ingest_ring.destroy();
    for (int i = 0; i < kRing; ++i) {
      if (pool->plan_ring[i].host) cudaFreeHost(pool->plan_ring[i].host);
      if (pool->plan_ring[i].ev) cudaEventDestroy(pool->plan_ring[i].ev);
      if (pool->plan_ring[i].up_ev) cudaEventDestroy(pool->plan_ring[i].up_ev);
    }
    for (ProfRing& r : pool->prof) r.destroy();
    if (pool->up_stream) { cudaStreamSynchronize(pool->up_stream); cudaStreamDestroy(pool->up_stream); }
    if (pool->copy_stream) { cudaStreamSynchronize(pool->copy_stream); cudaStreamDestroy(pool->copy_stream); }
    for (cudaEvent_t ev : pool->grp_ev) if (ev) cudaEventDestroy(ev);
    if (pool->stage_ev) cudaEventDestroy(pool->stage_ev);
  }
  delete pool;
  return KV_OK;
}

int32_t kv_reserve(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids, const int32_t* n_tokens) {
  if (!pool) return KV_ERR_INVALID;
  return pool->hs.reserve(n_req, req_ids, n_tokens);
}

// a1 (reserve or continuation check) + a2/a3 launch, atomic: any failure after the reservation rolls it back.
static int32_t ingest_reserved(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids, const int32_t* n_tokens,
                               const void* const* k_dev, const void* const* v_dev, int32_t layer_begin,
                               int32_t layer_count, cudaStream_t stream) {
  std::vector<int32_t> start(static_cast<size_t>(n_req));
  for (int32_t i = 0; i < n_req; ++i) start[static_cast<size_t>(i)] = pool->hs.reqs.find(req_ids[i])->second.len - n_tokens[i];
  int32_t rc = run_copy(pool, CopyKind::kScatter, nullptr, nullptr, n_req, req_ids, n_tokens, k_dev, v_dev, start.data(),
                        layer_begin, layer_count, stream);
  if (rc != KV_OK && layer_begin == 0) pool->hs.rollback_last_reserve();
  return rc;
}

static int32_t ingest_args_ok(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids, const int32_t* n_tokens,
                              const void* const* k_src, const void* const* v_src, int32_t layer_begin, int32_t layer_count,
                              bool need_aligned) {
  if (!pool || n_req < 0) return KV_ERR_INVALID;
  if (n_req > 0 && (!req_ids || !n_tokens || !k_src || !v_src)) return KV_ERR_INVALID;
  const kv_pool_config_t& c = pool->hs.cfg;
  if (layer_begin < 0 || layer_count < 1 || layer_begin + layer_count > c.num_layers) return KV_ERR_INVALID;
  if (!pool->has_device) return KV_ERR_NO_DEVICE;
  for (int32_t i = 0; i < n_req; ++i) {
    if (n_tokens[i] < 0) return KV_ERR_INVALID;
    if (n_tokens[i] > 0 && (!k_src[i] || !v_src[i])) return KV_ERR_INVALID;
    if (n_tokens[i] > 0 && need_aligned && (!aligned16(k_src[i]) || !aligned16(v_src[i]))) return KV_ERR_INVALID;
  }
  return KV_OK;
}

int32_t kv_ingest(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids, const int32_t* n_tokens,
                  const void* const* k_src, const void* const* v_src, int32_t layer_begin, int32_t layer_count,
                  void* cuda_stream) {
  int32_t rc = ingest_args_ok(pool, n_req, req_ids, n_tokens, k_src, v_src, layer_begin, layer_count, true);
  if (rc != KV_OK) return rc;
  KV_ON_DEVICE(pool);
  rc = layer_begin == 0 ? pool->hs.reserve(n_req, req_ids, n_tokens)      // a1
                        : pool->hs.check_batch(n_req, req_ids, n_tokens); // continuation of the last reservation
  if (rc != KV_OK) return rc;
  return ingest_reserved(pool, n_req, req_ids, n_tokens, k_src, v_src, layer_begin, layer_count,
                         static_cast<cudaStream_t>(cuda_stream));
}

int64_t kv_gather_bytes(const kv_pool_config_t* cfg, int32_t n_tokens) {
  if (!cfg || n_tokens < 0) return KV_ERR_INVALID;
  int32_t rc = HostState::validate(*cfg);
  if (rc != KV_OK) return rc;
  const int64_t rows = static_cast<int64_t>(cfg->num_layers) * cfg->num_kv_heads * n_tokens;
  if (cfg->kv_dtype == KV_DTYPE_FP8_E4M3) return (rows * cfg->head_dim + 15) / 16 * 16 + rows * 4;
  return rows * cfg->head_dim * 2;
}

int32_t kv_gather(kv_pool_t* pool, int64_t req_id, void* k_dst, void* v_dst, void* cuda_stream) {
  if (!pool || !k_dst || !v_dst || !aligned16(k_dst) || !aligned16(v_dst)) return KV_ERR_INVALID;
  if (!pool->has_device) return KV_ERR_NO_DEVICE;
  auto it = pool->hs.reqs.find(req_id);
  if (it == pool->hs.reqs.end()) return KV_ERR_UNKNOWN_REQUEST;
  KV_ON_DEVICE(pool);
  const int32_t n = it->second.len, zero = 0;
  const void* kp = k_dst;
  const void* vp = v_dst;
  return run_copy(pool, CopyKind::kGather, nullptr, nullptr, 1, &req_id, &n, &kp, &vp, &zero, 0, pool->hs.cfg.num_layers,
                  static_cast<cudaStream_t>(cuda_stream));
}

int32_t kv_transfer(kv_pool_t* dst, const kv_pool_t* src, int32_t n_req, const int64_t* dst_req_ids,
                    const int64_t* src_req_ids, int32_t layer_begin, int32_t layer_count, void* cuda_stream) {
  if (!dst || !src || dst == src || n_req < 0) return KV_ERR_INVALID;
  if (n_req > 0 && (!dst_req_ids || !src_req_ids)) return KV_ERR_INVALID;
  const kv_pool_config_t& a = src->hs.cfg;
  const kv_pool_config_t& b = dst->hs.cfg;
  if (a.num_layers != b.num_layers || a.num_kv_heads != b.num_kv_heads || a.head_dim != b.head_dim ||
      a.block_size != b.block_size || a.kv_dtype != b.kv_dtype)
    return KV_ERR_INVALID;
  if (layer_begin < 0 || layer_count < 1 || layer_begin + layer_count > b.num_layers) return KV_ERR_INVALID;
  if (!dst->has_device || !src->has_device) return KV_ERR_NO_DEVICE;
  std::vector<int32_t> lens(static_cast<size_t>(n_req)), zeros(static_cast<size_t>(n_req), 0);
  {
    int32_t rc = src->hs.check_batch(n_req, src_req_ids, nullptr);   // every producer id live, none repeated
    if (rc != KV_OK) return rc;
  }
  for (int32_t i = 0; i < n_req; ++i) {
    lens[static_cast<size_t>(i)] = src->hs.reqs.find(src_req_ids[i])->second.len;
    if (layer_begin == 0 && dst->hs.reqs.count(dst_req_ids[i])) return KV_ERR_INVALID;   // must be new on the consumer
  }
  KV_ON_DEVICE(dst);
  int32_t rc = layer_begin == 0 ? dst->hs.reserve(n_req, dst_req_ids, lens.data())
                                : dst->hs.check_batch(n_req, dst_req_ids, lens.data());
  if (rc != KV_OK) return rc;
  if (layer_begin > 0)
    for (int32_t i = 0; i < n_req; ++i)
      if (dst->hs.reqs.find(dst_req_ids[i])->second.len != lens[static_cast<size_t>(i)]) return KV_ERR_INVALID;
  rc = run_copy(dst, CopyKind::kTransfer, src, src_req_ids, n_req, dst_req_ids, lens.data(), nullptr, nullptr, zeros.data(),
                layer_begin, layer_count, static_cast<cudaStream_t>(cuda_stream));
  if (rc != KV_OK && layer_begin == 0) dst->hs.rollback_last_reserve();
  return rc;
}

int32_t kv_free(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids) {
  if (!pool) return KV_ERR_INVALID;
  return pool->hs.release(n_req, req_ids);
}

int32_t kv_block_table(const kv_pool_t* pool, int64_t req_id, int32_t* out_blocks, int32_t cap, int32_t* out_n_blocks,
                       int32_t* out_len) {
  if (!pool || cap < 0 || (cap > 0 && !out_blocks)) return KV_ERR_INVALID;
  auto it = pool->hs.reqs.find(req_id);
  if (it == pool->hs.reqs.end()) return KV_ERR_UNKNOWN_REQUEST;
  const Request& r = it->second;
  const int32_t nb = static_cast<int32_t>(r.blocks.size());
  for (int32_t i = 0; i < std::min(nb, cap); ++i) out_blocks[i] = r.blocks[static_cast<size_t>(i)];
  if (out_n_blocks) *out_n_blocks = nb;
  if (out_len) *out_len = r.len;
  return KV_OK;
}

int32_t kv_pool_stats(const kv_pool_t* pool, int64_t* blocks_total, int64_t* blocks_free, int32_t* live_requests,
                      int64_t* blocks_high_water) {
  if (!pool) return KV_ERR_INVALID;
  if (blocks_total) *blocks_total = pool->hs.alloc.total();
  if (blocks_free) *blocks_free = pool->hs.alloc.free_count();
  if (live_requests) *live_requests = static_cast<int32_t>(pool->hs.reqs.size());
  if (blocks_high_water) *blocks_high_water = pool->hs.alloc.high_water();
  return KV_OK;
}

int32_t kv_plan_decode(kv_pool_t* pool, int32_t batch, const int64_t* req_ids, int32_t* out_items, int32_t cap_items,
                       int32_t* out_n_items, int32_t* out_chunk_blocks) {
  if (!pool || cap_items < 0 || (cap_items > 0 && !out_items)) return KV_ERR_INVALID;
  DecodePlan plan;
  const bool use_tc = req_ids && batch > 0 && pool->tc_for(batch, req_ids);
  int32_t rc = pool->hs.plan_decode(batch, req_ids, pool->slots(false, use_tc), pool->ips(), pool->min_chunk(),
                                    kMaxPartials, &plan);
  if (rc != KV_OK) return rc;
  const int32_t Hkv = pool->hs.cfg.num_kv_heads;
  const int32_t n = static_cast<int32_t>(plan.items.size()) * Hkv;  // one unit per (item, kv_head), heads fastest
  for (int32_t u = 0; u < std::min(n, cap_items); ++u) {
    const WorkItem& w = plan.items[static_cast<size_t>(u / Hkv)];
    const int32_t h = u % Hkv;
    int32_t* o = out_items + 5 * u;
    o[0] = w.batch_idx; o[1] = h; o[2] = w.blk_begin; o[3] = w.n_blocks;
    o[4] = w.partial_base < 0 ? -1 : w.partial_base + h * (w.chunks >> 16) + (w.chunks & 0xffff);
  }
  if (out_n_items) *out_n_items = n;
  if (out_chunk_blocks) *out_chunk_blocks = plan.chunk_blocks;
  return KV_OK;
}

// Launch parameters common to the decode and the variable-q calls (plan staged in `s`).
static AttnParams attn_params(kv_pool_t* pool, int32_t layer, const void* q, void* out, float sm_scale,
                              const StageSlot& s, bool tc = false) {
  const kv_pool_config_t& c = pool->hs.cfg;
  const float scale = sm_scale > 0.f ? sm_scale : 1.0f / std::sqrt(static_cast<float>(c.head_dim));
  AttnParams p{};
  const int64_t layer_bytes = pool->lay.kv_bytes / c.num_layers;
  p.kv_layer = reinterpret_cast<uint16_t*>(pool->base + static_cast<int64_t>(layer) * layer_bytes);
  p.block_table = reinterpret_cast<int32_t*>(pool->base + pool->lay.block_table);
  p.bt_stride = c.max_blocks_per_request;
  p.items = reinterpret_cast<const WorkItemDev*>(s.dev);
  p.n_items = pool->plan_n_items;
  p.q = static_cast<const uint16_t*>(q);
  p.arrive = reinterpret_cast<int32_t*>(pool->base + pool->lay.arrive);
  p.fuse_combine = pool->fuse_combine ? 1 : 0;
  p.out = static_cast<uint16_t*>(out);
  p.part_o = reinterpret_cast<float*>(pool->base + pool->lay.part_o);
  p.part_ml = reinterpret_cast<float*>(pool->base + pool->lay.part_ml);
  p.counters = reinterpret_cast<int32_t*>(pool->base + pool->lay.counters);
  p.num_q_heads = c.num_q_heads;
  p.num_kv_heads = c.num_kv_heads;
  p.group = c.num_q_heads / c.num_kv_heads;
  p.scale_log2 = scale * 1.4426950408889634f;
  if (pool->tma && pool->tmap_ok) {
    p.tma_row0 = static_cast<int64_t>(layer) * (layer_bytes / 128);
    std::memcpy(p.tmap, &pool->tmap, sizeof(CUtensorMap));
  }
  if (tc) {
    p.tma_row0 = static_cast<int64_t>(layer) * (layer_bytes / 128);
    std::memcpy(p.tmap, &pool->tmap16, sizeof(CUtensorMap));
  }
  p.n_units = p.n_items * c.num_kv_heads;
  return p;
}

// a4 + a5 (and a3 when k_new / v_new are given) for layers [layer_begin, layer_begin + layer_count):
// (reserve,) plan (cached across the layers of a step), upload, one launch per layer.
static int32_t launch_attention(kv_pool_t* pool, int32_t layer_begin, int32_t layer_count, int32_t batch,
                                const int64_t* req_ids, const void* q, const void* k_new, const void* v_new, void* out,
                                int64_t q_stride, int64_t kv_stride, float sm_scale, bool reserve, void* cuda_stream) {
  if (!pool || !req_ids || !q || !out || !aligned16(q) || !aligned16(out)) return KV_ERR_INVALID;
  const kv_pool_config_t& c = pool->hs.cfg;
  if (layer_begin < 0 || layer_count < 1 || layer_begin + layer_count > c.num_layers || batch < 1) return KV_ERR_INVALID;
  if ((k_new == nullptr) != (v_new == nullptr)) return KV_ERR_INVALID;
  if (k_new && (!aligned16(k_new) || !aligned16(v_new))) return KV_ERR_INVALID;
  if (layer_count > 1 && ((q_stride & 15) != 0 || (k_new && (kv_stride & 15) != 0))) return KV_ERR_INVALID;
  if (reserve && (layer_begin != 0 || !k_new)) return KV_ERR_INVALID;
  if (!pool->has_device) return KV_ERR_NO_DEVICE;
  KV_ON_DEVICE(pool);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);

  if (reserve) {   // a1 for the step's token of every request
    if (static_cast<int32_t>(pool->ones.size()) < batch) pool->ones.assign(static_cast<size_t>(batch), 1);
    int32_t rc = pool->hs.reserve(batch, req_ids, pool->ones.data());
    if (rc != KV_OK) return rc;
  }
  auto fail = [&](int32_t rc) {
    if (reserve) pool->hs.rollback_last_reserve();
    return rc;
  };

  // plan: reuse across the layers of a step (same ids, no reserve/free since)
  const bool cached = pool->plan_slot >= 0 && pool->plan_kind == 0 && pool->plan_epoch == pool->hs.epoch &&
                      static_cast<int32_t>(pool->plan_ids.size()) == batch &&
                      std::memcmp(pool->plan_ids.data(), req_ids, sizeof(int64_t) * static_cast<size_t>(batch)) == 0;
  if (!cached) {
    pool->plan_tc = pool->tc_for(batch, req_ids);
    int32_t rc = pool->hs.plan_decode(batch, req_ids, pool->slots(false, pool->plan_tc), pool->ips(), pool->min_chunk(),
                                      kMaxPartials, &pool->plan);
    pool->plan_slot = -1;   // pool->plan no longer is what is staged
    if (rc != KV_OK) return fail(rc);
    const size_t item_bytes = pool->plan.items.size() * sizeof(WorkItem);
    const size_t comb_bytes = pool->plan.combines.size() * sizeof(CombineEntry);
    if (static_cast<int64_t>(item_bytes + comb_bytes) > pool->lay.plan_blob_bytes) return fail(KV_ERR_INVALID);
    pool->plan_append_ok = -1;
  }
  if (k_new) {  // fused append: every request's last reservation must be the one token being appended
    if (pool->plan_append_ok != 1) {
      pool->plan_append_ok = 1;
      for (int32_t i = 0; i < batch; ++i)
        if (pool->hs.reqs.find(req_ids[i])->second.last_n != 1) { pool->plan_append_ok = 0; break; }
    }
    if (!pool->plan_append_ok) return fail(KV_ERR_INVALID);
  }
  if (int32_t rc = order_attention(pool, stream); rc != KV_OK) return fail(rc);
  if (!cached) {
    StageSlot* s = nullptr;
    const int idx = acquire(pool, pool->plan_ring, &pool->plan_next, &s);
    if (idx < 0) return fail(idx);
    const size_t item_bytes = pool->plan.items.size() * sizeof(WorkItem);
    const size_t comb_bytes = pool->plan.combines.size() * sizeof(CombineEntry);
    std::memcpy(s->host, pool->plan.items.data(), item_bytes);
    std::memcpy(s->host + item_bytes, pool->plan.combines.data(), comb_bytes);
    pool->plan_slot = -1;
    pool->chain_slot = -1;
    const cudaError_t e = upload_plan(pool, *s, item_bytes + comb_bytes, stream);
    if (e != cudaSuccess) return fail(pool->cuda_fail(e));
    pool->plan_slot = idx;
    pool->plan_kind = 0;
    pool->plan_epoch = pool->hs.epoch;
    pool->plan_ids.assign(req_ids, req_ids + batch);
    pool->plan_n_items = static_cast<int32_t>(pool->plan.items.size());
    pool->plan_n_combines = static_cast<int32_t>(pool->plan.combines.size());
    pool->plan_combine_off = static_cast<int64_t>(item_bytes);
  }
  StageSlot& s = pool->plan_ring[pool->plan_slot];
  const int32_t G = c.num_q_heads / c.num_kv_heads;
  const int kind = k_new ? 1 : 0;
  const AttnVariant v = pick_variant(pool, k_new != nullptr, false, pool->plan_tc);
  const bool separate_combine = pool->plan_n_combines > 0 && !pool->fuse_combine;
  // From here on kernels are enqueued: an error is a CUDA error and leaves the stream in an undefined state
  // (KV_ERR_CUDA is sticky); the reservation stays, as the launches already issued refer to it.
  if (pool->profile) KV_CUDA(pool, pool->prof[KV_KERNEL_ATTN].begin(stream));
  for (int32_t ll = 0; ll < layer_count; ++ll) {
    AttnParams p = attn_params(pool, layer_begin + ll, static_cast<const char*>(q) + ll * q_stride,
                               static_cast<char*>(out) + ll * q_stride, sm_scale, s, pool->plan_tc);
    if (k_new) {
      p.k_new = reinterpret_cast<const uint16_t*>(static_cast<const char*>(k_new) + ll * kv_stride);
      p.v_new = reinterpret_cast<const uint16_t*>(static_cast<const char*>(v_new) + ll * kv_stride);
    }
    // the stream's previous kernel is an attention launch of this very plan and kind: its CTAs may read the work
    // items and block ids before griddepcontrol.wait
    p.chained = pool->pdl && pool->chain_slot == pool->plan_slot && pool->chain_kind == kind ? 1 : 0;
    pool->n_chained += p.chained;
    KV_CUDA(pool, launch_attn_kernel(pool, v, p, stream));
    ++pool->launches;
    pool->n_tc_launches += pool->plan_tc ? 1 : 0;
    pool->chain_slot = separate_combine ? -1 : pool->plan_slot;
    pool->chain_kind = kind;
    if (separate_combine) {
      CombineParams cp{};
      cp.entries = reinterpret_cast<const CombineEntryDev*>(s.dev + pool->plan_combine_off);
      cp.n_entries = pool->plan_n_combines;
      cp.part_o = p.part_o;
      cp.part_ml = p.part_ml;
      cp.out = p.out;
      cp.num_q_heads = c.num_q_heads;
      cp.group = G;
      cp.num_kv_heads = c.num_kv_heads;
      const unsigned cgrid = static_cast<unsigned>((static_cast<int64_t>(cp.n_entries) * c.num_q_heads + 3) / 4);
      if (pool->profile) KV_CUDA(pool, pool->prof[KV_KERNEL_COMBINE].begin(stream));
      if (c.head_dim == 128)
        combine_kernel<128><<<cgrid, 128, 0, stream>>>(cp);
      else
        combine_kernel<64><<<cgrid, 128, 0, stream>>>(cp);
      KV_CUDA(pool, cudaGetLastError());
      if (pool->profile) KV_CUDA(pool, pool->prof[KV_KERNEL_COMBINE].end(stream));
      ++pool->launches;
    }
  }
  if (pool->profile) KV_CUDA(pool, pool->prof[KV_KERNEL_ATTN].end(stream, layer_count));
  KV_CUDA(pool, cudaEventRecord(s.ev, stream));
  s.in_flight = true;
  attention_launched(pool, stream, s, kind);
  if (separate_combine) pool->chain_slot = -1;
  return KV_OK;
}

int32_t paged_decode_attention(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const void* q,
                               void* out, float sm_scale, void* cuda_stream) {
  return launch_attention(pool, layer, 1, batch, req_ids, q, nullptr, nullptr, out, 0, 0, sm_scale, false, cuda_stream);
}

int32_t paged_decode_step(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const void* q,
                          const void* k_new, const void* v_new, void* out, float sm_scale, void* cuda_stream) {
  if (!k_new || !v_new) return KV_ERR_INVALID;
  return launch_attention(pool, layer, 1, batch, req_ids, q, k_new, v_new, out, 0, 0, sm_scale, false, cuda_stream);
}

int32_t paged_decode_step_layers(kv_pool_t* pool, int32_t layer_begin, int32_t layer_count, int32_t batch,
                                 const int64_t* req_ids, const void* q, const void* k_new, const void* v_new, void* out,
                                 int64_t q_layer_stride_bytes, int64_t kv_layer_stride_bytes, float sm_scale,
                                 int32_t flags, void* cuda_stream) {
  if (flags & ~KV_STEP_RESERVE) return KV_ERR_INVALID;
  return launch_attention(pool, layer_begin, layer_count, batch, req_ids, q, k_new, v_new, out, q_layer_stride_bytes,
                          kv_layer_stride_bytes, sm_scale, (flags & KV_STEP_RESERVE) != 0, cuda_stream);
}

// a4 + a5 with the split-KV workspace in g_static_scratch: no cudaMalloc / cudaFree / allocating library call on this
// path (the plan goes through the staging slots kv_pool_create set up).  Same plan, same kernel and same merge as
// paged_decode_attention, so the same result; not profiled, not chained to its neighbours.
int64_t kv_static_scratch_bytes(void) { return kStaticScratchBytes; }

int32_t paged_decode_attention_static(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const void* q,
                                      void* out, float sm_scale, void* cuda_stream) {
  if (!pool || !req_ids || !q || !out || !aligned16(q) || !aligned16(out)) return KV_ERR_INVALID;
  const kv_pool_config_t& c = pool->hs.cfg;
  if (layer < 0 || layer >= c.num_layers || batch < 1) return KV_ERR_INVALID;
  if (!pool->has_device) return KV_ERR_NO_DEVICE;
  KV_ON_DEVICE(pool);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  unsigned char* scratch = nullptr;
  KV_CUDA(pool, static_scratch_address(pool->device, &scratch));   // set-up: once per device, pool's device current

  const bool use_tc = pool->tc_for(batch, req_ids);
  DecodePlan plan;
  int32_t rc = pool->hs.plan_decode(batch, req_ids, pool->slots(false, use_tc), pool->ips(), pool->min_chunk(),
                                    kMaxPartials, &plan);
  if (rc != KV_OK) return rc;
  if (plan.n_partials > KV_STATIC_MAX_PARTIALS) return KV_ERR_SCRATCH_LIMIT;
  const size_t item_bytes = plan.items.size() * sizeof(WorkItem);
  const size_t comb_bytes = plan.combines.size() * sizeof(CombineEntry);
  if (static_cast<int64_t>(item_bytes + comb_bytes) > pool->lay.plan_blob_bytes) return KV_ERR_INVALID;
  if (rc = order_attention(pool, stream); rc != KV_OK) return rc;

  // the staged plan of the pool's other attention calls is dropped (they re-plan), this call stages its own
  pool->plan_slot = -1;
  pool->chain_slot = -1;
  StageSlot* sp = nullptr;
  const int idx = acquire(pool, pool->plan_ring, &pool->plan_next, &sp);
  if (idx < 0) return idx;
  StageSlot& s = *sp;
  std::memcpy(s.host, plan.items.data(), item_bytes);
  std::memcpy(s.host + item_bytes, plan.combines.data(), comb_bytes);
  KV_CUDA(pool, upload_plan(pool, s, item_bytes + comb_bytes, stream));

  AttnParams p = attn_params(pool, layer, q, out, sm_scale, s, use_tc);
  p.n_items = static_cast<int32_t>(plan.items.size());
  p.n_units = p.n_items * c.num_kv_heads;
  p.arrive = reinterpret_cast<int32_t*>(scratch);
  p.part_ml = reinterpret_cast<float*>(scratch + kStaticArriveBytes);
  p.part_o = reinterpret_cast<float*>(scratch + kStaticArriveBytes + kStaticMlBytes);
  p.chained = 0;
  // the array keeps whatever the last call (of any pool) left: the arrival counters must start at zero; every
  // partial slot that is read has been written by this launch
  if (plan.n_partials > 0)
    KV_CUDA(pool, cudaMemsetAsync(scratch, 0, static_cast<size_t>(plan.n_partials) * 4, stream));
  const AttnVariant v = pick_variant(pool, false, false, use_tc);
  KV_CUDA(pool, launch_attn_kernel(pool, v, p, stream));
  ++pool->launches;
  pool->n_tc_launches += use_tc ? 1 : 0;
  if (!plan.combines.empty() && !pool->fuse_combine) {
    CombineParams cp{};
    cp.entries = reinterpret_cast<const CombineEntryDev*>(s.dev + item_bytes);
    cp.n_entries = static_cast<int32_t>(plan.combines.size());
    cp.part_o = p.part_o;
    cp.part_ml = p.part_ml;
    cp.out = p.out;
    cp.num_q_heads = c.num_q_heads;
    cp.group = c.num_q_heads / c.num_kv_heads;
    cp.num_kv_heads = c.num_kv_heads;
    const unsigned cgrid = static_cast<unsigned>((static_cast<int64_t>(cp.n_entries) * c.num_q_heads + 3) / 4);
    if (c.head_dim == 128)
      combine_kernel<128><<<cgrid, 128, 0, stream>>>(cp);
    else
      combine_kernel<64><<<cgrid, 128, 0, stream>>>(cp);
    KV_CUDA(pool, cudaGetLastError());
    ++pool->launches;
  }
  KV_CUDA(pool, cudaEventRecord(s.ev, stream));
  s.in_flight = true;
  attention_launched(pool, stream, s, 0);
  pool->chain_slot = -1;
  return KV_OK;
}

// NEXT-1: plan query tiles (cached while ids, q_lens and the pool epoch are unchanged, i.e. across
// the layers of a step), stage 48-byte items, one launch of attn_kernel<.., kVarQ = true>.
// Host half of the variable-q call: the plan for (ids, q_lens) at the pool's current epoch, reused if it is the one staged.
// No GPU work; on error nothing is staged.
static int32_t varlen_prepare(kv_pool_t* pool, int32_t batch, const int64_t* req_ids, const int32_t* q_lens, bool* cached_out) {
  const kv_pool_config_t& c = pool->hs.cfg;
  const int32_t G = c.num_q_heads / c.num_kv_heads;
  const bool cached = pool->plan_slot >= 0 && pool->plan_kind == 1 && pool->plan_epoch == pool->hs.epoch &&
                      static_cast<int32_t>(pool->plan_ids.size()) == batch &&
                      std::memcmp(pool->plan_ids.data(), req_ids, sizeof(int64_t) * static_cast<size_t>(batch)) == 0 &&
                      std::memcmp(pool->plan_qlens.data(), q_lens, sizeof(int32_t) * static_cast<size_t>(batch)) == 0;
  *cached_out = cached;
  if (!cached) {
    // a partial slot of this kernel is 8 columns wide; the workspace is sized in G-column slots
    const int32_t max_partials = static_cast<int32_t>(static_cast<int64_t>(kMaxPartials) * G / 8);
    int32_t rc = pool->hs.plan_varq(batch, req_ids, q_lens, pool->slots(true), pool->ips(), pool->min_chunk(),
                                    max_partials, &pool->plan, &pool->plan_tiles);
    pool->plan_slot = -1;   // pool->plan no longer matches what is staged
    if (rc != KV_OK) return rc;
    if (static_cast<int64_t>(pool->plan.items.size()) * 48 > pool->lay.plan_blob_bytes) return KV_ERR_TOO_LONG;
  }
  return KV_OK;
}

// Device half: stage the plan (unless cached) and launch.
static int32_t varlen_enqueue(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const int32_t* q_lens,
                              const void* q, void* out, float sm_scale, cudaStream_t stream, bool cached) {
  if (int32_t rc = order_attention(pool, stream); rc != KV_OK) return rc;
  if (!cached) {
    const size_t n_items = pool->plan.items.size();
    StageSlot* s = nullptr;
    const int idx = acquire(pool, pool->plan_ring, &pool->plan_next, &s);
    if (idx < 0) return idx;
    for (size_t k = 0; k < n_items; ++k) {
      char* dst = s->host + k * 48;
      std::memcpy(dst, &pool->plan.items[k], sizeof(WorkItem));
      const int32_t extra[4] = {pool->plan_tiles[k].pos0, pool->plan_tiles[k].n_qtok, 0, 0};
      std::memcpy(dst + sizeof(WorkItem), extra, sizeof extra);
    }
    pool->chain_slot = -1;
    KV_CUDA(pool, upload_plan(pool, *s, n_items * 48, stream));
    pool->plan_slot = idx;
    pool->plan_kind = 1;
    pool->plan_append_ok = -1;
    pool->plan_epoch = pool->hs.epoch;
    pool->plan_ids.assign(req_ids, req_ids + batch);
    pool->plan_qlens.assign(q_lens, q_lens + batch);
    pool->plan_n_items = static_cast<int32_t>(n_items);
    pool->plan_n_combines = 0;
  }
  StageSlot& s = pool->plan_ring[pool->plan_slot];
  AttnParams p = attn_params(pool, layer, q, out, sm_scale, s);
  p.chained = pool->pdl && pool->chain_slot == pool->plan_slot && pool->chain_kind == 2 ? 1 : 0;
  pool->n_chained += p.chained;
  if (pool->profile) KV_CUDA(pool, pool->prof[KV_KERNEL_VARQ].begin(stream));
  KV_CUDA(pool, launch_attn_kernel(pool, pick_variant(pool, false, true), p, stream));
  if (pool->profile) KV_CUDA(pool, pool->prof[KV_KERNEL_VARQ].end(stream));
  ++pool->launches;
  KV_CUDA(pool, cudaEventRecord(s.ev, stream));
  s.in_flight = true;
  attention_launched(pool, stream, s, 2);
  return KV_OK;
}

int32_t paged_varlen_attention(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids,
                               const int32_t* q_lens, const void* q, void* out, float sm_scale, void* cuda_stream) {
  if (!pool || !req_ids || !q_lens || !q || !out || !aligned16(q) || !aligned16(out)) return KV_ERR_INVALID;
  const kv_pool_config_t& c = pool->hs.cfg;
  if (layer < 0 || layer >= c.num_layers || batch < 1) return KV_ERR_INVALID;
  if (!pool->has_device) return KV_ERR_NO_DEVICE;
  KV_ON_DEVICE(pool);
  bool cached = false;
  if (int32_t rc = varlen_prepare(pool, batch, req_ids, q_lens, &cached); rc != KV_OK) return rc;
  return varlen_enqueue(pool, layer, batch, req_ids, q_lens, q, out, sm_scale, static_cast<cudaStream_t>(cuda_stream), cached);
}

// NEXT-1 with the new tokens' K/V written "as it goes": (a1,) a2 of this layer's rows, then the variable-q attention.
int32_t paged_varlen_step(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const int32_t* q_lens,
                          const void* q, const void* const* k_new, const void* const* v_new, void* out, float sm_scale,
                          int32_t flags, void* cuda_stream) {
  if (!pool || !req_ids || !q_lens || !q || !out || !aligned16(q) || !aligned16(out) || batch < 1) return KV_ERR_INVALID;
  if (flags & ~KV_STEP_RESERVE) return KV_ERR_INVALID;
  const bool reserve = (flags & KV_STEP_RESERVE) != 0;
  if (reserve && layer != 0) return KV_ERR_INVALID;
  int32_t rc = ingest_args_ok(pool, batch, req_ids, q_lens, k_new, v_new, layer, 1, true);
  if (rc != KV_OK) return rc;
  for (int32_t i = 0; i < batch; ++i)
    if (q_lens[i] < 1) return KV_ERR_INVALID;
  KV_ON_DEVICE(pool);
  rc = reserve ? pool->hs.reserve(batch, req_ids, q_lens)         // a1: the q_lens[i] new tokens of every request
               : pool->hs.check_batch(batch, req_ids, q_lens);    // reserved by the caller / by this step's layer 0
  if (rc != KV_OK) return rc;
  auto fail = [&](int32_t e) {
    if (reserve) pool->hs.rollback_last_reserve();
    return e;
  };
  bool cached = false;                                           // the attention's plan first: nothing is enqueued if it fails
  if (rc = varlen_prepare(pool, batch, req_ids, q_lens, &cached); rc != KV_OK) return fail(rc);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  std::vector<int32_t> start(static_cast<size_t>(batch));
  for (int32_t i = 0; i < batch; ++i) start[static_cast<size_t>(i)] = pool->hs.reqs.find(req_ids[i])->second.len - q_lens[i];
  rc = run_copy(pool, CopyKind::kScatter, nullptr, nullptr, batch, req_ids, q_lens, k_new, v_new, start.data(), layer, 1, stream);
  if (rc != KV_OK) return fail(rc);
  // from here on work is enqueued: the reservation stays (as in paged_decode_step_layers)
  return varlen_enqueue(pool, layer, batch, req_ids, q_lens, q, out, sm_scale, stream, cached);
}

int32_t kv_ingest_host(kv_pool_t* pool, int32_t n_req, const int64_t* req_ids, const int32_t* n_tokens,
                       const void* const* k_src, const void* const* v_src, int32_t layer_begin, int32_t layer_count,
                       void* staging, int64_t staging_bytes, void* cuda_stream) {
  int32_t rc = ingest_args_ok(pool, n_req, req_ids, n_tokens, k_src, v_src, layer_begin, layer_count, false);
  if (rc != KV_OK) return rc;
  const kv_pool_config_t& c = pool->hs.cfg;
  if (n_req > 0 && (!staging || (reinterpret_cast<uintptr_t>(staging) & (kAlign - 1)) != 0)) return KV_ERR_INVALID;
  const int64_t row_bytes = static_cast<int64_t>(layer_count) * pool->src_heads() * c.head_dim * 2;   // full-width source rows
  int64_t need = 0;
  for (int32_t i = 0; i < n_req; ++i) need += 2 * align_up(row_bytes * n_tokens[i]);
  if (need > staging_bytes) return KV_ERR_INVALID;
  KV_ON_DEVICE(pool);
  // a1 first: a call that cannot get its blocks must not have touched the stream
  rc = layer_begin == 0 ? pool->hs.reserve(n_req, req_ids, n_tokens) : pool->hs.check_batch(n_req, req_ids, n_tokens);
  if (rc != KV_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  std::vector<const void*> kd(static_cast<size_t>(n_req)), vd(static_cast<size_t>(n_req));
  // Zero-copy: when every source is pinned host memory the device can address (cudaHostAlloc / cudaHostRegister
  // under unified addressing) and 16-byte aligned, the scatter kernel reads it over PCIe itself — the KV crosses the
  // bus once, straight into its blocks, with no staging pass and no copy engine serialised in front of the kernel.
  bool direct = pool->host_zero_copy;
  for (int32_t i = 0; i < n_req && direct; ++i) {
    if (n_tokens[i] == 0) { kd[static_cast<size_t>(i)] = vd[static_cast<size_t>(i)] = nullptr; continue; }
    for (int pass = 0; pass < 2 && direct; ++pass) {
      cudaPointerAttributes pa{};
      const void* hp = pass ? v_src[i] : k_src[i];
      if (cudaPointerGetAttributes(&pa, hp) != cudaSuccess) { cudaGetLastError(); direct = false; break; }
      if (pa.type != cudaMemoryTypeHost || !pa.devicePointer || !aligned16(pa.devicePointer)) { direct = false; break; }
      (pass ? vd : kd)[static_cast<size_t>(i)] = pa.devicePointer;
    }
  }
  ++(direct ? pool->n_zero_copy : pool->n_staged);
  if (direct) return ingest_reserved(pool, n_req, req_ids, n_tokens, kd.data(), vd.data(), layer_begin, layer_count, stream);
  // Staged: the copy engine brings the sources into the caller's staging buffer (request after request, K then V,
  // each at a 256-byte aligned offset) on a stream the pool owns, in groups of requests; the scatter of a group is
  // enqueued on the caller's stream behind that group's copies, so it runs while the next group crosses the bus.
  // (A copy-engine transfer moves ~55 GB/s over PCIe 5 x16 where SM loads of pinned memory reach ~48: option
  // host_zero_copy = 0 selects this form for pinned sources too.)
  char* const stage0 = static_cast<char*>(staging);
  std::vector<int64_t> off(static_cast<size_t>(n_req) + 1, 0);
  for (int32_t i = 0; i < n_req; ++i) off[static_cast<size_t>(i) + 1] = off[static_cast<size_t>(i)] + 2 * align_up(row_bytes * n_tokens[i]);
  const int64_t total = off[static_cast<size_t>(n_req)];
  const int64_t group_bytes = std::max<int64_t>(64LL << 20, (total + kv_pool::kStageGroups - 1) / kv_pool::kStageGroups);
  cudaStream_t cs = pool->copy_stream;
  cudaError_t ce = cudaSuccess;
  if (pool->stage_busy) ce = cudaStreamWaitEvent(cs, pool->stage_ev, 0);   // the previous call's scatters have read the buffer
  // what precedes this call on the caller's stream may be what made `staging` available: order the copies behind it
  if (ce == cudaSuccess) ce = cudaEventRecord(pool->grp_ev[0], stream);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(cs, pool->grp_ev[0], 0);
  int32_t launched = 0;
  int g = 0;
  for (int32_t i0 = 0; i0 < n_req && ce == cudaSuccess;) {
    int32_t i1 = i0;
    while (i1 < n_req && (i1 == i0 || off[static_cast<size_t>(i1) + 1] - off[static_cast<size_t>(i0)] <= group_bytes)) ++i1;
    for (int32_t i = i0; i < i1 && ce == cudaSuccess; ++i) {
      const int64_t bytes = row_bytes * n_tokens[i];
      char* kdst = stage0 + off[static_cast<size_t>(i)];
      char* vdst = kdst + align_up(bytes);
      kd[static_cast<size_t>(i)] = kdst;
      vd[static_cast<size_t>(i)] = vdst;
      if (bytes == 0) continue;
      // pieces of 8 MiB: a small copy another stream hands to the same copy engine (a decode step's q) waits for
      // ~150 us at most, not for a whole request
      constexpr int64_t kPiece = 8LL << 20;
      for (int pass = 0; pass < 2 && ce == cudaSuccess; ++pass) {
        char* dstp = pass ? vdst : kdst;
        const char* srcp = static_cast<const char*>(pass ? v_src[i] : k_src[i]);
        for (int64_t o = 0; o < bytes && ce == cudaSuccess; o += kPiece)
          ce = cudaMemcpyAsync(dstp + o, srcp + o, static_cast<size_t>(std::min(kPiece, bytes - o)), cudaMemcpyHostToDevice, cs);
      }
    }
    if (ce == cudaSuccess) ce = cudaEventRecord(pool->grp_ev[g], cs);
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(stream, pool->grp_ev[g], 0);
    if (ce != cudaSuccess) break;
    const int32_t n = i1 - i0;
    const size_t o = static_cast<size_t>(i0);
    std::vector<int32_t> start(static_cast<size_t>(n));
    for (int32_t i = 0; i < n; ++i) start[static_cast<size_t>(i)] = pool->hs.reqs.find(req_ids[o + i])->second.len - n_tokens[o + i];
    rc = run_copy(pool, CopyKind::kScatter, nullptr, nullptr, n, req_ids + o, n_tokens + o, kd.data() + o, vd.data() + o, start.data(),
                  layer_begin, layer_count, stream);
    if (rc != KV_OK) {
      // nothing of this call has been launched yet: the reservation can go back; otherwise the error is a CUDA error
      // on a stream that already carries part of the call (KV_ERR_CUDA is sticky)
      if (launched == 0 && layer_begin == 0) pool->hs.rollback_last_reserve();
      return rc;
    }
    ++launched;
    g = (g + 1) % kv_pool::kStageGroups;
    i0 = i1;
  }
  if (ce == cudaSuccess && n_req > 0) {
    ce = cudaEventRecord(pool->stage_ev, stream);
    pool->stage_busy = ce == cudaSuccess;
  }
  if (ce != cudaSuccess) {
    if (launched == 0 && layer_begin == 0) pool->hs.rollback_last_reserve();
    return pool->cuda_fail(ce);
  }
  return KV_OK;
}

static int32_t attention_host(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const void* q,
                              const void* k_new, const void* v_new, void* out, float sm_scale, void* staging,
                              int64_t staging_bytes, void* cuda_stream) {
  if (!pool || !req_ids || !q || !out || !staging || batch < 1) return KV_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(staging) & (kAlign - 1)) != 0) return KV_ERR_INVALID;
  if (!pool->has_device) return KV_ERR_NO_DEVICE;
  const kv_pool_config_t& c = pool->hs.cfg;
  const int64_t qb = static_cast<int64_t>(batch) * c.num_q_heads * c.head_dim * 2;
  const int64_t kb = k_new ? static_cast<int64_t>(batch) * c.num_kv_heads * c.head_dim * 2 : 0;
  if (2 * align_up(qb) + 2 * align_up(kb) > staging_bytes) return KV_ERR_INVALID;
  {  // validate the batch before any copy is issued, so an error leaves the stream untouched
    int32_t rc = pool->hs.check_batch(batch, req_ids, nullptr);
    if (rc != KV_OK) return rc;
    for (int32_t i = 0; i < batch; ++i) {
      const Request& r = pool->hs.reqs.find(req_ids[i])->second;
      if (r.len < 1 || (k_new && r.last_n != 1)) return KV_ERR_INVALID;
    }
  }
  KV_ON_DEVICE(pool);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  char* dq = static_cast<char*>(staging);
  char* dout = dq + align_up(qb);
  char* dk = dout + align_up(qb);
  char* dv = dk + align_up(kb);
  KV_CUDA(pool, cudaMemcpyAsync(dq, q, static_cast<size_t>(qb), cudaMemcpyHostToDevice, stream));
  if (k_new) {
    KV_CUDA(pool, cudaMemcpyAsync(dk, k_new, static_cast<size_t>(kb), cudaMemcpyHostToDevice, stream));
    KV_CUDA(pool, cudaMemcpyAsync(dv, v_new, static_cast<size_t>(kb), cudaMemcpyHostToDevice, stream));
  }
  int32_t rc = launch_attention(pool, layer, 1, batch, req_ids, dq, k_new ? dk : nullptr, k_new ? dv : nullptr, dout, 0, 0,
                                sm_scale, false, cuda_stream);
  if (rc != KV_OK) return rc;
  KV_CUDA(pool, cudaMemcpyAsync(out, dout, static_cast<size_t>(qb), cudaMemcpyDeviceToHost, stream));
  pool->chain_slot = -1;   // a copy now sits between this launch and the next
  return KV_OK;
}

int32_t paged_decode_attention_host(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids,
                                    const void* q, void* out, float sm_scale, void* staging, int64_t staging_bytes,
                                    void* cuda_stream) {
  return attention_host(pool, layer, batch, req_ids, q, nullptr, nullptr, out, sm_scale, staging, staging_bytes,
                        cuda_stream);
}

int32_t paged_decode_step_host(kv_pool_t* pool, int32_t layer, int32_t batch, const int64_t* req_ids, const void* q,
                               const void* k_new, const void* v_new, void* out, float sm_scale, void* staging,
                               int64_t staging_bytes, void* cuda_stream) {
  if (!k_new || !v_new) return KV_ERR_INVALID;
  return attention_host(pool, layer, batch, req_ids, q, k_new, v_new, out, sm_scale, staging, staging_bytes,
                        cuda_stream);
}

int32_t kv_capacity(const kv_capacity_model_t* m, kv_capacity_t* out) {
  if (!m || !out) return KV_ERR_INVALID;
  const bool ok = m->m_gpu > 0 && m->m_reserved >= 0 && m->m_model >= 0 && m->tp >= 1 && m->bw > 0 && m->alpha > 0 &&
                  m->alpha <= 1.5 && m->t_d_slo > 0 && m->isl >= 0 && m->osl > 0 && m->m_token > 0;
  if (!ok) return KV_ERR_INVALID;   // NaNs fail every comparison above
  kv_capacity_t r{};
  r.v_mem = (m->m_gpu - m->m_reserved) * m->tp - m->m_model;          // Eq. 11
  r.v_bw = m->t_d_slo * m->alpha * m->tp * m->bw;                     // Eq. 12
  r.bandwidth_bound = r.v_bw < r.v_mem ? 1 : 0;
  const double v = r.v_bw < r.v_mem ? r.v_bw : r.v_mem;
  r.cc_d = v > 0 ? v / ((m->isl + m->osl / 2) * m->m_token) : 0.0;    // Eq. 13
  *out = r;
  return KV_OK;
}

int32_t kv_optimal_pd_ratio(double cc_d, double t_p, double t_d, double osl, double* out_ratio) {
  if (!out_ratio || !(cc_d > 0) || !(t_p > 0) || !(t_d > 0) || !(osl > 0)) return KV_ERR_INVALID;
  *out_ratio = cc_d * t_p / (t_d * osl);                              // Eq. 14 solved for n_p / n_d
  return KV_OK;
}

int64_t kv_token_bytes(const kv_pool_config_t* cfg) {
  if (!cfg) return KV_ERR_INVALID;
  int32_t rc = HostState::validate(*cfg);
  if (rc != KV_OK) return rc;
  const int64_t per_head = cfg->kv_dtype == KV_DTYPE_FP8_E4M3 ? 2LL * cfg->head_dim + 8 : 2LL * cfg->head_dim * 2;
  return static_cast<int64_t>(cfg->num_layers) * cfg->num_kv_heads * per_head;
}

int64_t kv_launch_count(const kv_pool_t* pool) { return pool ? pool->launches : KV_ERR_INVALID; }

int64_t kv_pool_counter(const kv_pool_t* pool, const char* name) {
  if (!pool || !name) return KV_ERR_INVALID;
  if (!std::strcmp(name, "launches")) return pool->launches;
  if (!std::strcmp(name, "plans_uploaded")) return pool->n_plans;
  if (!std::strcmp(name, "attn_chained_launches")) return pool->n_chained;
  if (!std::strcmp(name, "attn_stream_switches")) return pool->n_stream_switch;
  if (!std::strcmp(name, "host_ingest_zero_copy")) return pool->n_zero_copy;
  if (!std::strcmp(name, "host_ingest_staged")) return pool->n_staged;
  if (!std::strcmp(name, "attn_tc_launches")) return pool->n_tc_launches;
  return KV_ERR_INVALID;
}

int32_t kv_pool_set_option(kv_pool_t* pool, const char* key, int64_t value) {
  if (!pool || !key) return KV_ERR_INVALID;
  pool->plan_slot = -1;  // any option may change the plan
  pool->chain_slot = -1;
  if (!std::strcmp(key, "min_chunk_blocks") && value >= 1 && value <= 65536) { pool->min_chunk_blocks = static_cast<int32_t>(value); pool->min_chunk_set = true; return KV_OK; }
  if (!std::strcmp(key, "ctas_per_sm") && value >= 0 && value <= 8) { pool->ctas_per_sm = static_cast<int32_t>(value); return KV_OK; }
  if (!std::strcmp(key, "items_per_slot") && value >= 1 && value <= 1024) { pool->items_per_slot = static_cast<int32_t>(value); pool->items_per_slot_set = true; return KV_OK; }
  if (!std::strcmp(key, "profile") && (value == 0 || value == 1)) { pool->profile = value != 0; return KV_OK; }
  if (!std::strcmp(key, "fuse_combine") && (value == 0 || value == 1)) { pool->fuse_combine = value != 0; return KV_OK; }
  if (!std::strcmp(key, "pdl") && (value == 0 || value == 1)) { pool->pdl = value != 0; return KV_OK; }
  if (!std::strcmp(key, "side_upload") && (value == 0 || value == 1)) { pool->side_upload = value != 0; return KV_OK; }
  if (!std::strcmp(key, "tc") && value >= 0 && value <= 2) {   // FP8, head_dim 128 pools with a device slab only
    if (value == 1 && !pool->tmap16_ok) return KV_ERR_UNSUPPORTED;
    pool->tc = static_cast<int32_t>(value);
    pool->plan_slot = -1;                                         // the planner sizes chunks for the kernel that runs
    return KV_OK;
  }
  if (!std::strcmp(key, "tma") && (value == 0 || value == 1)) {   // bf16, head_dim 128 pools with a device slab only
    if (value == 1 && !pool->tmap_ok) return KV_ERR_UNSUPPORTED;
    pool->tma = value != 0;
    return KV_OK;
  }
  if (!std::strcmp(key, "host_zero_copy") && (value == 0 || value == 1)) { pool->host_zero_copy = value != 0; return KV_OK; }
  if (!std::strcmp(key, "ring") && (value == 2 || value == 3)) { pool->ring = static_cast<int32_t>(value); return KV_OK; }
  if (!std::strcmp(key, "src_kv_heads") && (value == 0 || (value >= pool->hs.cfg.num_kv_heads + pool->src_head_begin && value <= 65536))) {
    pool->src_kv_heads = static_cast<int32_t>(value);
    if (value == 0) pool->src_head_begin = 0;
    return KV_OK;
  }
  if (!std::strcmp(key, "src_head_begin") && value >= 0 && value + pool->hs.cfg.num_kv_heads <= pool->src_heads()) {
    pool->src_head_begin = static_cast<int32_t>(value);
    return KV_OK;
  }
  return KV_ERR_INVALID;
}

int32_t kv_profile_read(kv_pool_t* pool, int32_t kind, int64_t* out_launches, double* out_ms) {
  if (!pool || kind < 0 || kind >= KV_KERNEL_KINDS) return KV_ERR_INVALID;
  KV_ON_DEVICE(pool);
  ProfRing& r = pool->prof[kind];
  KV_CUDA(pool, r.drain());
  if (out_launches) *out_launches = r.launches;
  if (out_ms) *out_ms = r.ms;
  return KV_OK;
}

int32_t kv_profile_reset(kv_pool_t* pool) {
  if (!pool) return KV_ERR_INVALID;
  KV_ON_DEVICE(pool);
  for (ProfRing& r : pool->prof) {
    KV_CUDA(pool, r.drain());
    r.launches = 0;
    r.ms = 0.0;
  }
  return KV_OK;
}

int32_t kv_last_cuda_error(const kv_pool_t* pool) { return pool ? pool->last_cuda : KV_ERR_INVALID; }

const char* kv_strerror(int32_t status) {
  switch (status) {
    case KV_OK: return "ok";
    case KV_ERR_INVALID: return "invalid argument";
    case KV_ERR_NO_BLOCKS: return "KV pool exhausted (nothing changed)";
    case KV_ERR_UNKNOWN_REQUEST: return "unknown request id";
    case KV_ERR_TOO_LONG: return "request exceeds max_blocks_per_request";
    case KV_ERR_TOO_MANY_REQUESTS: return "more than max_requests live requests";
    case KV_ERR_CUDA: return "CUDA runtime error (see kv_last_cuda_error)";
    case KV_ERR_NO_DEVICE: return "pool has no device slab (host-only)";
    case KV_ERR_UNSUPPORTED: return "call not available for this pool's kv_dtype";
    case KV_ERR_SCRATCH_LIMIT: return "split-KV plan needs more partial slots than the static scratch holds (KV_STATIC_MAX_PARTIALS)";
    default: return "unknown status";
  }
}

const char* kv_version(void) { return "0.2.0"; }

}  // extern "C"
