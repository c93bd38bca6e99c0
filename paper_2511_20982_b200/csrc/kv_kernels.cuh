// kv_kernels.cuh — sm_100a kernels of the D-instance KV path.
//
//   ingest_kernel<D, kGather>   a2/a3 (and its inverse): contiguous [L][Hkv][n][d] <-> paged blocks
//   attn_splitkv_kernel<D,..>   a4 (+ a3, a5): split-KV paged attention, one warp per work item, KV tiles in REGISTER
//                               buffers — the round's first design, kept behind option ring = 0.  The default kernel,
//                               attn_ring_kernel (kv_attn_ring.cuh), shares everything below except the staging.
//   combine_kernel<D>           a5: log-sum-exp merge of split-KV partials (stand-alone form, option fuse_combine = 0)
//
// Both data-moving kernels are HBM-bound (0 and G <= 8 flop/byte), so the design
// targets bytes in flight, sector-exact 16-byte accesses and no re-reads; tensor cores
// (mma.sync m16n8k16 bf16, SASS HMMA) are used only to keep the ALUs out of the way:
//
// attn_splitkv_kernel — register-direct tiles.  A KV tile is one (block, kv_head): K[16][D] then
// V[16][D] bf16, 8 KiB contiguous at D = 128.  The MMAs are arranged with the 16 TOKENS of a
// block on M and the (<= 8) query heads of the GQA group on N:
//     S^T[16 tok x 8 heads] = K[16 x D] . q^T[D x 8]            D/16 MMAs, A = K straight from HBM
//     O^T[D x 8 heads]     += V^T[D x 16 tok] . P^T[16 x 8]     D/16 MMAs, B = P^T via movmatrix
// Because a dot product does not care in which order the contraction index is visited, each
// thread may feed the k-slots of its A fragment from ANY d-columns as long as the q fragment
// uses the same ones: thread (g = lane/4, c = lane%4) loads 16 contiguous bytes (8 bf16) of K
// row g at column chunk c + 4j and uses them for k-steps 2j and 2j+1.  Likewise the m index of
// O^T (the d column) may be permuted freely and is un-permuted when the result is stored.  So
// every global load is a 16-byte vector whose bytes all land in MMA fragment registers: no
// shared-memory staging, no ldmatrix, no barriers, no bank conflicts.  V needs its pairs along
// the token axis, which costs 4 PRMT per m-tile.  Two tiles (16 KiB) are in flight per warp.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace kvp {

constexpr int kBlockSize = 16;     // tokens per KV block (BASELINE.json: block size 16)
constexpr int kAttnThreads = 128;  // 4 warps per CTA, each an independent split-KV worker
constexpr int kAttnWarps = kAttnThreads / 32;
constexpr int kIngestThreads = 256;
constexpr int kIngestWarps = kIngestThreads / 32;

// ---------------------------------------------------------------------------------------------
// small PTX wrappers
// ---------------------------------------------------------------------------------------------

// 16-byte streaming load through the read-only path, not allocated in L1; zero if !pred.
__device__ __forceinline__ uint4 ldg_stream_pred(const void* ptr, bool pred) {
  uint4 r = make_uint4(0u, 0u, 0u, 0u);
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t"
      "@p ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];\n\t}"
      : "+r"(r.x), "+r"(r.y), "+r"(r.z), "+r"(r.w)
      : "l"(ptr), "r"(static_cast<int>(pred)));
  return r;
}

// Same, but an ordinary (weak) load: ptxas may not move it across the stores of a copy loop,
// so "all loads, then all stores" survives scheduling and keeps 16 x 16 B in flight per lane.
// (.nc loads were interleaved with the stores by ptxas, cutting the loads in flight to ~4.)
__device__ __forceinline__ uint4 ldg_copy_pred(const void* ptr, bool pred) {
  uint4 r = make_uint4(0u, 0u, 0u, 0u);
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t"
      "@p ld.global.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];\n\t}"
      : "+r"(r.x), "+r"(r.y), "+r"(r.z), "+r"(r.w)
      : "l"(ptr), "r"(static_cast<int>(pred))
      : "memory");
  return r;
}

__device__ __forceinline__ uint4 ldg_stream(const void* ptr) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(ptr));
  return r;
}

__device__ __forceinline__ void stg_stream_pred(void* ptr, const uint4& v, bool pred) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t"
      "@p st.global.L1::no_allocate.v4.u32 [%0], {%1, %2, %3, %4};\n\t}"
      :
      : "l"(ptr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "r"(static_cast<int>(pred))
      : "memory");
}

// D(16x8, f32) += A(16x16, bf16, row) * B(16x8, bf16, col)
__device__ __forceinline__ void mma_bf16_m16n8k16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                                  uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// warp-wide transpose of an 8x8 matrix of 16-bit elements held one row-pair per thread
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// (a.lo16, b.lo16) / (a.hi16, b.hi16): pair up one bf16 from each of two registers
__device__ __forceinline__ uint32_t pair_lo(uint32_t a, uint32_t b) { return __byte_perm(a, b, 0x5410); }
__device__ __forceinline__ uint32_t pair_hi(uint32_t a, uint32_t b) { return __byte_perm(a, b, 0x7632); }

__device__ __forceinline__ uint32_t u4_get(const uint4& v, int i) {
  return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w));
}

// ---------------------------------------------------------------------------------------------
// a2 / a3 KV ingest and its inverse
// ---------------------------------------------------------------------------------------------

// One request of an ingest/gather launch.  Units of request i are
// [unit_begin, unit_begin + n_touched * layer_count * Hkv), ordered (layer, head, touched block)
// with the touched block fastest, so consecutive warps stream consecutive source runs.
struct IngestReq {
  uint64_t k_src, v_src;  // device addresses of the contiguous [layer_count][Hkv][n_tokens][D] tensors
  int64_t unit_begin;
  int32_t n_tokens, start_pos, slot;
  int32_t blk0;       // first touched logical block = start_pos / 16
  int32_t n_touched;  // logical blocks touched by [start_pos, start_pos + n_tokens)
  int32_t blk_off;    // index of this request's first touched physical id in the id array
};
static_assert(sizeof(IngestReq) == 48, "IngestReq layout is shared with the host serialiser");

struct IngestParams {
  const IngestReq* reqs;     // device
  const int32_t* blk_ids;    // device: touched physical block ids, request after request
  int32_t n_req;
  int64_t total_units;
  uint16_t* kv;              // KV region base
  int32_t* block_table;      // device mirror [max_requests][bt_stride]
  int32_t bt_stride;
  int32_t layer_begin, layer_count, num_kv_heads;
  int64_t num_blocks;
  // KV-head sharding: the contiguous side is [layer_count][src_kv_heads][n][D] and this
  // pool's head h is its head src_head_begin + h.  Unsharded: src_kv_heads = num_kv_heads, src_head_begin = 0.
  int32_t src_kv_heads, src_head_begin;
};

template <int D, bool kGather>
__global__ void __launch_bounds__(kIngestThreads) ingest_kernel(const IngestParams p) {
  constexpr int kPiecesPerRow = D / 8;                       // 16-byte pieces per token row
  constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;  // 8 at D=128, 4 at D=64
  const int lane = threadIdx.x & 31;
  const int64_t u = static_cast<int64_t>(blockIdx.x) * kIngestWarps + (threadIdx.x >> 5);
  if (u >= p.total_units) return;

  // request of this unit: last i with unit_begin <= u.  The lanes test 32 candidates at a time (independent
  // loads, one ballot each) rather than walk a binary search of dependent loads.
  int lo = -1;
  for (int base = 0; base < p.n_req; base += 32) {
    const int i = base + lane;
    const bool le = i < p.n_req && __ldg(&p.reqs[i].unit_begin) <= u;
    lo += __popc(__ballot_sync(0xffffffffu, le));
  }
  const IngestReq r = p.reqs[lo];
  const int64_t local = u - r.unit_begin;
  const int jj = static_cast<int>(local % r.n_touched);
  const int rest = static_cast<int>(local / r.n_touched);
  const int h = rest % p.num_kv_heads;
  const int ll = rest / p.num_kv_heads;
  const int blk = __ldg(&p.blk_ids[r.blk_off + jj]);
  const int lb = r.blk0 + jj;                                 // logical block
  const int row0 = (jj == 0) ? (r.start_pos & (kBlockSize - 1)) : 0;
  const int row1 = min(kBlockSize, r.start_pos + r.n_tokens - lb * kBlockSize);
  const int t0 = lb * kBlockSize + row0 - r.start_pos;        // first source token of this unit
  const int pieces = (row1 - row0) * kPiecesPerRow;

  // rows row0..row1-1 are contiguous both in the source run and inside the block
  const int64_t src_off = ((static_cast<int64_t>(ll) * p.src_kv_heads + p.src_head_begin + h) * r.n_tokens + t0) * D;
  const int64_t dst_off =
      ((((static_cast<int64_t>(p.layer_begin + ll) * p.num_blocks + blk) * p.num_kv_heads + h) * 2) * kBlockSize +
       row0) * D;
  const uint4* lin_k = reinterpret_cast<const uint4*>(reinterpret_cast<const uint16_t*>(r.k_src) + src_off);
  const uint4* lin_v = reinterpret_cast<const uint4*>(reinterpret_cast<const uint16_t*>(r.v_src) + src_off);
  uint4* pag_k = reinterpret_cast<uint4*>(p.kv + dst_off);
  uint4* pag_v = reinterpret_cast<uint4*>(p.kv + dst_off + kBlockSize * D);

  uint4 bk[kMaxPerLane], bv[kMaxPerLane];
#pragma unroll
  for (int i = 0; i < kMaxPerLane; ++i) {                     // all loads first: 16 x 16 B in flight per lane
    const int idx = lane + 32 * i;
    const bool ok = idx < pieces;
    bk[i] = ldg_copy_pred((kGather ? pag_k : lin_k) + idx, ok);
    bv[i] = ldg_copy_pred((kGather ? pag_v : lin_v) + idx, ok);
  }
#pragma unroll
  for (int i = 0; i < kMaxPerLane; ++i) {
    const int idx = lane + 32 * i;
    const bool ok = idx < pieces;
    stg_stream_pred(const_cast<uint4*>(kGather ? lin_k : pag_k) + idx, bk[i], ok);
    stg_stream_pred(const_cast<uint4*>(kGather ? lin_v : pag_v) + idx, bv[i], ok);
  }
  if (!kGather && ll == 0 && h == 0 && lane == 0)             // device block_table mirror (a1, device half)
    p.block_table[static_cast<int64_t>(r.slot) * p.bt_stride + lb] = blk;
}

// ---------------------------------------------------------------------------------------------
// a4 split-KV paged decode attention
// ---------------------------------------------------------------------------------------------

struct WorkItemDev {  // == kvp::WorkItem (kv_host.h); one item = num_kv_heads units, heads fastest
  int32_t batch_idx, slot, blk_begin, n_blocks, n_tokens, partial_base, chunks, last_blk;
};

struct AttnParams {
  uint16_t* kv_layer;          // &kv[layer][0]...  (written only by the fused append)
  int32_t* block_table;        // device mirror (written only by the fused append)
  int32_t bt_stride;
  const WorkItemDev* items;
  int32_t n_items, n_units;    // n_units = n_items * num_kv_heads
  const uint16_t* q;
  const uint16_t* k_new;       // fused decode step: [batch][Hkv][D] rows of the token being appended
  const uint16_t* v_new;
  uint16_t* out;
  float* part_o;               // [n_partials][G][D]  un-normalised
  float* part_ml;              // [n_partials][G][2]  (m in log2 units, l)
  int32_t* counters;           // [0] next work item, [1] finished CTAs
  int32_t* arrive;             // per split (request, kv_head): chunks finished (fused combine); self-resetting
  int32_t num_q_heads, num_kv_heads, group;
  int32_t fuse_combine;
  float scale_log2;            // sm_scale * log2(e)
};

template <int D>
struct KVTile {
  uint4 k[2][D / 32];  // rows g, g+8; column chunks c + 4j
  uint4 v[4][D / 64];  // rows 2c, 2c+1, 2c+8, 2c+9; column chunks g + 8cs
};

template <int D>
__device__ __forceinline__ void load_tile(KVTile<D>& T, const uint16_t* tile, int nv, int g, int c) {
  const uint16_t* kp = tile + g * D + c * 8;
#pragma unroll
  for (int rs = 0; rs < 2; ++rs) {
    const bool ok = g + 8 * rs < nv;
#pragma unroll
    for (int j = 0; j < D / 32; ++j) T.k[rs][j] = ldg_stream_pred(kp + rs * 8 * D + j * 32, ok);
  }
  const uint16_t* vp = tile + kBlockSize * D + g * 8;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = 2 * c + (i & 1) + 8 * (i >> 1);
    const bool ok = row < nv;
#pragma unroll
    for (int cs = 0; cs < D / 64; ++cs) T.v[i][cs] = ldg_stream_pred(vp + row * D + cs * 64, ok);
  }
}

// Fused decode step (a3 inside a4): the request's last tile with the row of the token being
// appended (r_new = nv - 1) taken from k_new / v_new instead of the pool.  Same lanes, same
// registers as load_tile, so the MMAs downstream do not know the difference.
template <int D>
__device__ __forceinline__ void load_tile_append(KVTile<D>& T, const uint16_t* tile, const uint16_t* k_new,
                                                 const uint16_t* v_new, int nv, int g, int c) {
  const int r_new = nv - 1;
#pragma unroll
  for (int rs = 0; rs < 2; ++rs) {
    const int row = g + 8 * rs;
    const uint16_t* kp = (row == r_new ? k_new : tile + row * D) + c * 8;
#pragma unroll
    for (int j = 0; j < D / 32; ++j) T.k[rs][j] = ldg_stream_pred(kp + j * 32, row < nv);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = 2 * c + (i & 1) + 8 * (i >> 1);
    const uint16_t* vp = (row == r_new ? v_new : tile + kBlockSize * D + row * D) + g * 8;
#pragma unroll
    for (int cs = 0; cs < D / 64; ++cs) T.v[i][cs] = ldg_stream_pred(vp + cs * 64, row < nv);
  }
}

// ... and the append itself: the lanes that hold row r_new write it into the pool tile (a3).
template <int D>
__device__ __forceinline__ void store_new_row(const KVTile<D>& T, uint16_t* tile, int nv, int g, int c) {
  const int r_new = nv - 1;
#pragma unroll
  for (int rs = 0; rs < 2; ++rs) {
    if (g + 8 * rs == r_new) {
      uint16_t* kp = tile + r_new * D + c * 8;
#pragma unroll
      for (int j = 0; j < D / 32; ++j) *reinterpret_cast<uint4*>(kp + j * 32) = T.k[rs][j];
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (2 * c + (i & 1) + 8 * (i >> 1) == r_new) {
      uint16_t* vp = tile + kBlockSize * D + r_new * D + g * 8;
#pragma unroll
      for (int cs = 0; cs < D / 64; ++cs) *reinterpret_cast<uint4*>(vp + cs * 64) = T.v[i][cs];
    }
  }
}

// a5 for query heads [head0, head0 + NH) of one (request, kv head): out = sum_c 2^(m_c - M) O_c /
// sum_c 2^(m_c - M) l_c over the n_chunks partials starting at partial slot pb (one slot per chunk).
// One warp; lane owns D/32 columns of every head.  The merge is a running (online) one so the
// loads of all heads and of several chunks are independent and in flight together — this code is
// pure latency, it runs on warps that would otherwise be streaming KV.  Loads bypass L1 (.cg):
// the partials were written by other SMs, possibly earlier in this same kernel.
template <int D, int NH>
__device__ __forceinline__ void combine_heads(const float* part_o, const float* part_ml, int pb, int n_chunks,
                                              int G, int head0, uint16_t* out_row0, int lane) {
  constexpr int V = D / 32;
  const float* ml = part_ml + (static_cast<int64_t>(pb) * G + head0) * 2;
  const int64_t ml_stride = static_cast<int64_t>(G) * 2;
  const float* po = part_o + (static_cast<int64_t>(pb) * G + head0) * D + lane * V;
  const int64_t po_stride = static_cast<int64_t>(G) * D;
  float M[NH], den[NH], acc[NH][V];
#pragma unroll
  for (int hh = 0; hh < NH; ++hh) {
    M[hh] = -INFINITY; den[hh] = 0.f;
#pragma unroll
    for (int k = 0; k < V; ++k) acc[hh][k] = 0.f;
  }
#pragma unroll 2
  for (int ch = 0; ch < n_chunks; ++ch) {
    float2 mlv[NH];
    float x[NH][V];
#pragma unroll
    for (int hh = 0; hh < NH; ++hh) {
      mlv[hh] = __ldcg(reinterpret_cast<const float2*>(ml + ch * ml_stride + hh * 2));
      if constexpr (V == 4) {
        const float4 t = __ldcg(reinterpret_cast<const float4*>(po + ch * po_stride + hh * D));
        x[hh][0] = t.x; x[hh][1] = t.y; x[hh][2] = t.z; x[hh][3] = t.w;
      } else {
        const float2 t = __ldcg(reinterpret_cast<const float2*>(po + ch * po_stride + hh * D));
        x[hh][0] = t.x; x[hh][1] = t.y;
      }
    }
#pragma unroll
    for (int hh = 0; hh < NH; ++hh) {
      const float mn = fmaxf(M[hh], mlv[hh].x);                 // finite: every chunk holds >= 1 token
      const float r = fast_exp2(M[hh] - mn), a = fast_exp2(mlv[hh].x - mn);
      M[hh] = mn;
      den[hh] = den[hh] * r + a * mlv[hh].y;
#pragma unroll
      for (int k = 0; k < V; ++k) acc[hh][k] = acc[hh][k] * r + a * x[hh][k];
    }
  }
#pragma unroll
  for (int hh = 0; hh < NH; ++hh) {
    const float inv = 1.f / den[hh];
    uint16_t* op = out_row0 + hh * D + lane * V;
    if constexpr (V == 4) {
      *reinterpret_cast<uint2*>(op) = make_uint2(pack_bf16x2(acc[hh][0] * inv, acc[hh][1] * inv),
                                                 pack_bf16x2(acc[hh][2] * inv, acc[hh][3] * inv));
    } else {
      *reinterpret_cast<uint32_t*>(op) = pack_bf16x2(acc[hh][0] * inv, acc[hh][1] * inv);
    }
  }
}

// columns [col0, col0 + ncols) of a partial slot that is `stride` columns wide, widest groups first;
// their outputs are ncols consecutive rows of D at out_row0
template <int D>
__device__ __forceinline__ void combine_cols(const float* part_o, const float* part_ml, int pb, int n_chunks,
                                             int stride, int col0, int ncols, uint16_t* out_row0, int lane) {
  int head = 0;
  for (; head + 4 <= ncols; head += 4)
    combine_heads<D, 4>(part_o, part_ml, pb, n_chunks, stride, col0 + head, out_row0 + head * D, lane);
  for (; head + 2 <= ncols; head += 2)
    combine_heads<D, 2>(part_o, part_ml, pb, n_chunks, stride, col0 + head, out_row0 + head * D, lane);
  for (; head < ncols; ++head)
    combine_heads<D, 1>(part_o, part_ml, pb, n_chunks, stride, col0 + head, out_row0 + head * D, lane);
}

// all G <= 8 heads of a (request, kv head)
template <int D>
__device__ __forceinline__ void combine_group(const float* part_o, const float* part_ml, int pb, int n_chunks, int G,
                                              uint16_t* out_row0, int lane) {
  combine_cols<D>(part_o, part_ml, pb, n_chunks, G, 0, G, out_row0, lane);
}

// kVarQ (in-place prefill of ultra-short requests merged with
// decoding): the 8 MMA columns of a unit are (query token, head) pairs of ONE kv head —
// column j = query token j / G of the tile, head j % G of the group — instead of the G heads of
// one token.  A work item is then a QUERY TILE of 8 / G consecutive query tokens of one request
// (item words 8..9: pos0 = absolute position of the tile's first query token, n_qtok = tokens in
// the tile), `batch_idx` is the tile's first row in q / out, and the mask is causal: column j
// sees tokens 0 .. pos0 + j / G.  A column may see nothing of a later chunk: its running max
// stays -inf, handled by the guards below (chunk 0 always holds token 0, visible to every column).
template <int D, bool kAppend, bool kVarQ = false>
__global__ void __launch_bounds__(kAttnThreads, 2) attn_splitkv_kernel(const AttnParams p) {
  constexpr int KJ = D / 32;   // K vectors per row per thread
  constexpr int KS = D / 16;   // MMA k-steps of S^T = K q^T
  constexpr int MT = D / 16;   // MMA m-tiles of O^T = V^T P^T
  constexpr int NE = D / 8;    // d columns owned per thread and head: 8 per V chunk
  constexpr int64_t kTileElems = 2 * kBlockSize * D;
  const int lane = threadIdx.x & 31;
  const int g = lane >> 2, c = lane & 3;
  const int G = p.group;
  const int64_t blk_stride = static_cast<int64_t>(p.num_kv_heads) * kTileElems;

  // Dynamic scheduling: the first unit of every warp is its global warp index (no atomic on the way to
  // the first byte), the rest come from a counter that starts at the number of warps.
  const int n_warps = gridDim.x * kAttnWarps;
  for (int item = blockIdx.x * kAttnWarps + (threadIdx.x >> 5);;) {
    if (item >= p.n_units) break;
    const int h = item % p.num_kv_heads;
    const int4* wi = reinterpret_cast<const int4*>(p.items) + (item / p.num_kv_heads) * (kVarQ ? 3 : 2);
    const int4 w0 = __ldg(wi);
    const int4 w1 = __ldg(wi + 1);
    const int batch_idx = w0.x, slot = w0.y, blk_begin = w0.z, n_blocks = w0.w;
    const int n_tokens = w1.x;
    const int n_chunks = w1.z >> 16, chunk_idx = w1.z & 0xffff, last_blk = w1.w;
    const int pbase = w1.y < 0 ? -1 : w1.y + h * n_chunks;     // first partial slot of (request, kv head)
    const int pidx = w1.y < 0 ? -1 : pbase + chunk_idx;
    // Fused append: the unit that owns the request's last block takes that tile FIRST (the order of
    // tiles does not matter to an online softmax), with the new token's row read from k_new / v_new.
    const bool special = kAppend && chunk_idx == n_chunks - 1;
    const int sp = special ? 1 : 0;
    // kVarQ: tokens in the tile, and the last visible token of columns 2c, 2c+1 relative to the chunk start
    int n_qtok = 1, rel0 = 0, rel1 = 0;
    if constexpr (kVarQ) {
      const int4 w2 = __ldg(wi + 2);
      n_qtok = w2.y;
      const int t0 = (2 * c) / G, t1 = (2 * c + 1) / G;
      rel0 = t0 < n_qtok ? w2.x + t0 - blk_begin * kBlockSize : 0x3fffffff;   // unused columns: q = 0, never stored
      rel1 = t1 < n_qtok ? w2.x + t1 - blk_begin * kBlockSize : 0x3fffffff;
    }

    // q^T as B fragments: lane (g, c) holds head g, columns of chunk c + 4j (zero for g >= G)
    uint32_t qf[KS][2];
    {
      bool ok = g < G;
      const uint16_t* qp =
          p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + (ok ? g : 0)) * D + c * 8;
      if constexpr (kVarQ) {                                     // column g = (query token g / G, head g % G)
        const int qt = g / G;
        ok = qt < n_qtok;
        qp = p.q + (static_cast<int64_t>(batch_idx + (ok ? qt : 0)) * p.num_q_heads + h * G + (ok ? g - qt * G : 0)) * D + c * 8;
      }
#pragma unroll
      for (int j = 0; j < KJ; ++j) {
        const uint4 v = ldg_stream_pred(qp + j * 32, ok);
        qf[2 * j][0] = v.x; qf[2 * j][1] = v.y; qf[2 * j + 1][0] = v.z; qf[2 * j + 1][1] = v.w;
      }
    }

    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // heads 2c, 2c+1 (l: this lane's rows only)
    float o[MT][4];
#pragma unroll
    for (int i = 0; i < MT; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;

    const int32_t* bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
    uint16_t* kvh = p.kv_layer + static_cast<int64_t>(h) * kTileElems;
    int32_t ids = lane < n_blocks ? __ldg(bt + lane) : 0;       // physical ids of blocks [32k, 32k+32)
    int32_t ids_next = 0;

    auto issue = [&](KVTile<D>& T, int t) {                     // start the loads of tile t
      if ((t & 31) == 0 && t > 0) ids = ids_next;
      if ((t & 31) == 8 && t + 24 + lane < n_blocks) ids_next = __ldg(bt + t + 24 + lane);
      const int blk = __shfl_sync(0xffffffffu, ids, t & 31);
      load_tile<D>(T, kvh + blk * blk_stride, n_tokens - t * kBlockSize, g, c);
    };

    auto consume = [&](const KVTile<D>& T, int t) {
      // ---- S^T = K q^T : two independent accumulation chains ----
      float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < KJ; ++j) {
        mma_bf16_m16n8k16(sa, T.k[0][j].x, T.k[1][j].x, T.k[0][j].y, T.k[1][j].y, qf[2 * j][0], qf[2 * j][1]);
        mma_bf16_m16n8k16(sb, T.k[0][j].z, T.k[1][j].z, T.k[0][j].w, T.k[1][j].w, qf[2 * j + 1][0],
                          qf[2 * j + 1][1]);
      }
      // s[0], s[1]: token g, heads 2c, 2c+1;  s[2], s[3]: token g+8
      float s[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) s[i] = (sa[i] + sb[i]) * p.scale_log2;
      const int nv = n_tokens - t * kBlockSize;
      if (nv < kBlockSize) {                                    // ragged last block: mask by index, not value
        if (g >= nv) s[0] = s[1] = -INFINITY;
        if (g + 8 >= nv) s[2] = s[3] = -INFINITY;
      }
      if constexpr (kVarQ) {                                    // causal: column sees tokens <= its own position
        const int tok = t * kBlockSize + g;
        if (tok > rel0) s[0] = -INFINITY;
        if (tok > rel1) s[1] = -INFINITY;
        if (tok + 8 > rel0) s[2] = -INFINITY;
        if (tok + 8 > rel1) s[3] = -INFINITY;
      }
      // ---- online softmax over the token axis (= across the 8 lanes sharing c) ----
      float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
#pragma unroll
      for (int off = 4; off < 32; off <<= 1) {
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, off));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, off));
      }
      const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);   // finite: every tile has >= 1 valid token ...
      float ms0 = mn0, ms1 = mn1;
      if constexpr (kVarQ) {                                    // ... except for a column that sees nothing yet
        ms0 = mn0 == -INFINITY ? 0.f : mn0;
        ms1 = mn1 == -INFINITY ? 0.f : mn1;
      }
      const float a0 = fast_exp2(m0 - ms0), a1 = fast_exp2(m1 - ms1);
      m0 = mn0; m1 = mn1;
      const float p0 = fast_exp2(s[0] - ms0), p1 = fast_exp2(s[1] - ms1);
      const float p2 = fast_exp2(s[2] - ms0), p3 = fast_exp2(s[3] - ms1);
      l0 = l0 * a0 + (p0 + p2);
      l1 = l1 * a1 + (p1 + p3);
#pragma unroll
      for (int i = 0; i < MT; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
      // ---- P^T as the B fragment: transpose the two 8x8 halves across the warp.  P is fed to the
      // tensor core as bf16 hi + bf16 lo (p = hi + lo up to 2^-17 p), so the weights keep ~16 mantissa
      // bits and the only bf16-sized error left in the result is the final rounding of `out`.
      const uint32_t ph01 = pack_bf16x2(p0, p1), ph23 = pack_bf16x2(p2, p3);
      const uint32_t pl01 = pack_bf16x2(p0 - __uint_as_float(ph01 << 16), p1 - __uint_as_float(ph01 & 0xffff0000u));
      const uint32_t pl23 = pack_bf16x2(p2 - __uint_as_float(ph23 << 16), p3 - __uint_as_float(ph23 & 0xffff0000u));
      const uint32_t b0 = movmatrix_trans(ph01);                 // tokens 2c, 2c+1   of head g
      const uint32_t b1 = movmatrix_trans(ph23);                 // tokens 2c+8, 2c+9 of head g
      const uint32_t c0 = movmatrix_trans(pl01);
      const uint32_t c1 = movmatrix_trans(pl23);
      // ---- O^T += V^T P^T : m-tile i takes d column e = i (row g) and e = i + NE/2 (row g+8) ----
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        const int e1 = i, e2 = i + NE / 2;
        const int r1 = (e1 & 7) >> 1, r2 = (e2 & 7) >> 1, cs1 = e1 >> 3, cs2 = e2 >> 3;
        uint32_t a0_, a1_, a2_, a3_;
        if (e1 & 1) {
          a0_ = pair_hi(u4_get(T.v[0][cs1], r1), u4_get(T.v[1][cs1], r1));
          a2_ = pair_hi(u4_get(T.v[2][cs1], r1), u4_get(T.v[3][cs1], r1));
        } else {
          a0_ = pair_lo(u4_get(T.v[0][cs1], r1), u4_get(T.v[1][cs1], r1));
          a2_ = pair_lo(u4_get(T.v[2][cs1], r1), u4_get(T.v[3][cs1], r1));
        }
        if (e2 & 1) {
          a1_ = pair_hi(u4_get(T.v[0][cs2], r2), u4_get(T.v[1][cs2], r2));
          a3_ = pair_hi(u4_get(T.v[2][cs2], r2), u4_get(T.v[3][cs2], r2));
        } else {
          a1_ = pair_lo(u4_get(T.v[0][cs2], r2), u4_get(T.v[1][cs2], r2));
          a3_ = pair_lo(u4_get(T.v[2][cs2], r2), u4_get(T.v[3][cs2], r2));
        }
        mma_bf16_m16n8k16(o[i], a0_, a1_, a2_, a3_, b0, b1);
        mma_bf16_m16n8k16(o[i], a0_, a1_, a2_, a3_, c0, c1);
      }
    };

    KVTile<D> A, B;
    uint16_t* last_tile = kvh + last_blk * blk_stride;
    const int nv_last = n_tokens - (n_blocks - 1) * kBlockSize;
    if (special) {
      const int64_t row = (static_cast<int64_t>(batch_idx) * p.num_kv_heads + h) * D;
      load_tile_append<D>(A, last_tile, p.k_new + row, p.v_new + row, nv_last, g, c);
      if (h == 0 && lane == 0) p.block_table[static_cast<int64_t>(slot) * p.bt_stride + blk_begin + n_blocks - 1] = last_blk;
    } else {
      issue(A, 0);
    }
    // virtual tile v -> real tile: special ? (v == 0 ? n_blocks - 1 : v - 1) : v
    for (int v = 0; v < n_blocks; v += 2) {
      const bool has_b = v + 1 < n_blocks;
      if (has_b) issue(B, v + 1 - sp);
      if (special && v == 0) {
        consume(A, n_blocks - 1);
        store_new_row<D>(A, last_tile, nv_last, g, c);
      } else {
        consume(A, v - sp);
      }
      if (has_b) {
        if (v + 2 < n_blocks) issue(A, v + 2 - sp);
        consume(B, v + 1 - sp);
      }
    }

    // ---- epilogue: finish l over the token lanes, then store ----
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {
      l0 += __shfl_xor_sync(0xffffffffu, l0, off);
      l1 += __shfl_xor_sync(0xffffffffu, l1, off);
    }
    const int PG = kVarQ ? 8 : G;                                // columns per partial slot
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
      const int head = 2 * c + hh;                               // MMA column
      int64_t out_row;
      if constexpr (kVarQ) {
        const int qt = head / G;
        if (qt >= n_qtok) continue;
        out_row = static_cast<int64_t>(batch_idx + qt) * p.num_q_heads + h * G + (head - qt * G);
      } else {
        if (head >= G) continue;
        out_row = static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + head;
      }
      const float l = hh ? l1 : l0, m = hh ? m1 : m0;
      // element e of this lane: d column (g + 8*(e/8))*8 + e%8, register o[e % (NE/2)][2*(e/(NE/2)) + hh]
      if (pidx < 0) {
        const float inv = 1.f / l;
        uint16_t* op = p.out + out_row * D;
#pragma unroll
        for (int cs = 0; cs < D / 64; ++cs) {
          uint32_t w[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int e = cs * 8 + 2 * k;
            w[k] = pack_bf16x2(o[e % (NE / 2)][2 * (e / (NE / 2)) + hh] * inv,
                               o[(e + 1) % (NE / 2)][2 * ((e + 1) / (NE / 2)) + hh] * inv);
          }
          *reinterpret_cast<uint4*>(op + (g + 8 * cs) * 8) = make_uint4(w[0], w[1], w[2], w[3]);
        }
      } else {
        float* po = p.part_o + (static_cast<int64_t>(pidx) * PG + head) * D;
#pragma unroll
        for (int cs = 0; cs < D / 64; ++cs) {
          float f[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const int e = cs * 8 + k;
            f[k] = o[e % (NE / 2)][2 * (e / (NE / 2)) + hh];
          }
          float4* dst = reinterpret_cast<float4*>(po + (g + 8 * cs) * 8);
          dst[0] = make_float4(f[0], f[1], f[2], f[3]);
          dst[1] = make_float4(f[4], f[5], f[6], f[7]);
        }
        if (g == 0) *reinterpret_cast<float2*>(p.part_ml + (static_cast<int64_t>(pidx) * PG + head) * 2) = make_float2(m, l);
      }
    }
    // ---- fused a5: the unit that completes its (request, kv head) merges the partials ----
    if (pidx >= 0 && (kVarQ || p.fuse_combine)) {
      __threadfence();                                           // this lane's partial stores, device-wide
      __syncwarp();
      int last = 0;
      if (lane == 0) {
        last = atomicAdd(&p.arrive[pbase], 1) == n_chunks - 1;
        if (last) p.arrive[pbase] = 0;                           // ready for the next launch
      }
      last = __shfl_sync(0xffffffffu, last, 0);
      if (last) {
        __threadfence();
        if constexpr (kVarQ) {
          for (int qt = 0; qt < n_qtok; ++qt)
            combine_cols<D>(p.part_o, p.part_ml, pbase, n_chunks, 8, qt * G, G,
                            p.out + (static_cast<int64_t>(batch_idx + qt) * p.num_q_heads + h * G) * D, lane);
        } else {
          combine_group<D>(p.part_o, p.part_ml, pbase, n_chunks, G,
                           p.out + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G) * D, lane);
        }
      }
    }
    if (lane == 0) item = n_warps + atomicAdd(&p.counters[0], 1);
    item = __shfl_sync(0xffffffffu, item, 0);
  }

  // Last CTA out rewinds the work counter for the next launch (launches on one pool are
  // stream-ordered; counters[1] wraps to 0 by itself).
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned prev = atomicInc(reinterpret_cast<unsigned*>(&p.counters[1]), gridDim.x - 1);
    if (prev == gridDim.x - 1) p.counters[0] = 0;
  }
}

// ---------------------------------------------------------------------------------------------
// a5 log-sum-exp combine: one warp per (combine entry, head of the group)
// ---------------------------------------------------------------------------------------------

struct CombineEntryDev { int32_t batch_idx, partial_begin, n_chunks, pad; };  // == kvp::CombineEntry

struct CombineParams {
  const CombineEntryDev* entries;
  int32_t n_entries;
  const float* part_o;
  const float* part_ml;
  uint16_t* out;
  int32_t num_q_heads, num_kv_heads, group;
};

template <int D>
__global__ void __launch_bounds__(128) combine_kernel(const CombineParams p) {
  const int lane = threadIdx.x & 31;
  const int w = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (w >= p.n_entries * p.num_q_heads) return;
  const int ei = w / p.num_q_heads, qh = w % p.num_q_heads;
  const int kvh = qh / p.group, head = qh % p.group;
  const CombineEntryDev e = p.entries[ei];
  // partials of (request, kv head) are contiguous over chunks
  combine_heads<D, 1>(p.part_o, p.part_ml, e.partial_begin + kvh * e.n_chunks, e.n_chunks, p.group, head,
                      p.out + (static_cast<int64_t>(e.batch_idx) * p.num_q_heads + qh) * D, lane);
}

}  // namespace kvp
