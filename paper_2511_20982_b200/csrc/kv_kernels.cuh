// kv_kernels.cuh — sm_100a kernels of the D-instance KV path.
//
//   ingest_kernel<D, kGather>   a2/a3 (and its inverse): contiguous [L][Hkv][n][d] <-> paged blocks
//   attn_splitkv_kernel<D>      a4: split-KV paged decode attention, one warp per work item
//   combine_kernel<D>           a5: log-sum-exp merge of split-KV partials
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
};

template <int D, bool kGather>
__global__ void __launch_bounds__(kIngestThreads) ingest_kernel(const IngestParams p) {
  constexpr int kPiecesPerRow = D / 8;                       // 16-byte pieces per token row
  constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;  // 8 at D=128, 4 at D=64
  const int lane = threadIdx.x & 31;
  const int64_t u = static_cast<int64_t>(blockIdx.x) * kIngestWarps + (threadIdx.x >> 5);
  if (u >= p.total_units) return;

  // request of this unit: last i with unit_begin <= u
  int lo = 0, hi = p.n_req - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (__ldg(&p.reqs[mid].unit_begin) <= u) lo = mid; else hi = mid - 1;
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
  const int64_t src_off = ((static_cast<int64_t>(ll) * p.num_kv_heads + h) * r.n_tokens + t0) * D;
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
  int32_t batch_idx, slot, blk_begin, n_blocks, n_tokens, partial_base, n_chunks, chunk_idx;
};

struct AttnParams {
  const uint16_t* kv_layer;    // &kv[layer][0]...
  const int32_t* block_table;
  int32_t bt_stride;
  const WorkItemDev* items;
  int32_t n_items, n_units;    // n_units = n_items * num_kv_heads
  const uint16_t* q;
  uint16_t* out;
  float* part_o;               // [n_partials][G][D]  un-normalised
  float* part_ml;              // [n_partials][G][2]  (m in log2 units, l)
  int32_t* counters;           // [0] next work item, [1] finished CTAs
  int32_t num_q_heads, num_kv_heads, group;
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

template <int D>
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

  for (;;) {
    int item = 0;
    if (lane == 0) item = atomicAdd(&p.counters[0], 1);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= p.n_units) break;
    const int h = item % p.num_kv_heads;
    const WorkItemDev* wi = p.items + item / p.num_kv_heads;
    const int4 w0 = __ldg(reinterpret_cast<const int4*>(wi));
    const int4 w1 = __ldg(reinterpret_cast<const int4*>(wi) + 1);
    const int batch_idx = w0.x, slot = w0.y, blk_begin = w0.z, n_blocks = w0.w;
    const int n_tokens = w1.x;
    const int pidx = w1.y < 0 ? -1 : w1.y + h * w1.z + w1.w;

    // q^T as B fragments: lane (g, c) holds head g, columns of chunk c + 4j (zero for g >= G)
    uint32_t qf[KS][2];
    {
      const bool ok = g < G;
      const uint16_t* qp =
          p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + (ok ? g : 0)) * D + c * 8;
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
    const uint16_t* kvh = p.kv_layer + static_cast<int64_t>(h) * kTileElems;
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
      // ---- online softmax over the token axis (= across the 8 lanes sharing c) ----
      float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
#pragma unroll
      for (int off = 4; off < 32; off <<= 1) {
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, off));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, off));
      }
      const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);   // finite: every tile has >= 1 valid token
      const float a0 = fast_exp2(m0 - mn0), a1 = fast_exp2(m1 - mn1);
      m0 = mn0; m1 = mn1;
      const float p0 = fast_exp2(s[0] - mn0), p1 = fast_exp2(s[1] - mn1);
      const float p2 = fast_exp2(s[2] - mn0), p3 = fast_exp2(s[3] - mn1);
      l0 = l0 * a0 + (p0 + p2);
      l1 = l1 * a1 + (p1 + p3);
#pragma unroll
      for (int i = 0; i < MT; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
      // ---- P^T as the B fragment: transpose the two 8x8 halves across the warp ----
      const uint32_t b0 = movmatrix_trans(pack_bf16x2(p0, p1));  // tokens 2c, 2c+1   of head g
      const uint32_t b1 = movmatrix_trans(pack_bf16x2(p2, p3));  // tokens 2c+8, 2c+9 of head g
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
      }
    };

    KVTile<D> A, B;
    issue(A, 0);
    for (int t = 0; t < n_blocks; t += 2) {
      const bool has_b = t + 1 < n_blocks;
      if (has_b) issue(B, t + 1);
      consume(A, t);
      if (has_b) {
        if (t + 2 < n_blocks) issue(A, t + 2);
        consume(B, t + 1);
      }
    }

    // ---- epilogue: finish l over the token lanes, then store ----
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {
      l0 += __shfl_xor_sync(0xffffffffu, l0, off);
      l1 += __shfl_xor_sync(0xffffffffu, l1, off);
    }
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
      const int head = 2 * c + hh;
      if (head >= G) continue;
      const float l = hh ? l1 : l0, m = hh ? m1 : m0;
      // element e of this lane: d column (g + 8*(e/8))*8 + e%8, register o[e % (NE/2)][2*(e/(NE/2)) + hh]
      if (pidx < 0) {
        const float inv = 1.f / l;
        uint16_t* op = p.out + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + head) * D;
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
        float* po = p.part_o + (static_cast<int64_t>(pidx) * G + head) * D;
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
        if (g == 0) *reinterpret_cast<float2*>(p.part_ml + (static_cast<int64_t>(pidx) * G + head) * 2) = make_float2(m, l);
      }
    }
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
  constexpr int V = D / 32;  // floats per lane
  const int lane = threadIdx.x & 31;
  const int w = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (w >= p.n_entries * p.num_q_heads) return;
  const int ei = w / p.num_q_heads, qh = w % p.num_q_heads;
  const int kvh = qh / p.group, head = qh % p.group;
  CombineEntryDev e = p.entries[ei];
  e.partial_begin += kvh * e.n_chunks;                        // partials of (request, kv head): contiguous over chunks
  const float* ml = p.part_ml + (static_cast<int64_t>(e.partial_begin) * p.group + head) * 2;
  const int64_t ml_stride = static_cast<int64_t>(p.group) * 2;
  const float* po = p.part_o + (static_cast<int64_t>(e.partial_begin) * p.group + head) * D + lane * V;
  const int64_t po_stride = static_cast<int64_t>(p.group) * D;

  float M = -INFINITY;
  for (int ch = lane; ch < e.n_chunks; ch += 32) M = fmaxf(M, __ldg(ml + ch * ml_stride));
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, off));

  float acc[V];
#pragma unroll
  for (int k = 0; k < V; ++k) acc[k] = 0.f;
  float den = 0.f;
#pragma unroll 4
  for (int ch = 0; ch < e.n_chunks; ++ch) {
    const float2 mlv = __ldg(reinterpret_cast<const float2*>(ml + ch * ml_stride));
    const float a = fast_exp2(mlv.x - M);
    den += a * mlv.y;
    if constexpr (V == 4) {
      const float4 x = __ldg(reinterpret_cast<const float4*>(po + ch * po_stride));
      acc[0] += a * x.x; acc[1] += a * x.y; acc[2] += a * x.z; acc[3] += a * x.w;
    } else {
      const float2 x = __ldg(reinterpret_cast<const float2*>(po + ch * po_stride));
      acc[0] += a * x.x; acc[1] += a * x.y;
    }
  }
  const float inv = 1.f / den;
  uint16_t* op = p.out + (static_cast<int64_t>(e.batch_idx) * p.num_q_heads + qh) * D + lane * V;
  if constexpr (V == 4) {
    *reinterpret_cast<uint2*>(op) = make_uint2(pack_bf16x2(acc[0] * inv, acc[1] * inv), pack_bf16x2(acc[2] * inv, acc[3] * inv));
  } else {
    *reinterpret_cast<uint32_t*>(op) = pack_bf16x2(acc[0] * inv, acc[1] * inv);
  }
}

}  // namespace kvp
