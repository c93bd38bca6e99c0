// kv_copy.cuh — the relocation kernels of the D-instance KV path (no arithmetic except the FP8 pool's quantisation):
//
//   ingest_kernel<D, kGather>    a2 / a3 and its inverse: contiguous [L][Hkv][n][D] bf16 <-> paged bf16 blocks
//   ingest_fp8_kernel<D>         a2 / a3 into an FP8 pool: quantising scatter (NEXT-2)
//   gather_fp8_kernel<D>         paged FP8 blocks -> contiguous codes + scales (producer half of NEXT-4 on an FP8 pool)
//   transfer_kernel<D, kFp8>     NEXT-4: paged -> paged, producer pool's blocks to consumer pool's blocks, each side
//                                addressed through its own block list; no contiguous staging
//
// All are HBM-bound at 0 flop/byte: one warp per (request, layer, kv head, touched block) unit, whose rows are
// contiguous on both sides; a lane issues ALL its 16-byte loads and then all its stores (sector-exact, L1 bypassed).
#pragma once

#include "kv_common.cuh"

namespace kvp {

constexpr int kIngestThreads = 256;
constexpr int kIngestWarps = kIngestThreads / 32;

// A unit of an ingest / gather / transfer launch, located from its global index.
struct IngestUnit {
  IngestReq r;
  int jj;          // touched block index within the request
  int h, ll;       // kv head, layer index within [0, layer_count)
  int lb;          // logical block
  int row0, row1;  // rows [row0, row1) of the block belong to this call
  int t0;          // first source token of the unit (relative to the call's first token)
};

// Request of unit u: last i with unit_begin <= u.  The lanes test 32 candidates at a time (independent loads, one
// ballot each) rather than walk a binary search of dependent loads.  kRun > 1: a unit is a RUN of up to kRun
// consecutive touched blocks of one (request, layer, kv head) — the returned fields describe the run's first block.
template <int kRun = 1>
__device__ __forceinline__ IngestUnit locate_unit(const IngestParams& p, int64_t u, int lane) {
  int lo = -1;
  for (int base = 0; base < p.n_req; base += 32) {
    const int i = base + lane;
    const bool le = i < p.n_req && __ldg(&p.reqs[i].unit_begin) <= u;
    lo += __popc(__ballot_sync(kFull, le));
  }
  IngestUnit x;
  x.r = p.reqs[lo];
  const int64_t local = u - x.r.unit_begin;
  const int runs = (x.r.n_touched + kRun - 1) / kRun;
  x.jj = static_cast<int>(local % runs) * kRun;
  const int rest = static_cast<int>(local / runs);
  x.h = rest % p.num_kv_heads;
  x.ll = rest / p.num_kv_heads;
  x.lb = x.r.blk0 + x.jj;
  x.row0 = (x.jj == 0) ? (x.r.start_pos & (kBlockSize - 1)) : 0;
  x.row1 = min(kBlockSize, x.r.start_pos + x.r.n_tokens - x.lb * kBlockSize);
  x.t0 = x.lb * kBlockSize + x.row0 - x.r.start_pos;
  return x;
}

template <int D, bool kGather>
__global__ void __launch_bounds__(kIngestThreads) ingest_kernel(const IngestParams p) {
  constexpr int kPiecesPerRow = D / 8;                       // 16-byte pieces per token row
  constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;  // 8 at D=128, 4 at D=64
  const int lane = threadIdx.x & 31;
  const int64_t u = static_cast<int64_t>(blockIdx.x) * kIngestWarps + (threadIdx.x >> 5);
  if (u >= p.total_units) return;
  const IngestUnit x = locate_unit(p, u, lane);
  const int blk = __ldg(&p.blk_ids[x.r.blk_off + x.jj]);
  const int pieces = (x.row1 - x.row0) * kPiecesPerRow;

  // rows row0..row1-1 are contiguous both in the source run and inside the block
  const int64_t src_off = ((static_cast<int64_t>(x.ll) * p.src_kv_heads + p.src_head_begin + x.h) * x.r.n_tokens + x.t0) * D;
  const int64_t dst_off =
      ((((static_cast<int64_t>(p.layer_begin + x.ll) * p.num_blocks + blk) * p.num_kv_heads + x.h) * 2) * kBlockSize +
       x.row0) * D;
  const uint4* lin_k = reinterpret_cast<const uint4*>(reinterpret_cast<const uint16_t*>(x.r.k_src) + src_off);
  const uint4* lin_v = reinterpret_cast<const uint4*>(reinterpret_cast<const uint16_t*>(x.r.v_src) + src_off);
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
  if (!kGather && x.ll == 0 && x.h == 0 && lane == 0)         // device block_table mirror (a1, device half)
    p.block_table[static_cast<int64_t>(x.r.slot) * p.bt_stride + x.lb] = blk;
}

// ---------------------------------------------------------------------------------------------
// quantising scatter (NEXT-2): same descriptors as ingest_kernel (IngestParams::kv = the FP8 region).  Unlike the
// plain copies this kernel has arithmetic between its loads and its stores, and the first version (one warp per
// (block, K|V), every lane dividing for every piece) was ISSUE-bound: 74 % issue slots, 990 instructions per 4 KiB of
// source (profiles/r02).  This one
//   * gives a warp a RUN of kIngest8Run consecutive blocks of one (request, layer, kv head, K|V): one descriptor
//     lookup per run, 16 KiB of contiguous source per warp, the next block's loads issued before the current
//     block is quantised (two register buffers);
//   * finds the 16 row maxima of a block with a halving butterfly (8 shuffles per lane instead of 32): after it
//     every lane OWNS one row, computes that row's scale and inverse once (two IEEE divisions per lane instead of
//     sixteen), stores the scale, and hands the inverse to the lanes holding the row's pieces (one shuffle each).
// The arithmetic that decides a code is unchanged (C3): amax exact, fl32 divisions, fl32 product, RNE
// e4m3 saturating — byte-exact against oracle_scatter_fp8.  Launch with 2 * total_units warps (unit = run).
// ---------------------------------------------------------------------------------------------
constexpr int kIngest8Threads = 64;
constexpr int kIngest8Warps = kIngest8Threads / 32;
constexpr int kIngest8Run = 4;
template <int D>
__global__ void __launch_bounds__(kIngest8Threads) ingest_fp8_kernel(const IngestParams p) {
  constexpr int kPiecesPerRow = D / 8;                          // 16-byte source pieces (8 bf16) per token row
  constexpr int NV = kBlockSize * kPiecesPerRow / 32;           // pieces per lane and block: 8 at D=128, 4 at D=64
  static_assert(kPiecesPerRow == 2 * NV, "a row's pieces sit on 2 * NV neighbouring lanes");
  const int lane = threadIdx.x & 31;
  const int64_t u2 = static_cast<int64_t>(blockIdx.x) * kIngest8Warps + (threadIdx.x >> 5);
  const int64_t u = u2 >> 1;
  const int c = static_cast<int>(u2 & 1);                        // 0: the K rows of the run, 1: the V rows
  if (u >= p.total_units) return;
  const IngestUnit x = locate_unit<kIngest8Run>(p, u, lane);
  const int n_run = min(kIngest8Run, x.r.n_touched - x.jj);
  const int32_t blk_id = lane < n_run ? __ldg(&p.blk_ids[x.r.blk_off + x.jj + lane]) : 0;
  const int grp = lane / kPiecesPerRow;                          // which of the 32 / kPiecesPerRow rows a piece index step covers
  const int own = (lane >> 1) & (NV - 1);                        // the value index this lane owns after the butterfly
  const uint16_t* src = reinterpret_cast<const uint16_t*>(c ? x.r.v_src : x.r.k_src) +
                        (static_cast<int64_t>(x.ll) * p.src_kv_heads + p.src_head_begin + x.h) * x.r.n_tokens * D;
  uint8_t* const layer_head = reinterpret_cast<uint8_t*>(p.kv) +
                              (static_cast<int64_t>(p.layer_begin + x.ll) * p.num_blocks * p.num_kv_heads + x.h) * fp8_tile_bytes<D>();

  // rows [row0, row1) of run block b and its first source token
  auto rows_of = [&](int b, int& row0, int& row1, int& t0) {
    const int lb = x.lb + b;
    row0 = (x.jj + b == 0) ? (x.r.start_pos & (kBlockSize - 1)) : 0;
    row1 = min(kBlockSize, x.r.start_pos + x.r.n_tokens - lb * kBlockSize);
    t0 = lb * kBlockSize + row0 - x.r.start_pos;
  };
  // kWhole (a literal at every call site, folded after inlining): the block is known to hold 16 of this call's rows —
  // no per-piece predicates (the common case: the run lies inside the request; the kernel is issue-bound)
  auto load = [&](uint4 (&buf)[NV], int b, const bool kWhole) {
    int row0 = 0, row1 = kBlockSize, t0 = (x.lb + b) * kBlockSize - x.r.start_pos;
    if (!kWhole) rows_of(b, row0, row1, t0);
    const uint4* lin = reinterpret_cast<const uint4*>(src + static_cast<int64_t>(t0) * D);
    const int pieces = (row1 - row0) * kPiecesPerRow;
#pragma unroll
    for (int i = 0; i < NV; ++i) buf[i] = ldg_copy_pred(lin + lane + 32 * i, kWhole || lane + 32 * i < pieces);
  };
  auto quantise_store = [&](const uint4 (&buf)[NV], int b, const bool kWhole) {
    int row0 = 0, row1 = kBlockSize, t0 = 0;
    if (!kWhole) rows_of(b, row0, row1, t0);
    const int rows = row1 - row0;
    const int32_t blk = __shfl_sync(kFull, blk_id, b);
    uint8_t* tile = layer_head + static_cast<int64_t>(blk) * p.num_kv_heads * fp8_tile_bytes<D>();
    // packed |x| maxima of the lane's NV pieces (piece i belongs to row (32 / kPiecesPerRow) * i + grp of the block's rows)
    uint32_t m[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i)
      m[i] = __vmaxu2(__vmaxu2(buf[i].x & 0x7fff7fffu, buf[i].y & 0x7fff7fffu), __vmaxu2(buf[i].z & 0x7fff7fffu, buf[i].w & 0x7fff7fffu));
    // halving butterfly over the 2 * NV lanes that share rows: each step keeps half of the values and swaps the other half
#pragma unroll
    for (int n = NV, off = NV; n > 1; n >>= 1, off >>= 1) {
      const bool up = (lane & off) != 0;
#pragma unroll
      for (int k = 0; k < n / 2; ++k) {
        const uint32_t send = up ? m[k] : m[k + n / 2];
        const uint32_t keep = up ? m[k + n / 2] : m[k];
        m[k] = __vmaxu2(keep, __shfl_xor_sync(kFull, send, off));
      }
    }
    m[0] = __vmaxu2(m[0], __shfl_xor_sync(kFull, m[0], 1));
    const uint32_t mx = max(m[0] & 0xffffu, m[0] >> 16);          // row maximum of the row this lane owns (bf16 bits)
    const float amax = __uint_as_float(mx << 16);
    const float scale = mx == 0 ? 1.f : __fdiv_rn(amax, 448.f);
    const float inv = mx == 0 ? 1.f : __fdiv_rn(448.f, amax);
    const int own_row = (32 / kPiecesPerRow) * own + grp;          // relative to row0
    if ((lane & 1) == 0 && (kWhole || own_row < rows))
      *reinterpret_cast<float*>(tile + 2 * kBlockSize * D + (row0 + own_row) * 8 + c * 4) = scale;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const float inv_i = __shfl_sync(kFull, inv, (lane & ~(2 * NV - 1)) | (i << 1));
      const int idx = lane + 32 * i;
      uint32_t w[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t e = u4_get(buf[i], k);
        w[k] = f32x2_to_e4m3x2(__fmul_rn(__uint_as_float(e << 16), inv_i), __fmul_rn(__uint_as_float(e & 0xffff0000u), inv_i));
      }
      if (kWhole || idx < rows * kPiecesPerRow)
        *reinterpret_cast<uint2*>(tile + c * (kBlockSize * D) + row0 * D + idx * 8) = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
    }
    if (c == 0 && x.ll == 0 && x.h == 0 && lane == 0)             // device block_table mirror (a1, device half)
      p.block_table[static_cast<int64_t>(x.r.slot) * p.bt_stride + x.lb + b] = blk;
  };

  uint4 bufa[NV], bufb[NV];
  // the whole run lies inside this call's rows: four full blocks, no predicates
  const bool run_full = n_run == kIngest8Run && (x.jj > 0 || (x.r.start_pos & (kBlockSize - 1)) == 0) &&
                        x.r.start_pos + x.r.n_tokens >= (x.lb + kIngest8Run) * kBlockSize;
  if (run_full) {
    load(bufa, 0, true);
#pragma unroll
    for (int b = 0; b < kIngest8Run; b += 2) {
      load(bufb, b + 1, true);
      quantise_store(bufa, b, true);
      if (b + 2 < kIngest8Run) load(bufa, b + 2, true);
      quantise_store(bufb, b + 1, true);
    }
    return;
  }
  load(bufa, 0, false);
#pragma unroll
  for (int b = 0; b < kIngest8Run; b += 2) {
    if (b < n_run) {
      if (b + 1 < n_run) load(bufb, b + 1, false);
      quantise_store(bufa, b, false);
    }
    if (b + 1 < n_run) {
      if (b + 2 < n_run) load(bufa, b + 2, false);
      quantise_store(bufb, b + 1, false);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// FP8 gather: stored codes and row scales of a request, contiguous (include/kv_pool.h, kv_gather on an FP8 pool):
//   r.k_src / r.v_src = destination of the K / V side:  codes u8 [layer_count][src_kv_heads][n][D], then, at the next
//   16-byte boundary, scales fp32 [layer_count][src_kv_heads][n].  One warp per unit, K and V both.
// ---------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kIngestThreads) gather_fp8_kernel(const IngestParams p) {
  constexpr int kPiecesPerRow = D / 16;                         // 16-byte pieces (16 codes) per token row
  constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;  // 4 at D=128, 2 at D=64
  const int lane = threadIdx.x & 31;
  const int64_t u = static_cast<int64_t>(blockIdx.x) * kIngestWarps + (threadIdx.x >> 5);
  if (u >= p.total_units) return;
  const IngestUnit x = locate_unit(p, u, lane);
  const int blk = __ldg(&p.blk_ids[x.r.blk_off + x.jj]);
  const int rows = x.row1 - x.row0, pieces = rows * kPiecesPerRow;
  const uint8_t* tile = reinterpret_cast<const uint8_t*>(p.kv) +
                        ((static_cast<int64_t>(p.layer_begin + x.ll) * p.num_blocks + blk) * p.num_kv_heads + x.h) * fp8_tile_bytes<D>();
  const int64_t row_idx = (static_cast<int64_t>(x.ll) * p.src_kv_heads + p.src_head_begin + x.h) * x.r.n_tokens + x.t0;
  const int64_t codes_bytes = (static_cast<int64_t>(p.layer_count) * p.src_kv_heads * x.r.n_tokens * D + 15) / 16 * 16;
  uint8_t* kd = reinterpret_cast<uint8_t*>(x.r.k_src);
  uint8_t* vd = reinterpret_cast<uint8_t*>(x.r.v_src);

  uint4 bk[kMaxPerLane], bv[kMaxPerLane];
#pragma unroll
  for (int i = 0; i < kMaxPerLane; ++i) {
    const int idx = lane + 32 * i;
    bk[i] = ldg_copy_pred(tile + x.row0 * D + idx * 16, idx < pieces);
    bv[i] = ldg_copy_pred(tile + kBlockSize * D + x.row0 * D + idx * 16, idx < pieces);
  }
  const uint2 sc = ldg_copy8_pred(tile + 2 * kBlockSize * D + (x.row0 + lane) * 8, lane < rows);
#pragma unroll
  for (int i = 0; i < kMaxPerLane; ++i) {
    const int idx = lane + 32 * i;
    stg_stream_pred(kd + row_idx * D + idx * 16, bk[i], idx < pieces);
    stg_stream_pred(vd + row_idx * D + idx * 16, bv[i], idx < pieces);
  }
  if (lane < rows) {
    reinterpret_cast<uint32_t*>(kd + codes_bytes)[row_idx + lane] = sc.x;
    reinterpret_cast<uint32_t*>(vd + codes_bytes)[row_idx + lane] = sc.y;
  }
}

// ---------------------------------------------------------------------------------------------
// NEXT-4 — producer -> consumer transfer, paged -> paged ("KV-cache transmission ... depending on
// block fragmentation and count"; the KV-cache transmitter writes into the consumer's KV-cache
// blocks).  Unit = (request, layer, kv head, block): the block's valid rows move tile to tile, the source address
// through the producer's block list, the destination through the consumer's — no contiguous staging buffer, one
// launch for any number of requests.  p.src_kv is a plain pointer: a peer-mapped producer slab (NVLink) is read by
// the same code.  FP8 pools move codes and row scales verbatim.  blk_ids of request i: n_touched consumer ids,
// then n_touched producer ids.
// ---------------------------------------------------------------------------------------------
template <int D, bool kFp8>
__global__ void __launch_bounds__(kIngestThreads) transfer_kernel(const IngestParams p) {
  const int lane = threadIdx.x & 31;
  const int64_t u = static_cast<int64_t>(blockIdx.x) * kIngestWarps + (threadIdx.x >> 5);
  if (u >= p.total_units) return;
  const IngestUnit x = locate_unit(p, u, lane);
  const int dblk = __ldg(&p.blk_ids[x.r.blk_off + x.jj]);
  const int sblk = __ldg(&p.blk_ids[x.r.blk_off + x.r.n_touched + x.jj]);
  const int rows = x.row1;                                      // whole requests: row0 = 0
  const int64_t layer = p.layer_begin + x.ll;
  if constexpr (!kFp8) {
    constexpr int kPiecesPerRow = D / 8;
    constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;
    constexpr int64_t kTile = 2 * kBlockSize * D;               // elements
    const uint16_t* st = p.src_kv + ((layer * p.src_num_blocks + sblk) * p.num_kv_heads + x.h) * kTile;
    uint16_t* dt = p.kv + ((layer * p.num_blocks + dblk) * p.num_kv_heads + x.h) * kTile;
    const int pieces = rows * kPiecesPerRow;
    uint4 bk[kMaxPerLane], bv[kMaxPerLane];
#pragma unroll
    for (int i = 0; i < kMaxPerLane; ++i) {
      const int idx = lane + 32 * i;
      bk[i] = ldg_copy_pred(reinterpret_cast<const uint4*>(st) + idx, idx < pieces);
      bv[i] = ldg_copy_pred(reinterpret_cast<const uint4*>(st + kBlockSize * D) + idx, idx < pieces);
    }
#pragma unroll
    for (int i = 0; i < kMaxPerLane; ++i) {
      const int idx = lane + 32 * i;
      stg_stream_pred(reinterpret_cast<uint4*>(dt) + idx, bk[i], idx < pieces);
      stg_stream_pred(reinterpret_cast<uint4*>(dt + kBlockSize * D) + idx, bv[i], idx < pieces);
    }
  } else {
    constexpr int kPiecesPerRow = D / 16;
    constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;
    const uint8_t* st = reinterpret_cast<const uint8_t*>(p.src_kv) +
                        ((layer * p.src_num_blocks + sblk) * p.num_kv_heads + x.h) * fp8_tile_bytes<D>();
    uint8_t* dt = reinterpret_cast<uint8_t*>(p.kv) + ((layer * p.num_blocks + dblk) * p.num_kv_heads + x.h) * fp8_tile_bytes<D>();
    const int pieces = rows * kPiecesPerRow;
    uint4 bk[kMaxPerLane], bv[kMaxPerLane];
#pragma unroll
    for (int i = 0; i < kMaxPerLane; ++i) {
      const int idx = lane + 32 * i;
      bk[i] = ldg_copy_pred(st + idx * 16, idx < pieces);
      bv[i] = ldg_copy_pred(st + kBlockSize * D + idx * 16, idx < pieces);
    }
    const uint2 sc = ldg_copy8_pred(st + 2 * kBlockSize * D + lane * 8, lane < rows);
#pragma unroll
    for (int i = 0; i < kMaxPerLane; ++i) {
      const int idx = lane + 32 * i;
      stg_stream_pred(dt + idx * 16, bk[i], idx < pieces);
      stg_stream_pred(dt + kBlockSize * D + idx * 16, bv[i], idx < pieces);
    }
    stg_stream8_pred(dt + 2 * kBlockSize * D + lane * 8, sc, lane < rows);
  }
  if (x.ll == 0 && x.h == 0 && lane == 0)                       // consumer's device block_table mirror
    p.block_table[static_cast<int64_t>(x.r.slot) * p.bt_stride + x.lb] = dblk;
}

}  // namespace kvp
