// kv_attn_stream.cuh — a4 (+ a3, a5): split-KV paged decode attention as ONE tile stream per warp.
//
// Same arithmetic, tiles and register-direct MMA fragments as attn_splitkv_kernel (kv_kernels.cuh);
// what changes is the control structure.  attn_splitkv_kernel finishes a work unit (epilogue, fence,
// arrival atomic, maybe the merge), THEN claims the next one and walks atomic -> work item -> block
// ids -> first tile, four dependent memory latencies (~2.7 us measured) during which the warp has
// nothing in flight: 10 % of a 27 us unit, and most of the time of a short request.  Here a warp
// sees its units as one flat sequence of KV tiles and keeps a PRODUCER cursor two tiles ahead of
// the CONSUMER cursor across unit boundaries:
//
//     producer (issue):   loads tile k+2 into the buffer the consumer just released; when it steps
//                         into a new unit it stages that unit's q rows into shared memory with
//                         cp.async, and it walks the claim -> work item -> block ids chain of the
//                         unit AFTER that one stage per tile, so no dependent load is ever waited on
//     consumer (consume): S^T = K q^T, online softmax, O^T += V^T P^T on tile k; at a unit's last
//                         tile it runs the epilogue while tiles k+1, k+2 (already the next unit's)
//                         are in flight
//
// Up to three units are alive per warp (consumer's, and two ahead): their descriptors wait in a
// two-entry shift register of lane-distributed words (one register each), their q in a ring of three
// shared-memory slots.  q fragments are re-read from shared memory per tile (rows padded to
// D*2 + 64 bytes: conflict-free LDS.128), which frees the 16 registers that paid for the cursors.
#pragma once

#include "kv_kernels.cuh"

namespace kvp {

__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t smem_addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(smem_addr));
  return r;
}

constexpr int kQSlots = 3;  // units alive per warp: the consumer's and two ahead

template <int D>
struct QSmem {
  static constexpr int kRowBytes = D * 2 + 64;        // 320 B at D = 128: quarter-warps hit 32 distinct banks
  static constexpr int kSlotBytes = 8 * kRowBytes;    // up to 8 heads of a GQA group
  static constexpr int kWarpBytes = kQSlots * kSlotBytes;
};

// Lane-distributed unit descriptor: lanes 0..7 hold the eight words of the WorkItemDev, lane 8 the kv
// head, lane 9 the validity flag.  One register per unit.
__device__ __forceinline__ int32_t fetch_unit_word(const AttnParams& p, int item, int lane) {
  const bool valid = item < p.n_units;
  const int h = valid ? item % p.num_kv_heads : 0;
  int32_t d = 0;
  if (valid && lane < 8) d = __ldg(reinterpret_cast<const int32_t*>(p.items + item / p.num_kv_heads) + lane);
  if (lane == 8) d = h;
  if (lane == 9) d = valid ? 1 : 0;
  return d;
}


template <int D, bool kAppend>
__global__ void __launch_bounds__(kAttnThreads, 2) attn_stream_kernel(const AttnParams p) {
  constexpr int KJ = D / 32;   // K vectors per row per thread
  constexpr int MT = D / 16;   // MMA m-tiles of O^T = V^T P^T
  constexpr int NE = D / 8;    // d columns owned per thread and head
  constexpr int64_t kTileElems = 2 * kBlockSize * D;
  constexpr unsigned kFull = 0xffffffffu;
  using QS = QSmem<D>;
  __shared__ __align__(16) unsigned char q_smem[kAttnWarps * QS::kWarpBytes];

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane >> 2, c = lane & 3;
  const int G = p.group;
  const int64_t blk_stride = static_cast<int64_t>(p.num_kv_heads) * kTileElems;
  const uint32_t q_base = static_cast<uint32_t>(__cvta_generic_to_shared(q_smem)) + warp * QS::kWarpBytes;
  const int n_warps = gridDim.x * kAttnWarps;

  // ---- N: the unit after the producer's, fetched one dependent load per issued tile ----------
  int n_claim = blockIdx.x * kAttnWarps + warp;  // first unit: the global warp index, no atomic
  int32_t n_desc = 0, n_ids = 0;
  int n_stage = 1;                               // 1: claimed, 2: descriptor requested, 3: block ids requested
  auto n_step = [&]() {
    if (n_stage == 1) {
      n_claim = __shfl_sync(kFull, n_claim, 0);
      n_desc = fetch_unit_word(p, n_claim, lane);
      n_stage = 2;
    } else if (n_stage == 2) {
      const int slot = __shfl_sync(kFull, n_desc, 1), blk_begin = __shfl_sync(kFull, n_desc, 2);
      const int nb = __shfl_sync(kFull, n_desc, 3), valid = __shfl_sync(kFull, n_desc, 9);
      n_ids = (valid && lane < nb) ? __ldg(p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin + lane) : 0;
      n_stage = 3;
    }
  };

  // ---- P: producer cursor -----------------------------------------------------------------
  bool p_valid = true, p_special = false;
  int p_t = 0, p_nblocks = 0, p_ntok = 0, p_qslot = 0;
  int32_t p_desc = 0, p_ids = 0, p_ids_next = 0;
  const int32_t* p_bt = p.block_table;
  uint16_t* p_kvh = p.kv_layer;
  // units whose first tile has been issued but which the consumer has not started
  int32_t dq0 = 0, dq1 = 0;
  int dq_cnt = 0;

  auto p_advance = [&]() {
    while (n_stage < 3) n_step();                // only a unit shorter than two tiles makes this wait
    p_desc = n_desc;
    p_valid = __shfl_sync(kFull, p_desc, 9) != 0;
    if (!p_valid) return;
    const int batch_idx = __shfl_sync(kFull, p_desc, 0), slot = __shfl_sync(kFull, p_desc, 1);
    const int blk_begin = __shfl_sync(kFull, p_desc, 2), chunks = __shfl_sync(kFull, p_desc, 6);
    const int h = __shfl_sync(kFull, p_desc, 8);
    p_nblocks = __shfl_sync(kFull, p_desc, 3);
    p_ntok = __shfl_sync(kFull, p_desc, 4);
    p_special = kAppend && (chunks & 0xffff) == (chunks >> 16) - 1;
    p_kvh = p.kv_layer + static_cast<int64_t>(h) * kTileElems;
    p_bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
    p_ids = n_ids;
    p_t = 0;
    {  // q rows of the G heads of this (request, kv head) -> shared-memory slot p_qslot
      const uint16_t* qrow = p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G) * D;
      const uint32_t dst = q_base + p_qslot * QS::kSlotBytes;
#pragma unroll
      for (int r = 0; r < (8 * NE) / 32; ++r) {
        const int i = lane + 32 * r, head = i / NE, col = i % NE;
        if (head < G) cp_async16(dst + head * QS::kRowBytes + col * 16, qrow + head * D + col * 8);
      }
      cp_async_commit();
      p_qslot = p_qslot == kQSlots - 1 ? 0 : p_qslot + 1;
    }
    if (dq_cnt == 0) dq0 = p_desc; else dq1 = p_desc;
    ++dq_cnt;
    if (lane == 0) n_claim = n_warps + atomicAdd(&p.counters[0], 1);
    n_stage = 1;
  };

  auto issue = [&](KVTile<D>& T) {
    if (!p_valid) return;
    if (p_t == p_nblocks) {
      p_advance();
      if (!p_valid) return;
    } else if (n_stage < 3) {
      n_step();
    }
    const int v = p_t++;
    if (p_special && v == 0) {
      const int batch_idx = __shfl_sync(kFull, p_desc, 0), last_blk = __shfl_sync(kFull, p_desc, 7);
      const int h = __shfl_sync(kFull, p_desc, 8);
      const int64_t row = (static_cast<int64_t>(batch_idx) * p.num_kv_heads + h) * D;
      load_tile_append<D>(T, p_kvh + last_blk * blk_stride, p.k_new + row, p.v_new + row,
                          p_ntok - (p_nblocks - 1) * kBlockSize, g, c);
      return;
    }
    const int t = p_special ? v - 1 : v;
    if ((t & 31) == 0 && t > 0) p_ids = p_ids_next;
    if ((t & 31) == 8 && t + 24 + lane < p_nblocks) p_ids_next = __ldg(p_bt + t + 24 + lane);
    const int blk = __shfl_sync(kFull, p_ids, t & 31);
    load_tile<D>(T, p_kvh + blk * blk_stride, p_ntok - t * kBlockSize, g, c);
  };

  // ---- C: consumer cursor -----------------------------------------------------------------
  bool c_valid = true, c_special = false;
  int c_t = 0, c_nblocks = 0, c_ntok = 0, c_qslot = kQSlots - 1;
  int32_t c_desc = 0;
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // heads 2c, 2c+1 (l: this lane's rows only)
  float o[MT][4];

  auto c_start = [&]() {                         // pop the next unit; wait for its q rows
    if (dq_cnt == 0) { c_valid = false; return; }
    c_desc = dq0;
    dq0 = dq1;
    --dq_cnt;
    c_nblocks = __shfl_sync(kFull, c_desc, 3);
    c_ntok = __shfl_sync(kFull, c_desc, 4);
    const int chunks = __shfl_sync(kFull, c_desc, 6);
    c_special = kAppend && (chunks & 0xffff) == (chunks >> 16) - 1;
    c_qslot = c_qslot == kQSlots - 1 ? 0 : c_qslot + 1;
    c_t = 0;
    if (dq_cnt == 0) cp_async_wait<0>();         // groups committed after this unit's may stay pending
    else if (dq_cnt == 1) cp_async_wait<1>();
    else cp_async_wait<2>();
    __syncwarp();
    m0 = m1 = -INFINITY;
    l0 = l1 = 0.f;
#pragma unroll
    for (int i = 0; i < MT; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
  };

  auto epilogue = [&]() {
    const int batch_idx = __shfl_sync(kFull, c_desc, 0), pb = __shfl_sync(kFull, c_desc, 5);
    const int chunks = __shfl_sync(kFull, c_desc, 6), h = __shfl_sync(kFull, c_desc, 8);
    const int n_chunks = chunks >> 16, chunk_idx = chunks & 0xffff;
    const int pbase = pb < 0 ? -1 : pb + h * n_chunks;         // first partial slot of (request, kv head)
    const int pidx = pb < 0 ? -1 : pbase + chunk_idx;
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {                    // finish l over the token lanes
      l0 += __shfl_xor_sync(kFull, l0, off);
      l1 += __shfl_xor_sync(kFull, l1, off);
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
    // fused a5: the unit that completes its (request, kv head) merges the partials
    if (pidx >= 0 && p.fuse_combine) {
      __threadfence();                                           // this lane's partial stores, device-wide
      __syncwarp();
      int last = 0;
      if (lane == 0) {
        last = atomicAdd(&p.arrive[pbase], 1) == n_chunks - 1;
        if (last) p.arrive[pbase] = 0;                           // ready for the next launch
      }
      last = __shfl_sync(kFull, last, 0);
      if (last) {
        __threadfence();
        combine_group<D>(p.part_o, p.part_ml, pbase, n_chunks, G,
                         p.out + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G) * D, lane);
      }
    }
  };

  auto consume = [&](const KVTile<D>& T) {
    const int v = c_t;
    const int t = c_special ? (v == 0 ? c_nblocks - 1 : v - 1) : v;   // real tile index inside the unit
    const int nv = c_ntok - t * kBlockSize;
    // ---- S^T = K q^T : two independent accumulation chains; q fragments from shared memory ----
    float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
    const uint32_t qaddr = q_base + c_qslot * QS::kSlotBytes + g * QS::kRowBytes + c * 16;
#pragma unroll
    for (int j = 0; j < KJ; ++j) {
      uint4 qv = make_uint4(0u, 0u, 0u, 0u);
      if (g < G) qv = lds128(qaddr + j * 64);                  // head g, column chunk c + 4j
      mma_bf16_m16n8k16(sa, T.k[0][j].x, T.k[1][j].x, T.k[0][j].y, T.k[1][j].y, qv.x, qv.y);
      mma_bf16_m16n8k16(sb, T.k[0][j].z, T.k[1][j].z, T.k[0][j].w, T.k[1][j].w, qv.z, qv.w);
    }
    float s[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) s[i] = (sa[i] + sb[i]) * p.scale_log2;
    if (nv < kBlockSize) {                                      // ragged last block: mask by index, not value
      if (g >= nv) s[0] = s[1] = -INFINITY;
      if (g + 8 >= nv) s[2] = s[3] = -INFINITY;
    }
    // ---- online softmax over the token axis (= across the 8 lanes sharing c) ----
    float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {
      mx0 = fmaxf(mx0, __shfl_xor_sync(kFull, mx0, off));
      mx1 = fmaxf(mx1, __shfl_xor_sync(kFull, mx1, off));
    }
    const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);     // finite: every tile has >= 1 valid token
    const float a0 = fast_exp2(m0 - mn0), a1 = fast_exp2(m1 - mn1);
    m0 = mn0; m1 = mn1;
    const float p0 = fast_exp2(s[0] - mn0), p1 = fast_exp2(s[1] - mn1);
    const float p2 = fast_exp2(s[2] - mn0), p3 = fast_exp2(s[3] - mn1);
    l0 = l0 * a0 + (p0 + p2);
    l1 = l1 * a1 + (p1 + p3);
#pragma unroll
    for (int i = 0; i < MT; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
    // P^T as the B fragment, bf16 hi + bf16 lo (see attn_splitkv_kernel)
    const uint32_t ph01 = pack_bf16x2(p0, p1), ph23 = pack_bf16x2(p2, p3);
    const uint32_t pl01 = pack_bf16x2(p0 - __uint_as_float(ph01 << 16), p1 - __uint_as_float(ph01 & 0xffff0000u));
    const uint32_t pl23 = pack_bf16x2(p2 - __uint_as_float(ph23 << 16), p3 - __uint_as_float(ph23 & 0xffff0000u));
    const uint32_t b0 = movmatrix_trans(ph01), b1 = movmatrix_trans(ph23);
    const uint32_t c0 = movmatrix_trans(pl01), c1 = movmatrix_trans(pl23);
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
    if (c_special && v == 0) {                                  // a3: the appended row goes into the pool
      const int slot = __shfl_sync(kFull, c_desc, 1), blk_begin = __shfl_sync(kFull, c_desc, 2);
      const int last_blk = __shfl_sync(kFull, c_desc, 7), h = __shfl_sync(kFull, c_desc, 8);
      store_new_row<D>(T, p.kv_layer + static_cast<int64_t>(h) * kTileElems + last_blk * blk_stride, nv, g, c);
      if (h == 0 && lane == 0)
        p.block_table[static_cast<int64_t>(slot) * p.bt_stride + blk_begin + c_nblocks - 1] = last_blk;
    }
    if (++c_t == c_nblocks) {
      epilogue();
      c_start();
    }
  };

  KVTile<D> A, B;
  issue(A);
  issue(B);
  c_start();
  while (c_valid) {
    consume(A);
    issue(A);
    if (!c_valid) break;
    consume(B);
    issue(B);
  }

  // Last CTA out rewinds the work counter for the next launch (launches on one pool are
  // stream-ordered; counters[1] wraps to 0 by itself).
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned prev = atomicInc(reinterpret_cast<unsigned*>(&p.counters[1]), gridDim.x - 1);
    if (prev == gridDim.x - 1) p.counters[0] = 0;
  }
}

}  // namespace kvp
