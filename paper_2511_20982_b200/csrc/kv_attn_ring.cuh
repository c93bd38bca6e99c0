// kv_attn_ring.cuh — a4 (+ a3, a5): attn_splitkv_kernel's arithmetic with the KV tiles staged through a
// per-warp shared-memory ring instead of register tile buffers (the design that paid +13-15 % on the FP8
// pool, kv_fp8.cuh): 16-byte cp.async copies, zero-filled past the request's end, XOR-swizzled chunks so that
// both fragment access patterns are bank-conflict free, no block-wide barrier.  Without 128 tile registers
// the kernel fits 3 CTAs = 12 warps per SM, which is what hides the unit switches (claim -> work item ->
// block ids -> first tile) that cost the register kernel its last few percent on short launches.
// The fused append sources the new token's row straight from k_new / v_new into the ring and copies it
// global -> global into the pool.
#pragma once

#include "kv_kernels.cuh"

namespace kvp {

__device__ __forceinline__ uint4 lds128_16(uint32_t smem_addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(smem_addr));
  return r;
}

// byte offset of 16-byte chunk `chunk` of bf16 row `row` inside a K or V half of a ring slot:
// chunk' = chunk ^ (row bit 1) << 1 ^ (row bit 2 ^ row bit 0) << 2
template <int D>
__device__ __forceinline__ uint32_t ring_chunk_off16(int row, int chunk) {
  return row * (D * 2) + ((chunk ^ (((row >> 1) & 1) << 1) ^ ((((row >> 2) ^ row) & 1) << 2)) << 4);
}

template <int D, bool kAppend, bool kVarQ, int R, int kCtas>
__global__ void __launch_bounds__(kAttnThreads, kCtas) attn_ring_kernel(const AttnParams p) {
  extern __shared__ __align__(128) unsigned char ring_smem16[];
  constexpr uint32_t kTileB = 2 * kBlockSize * D * 2;           // bytes of a (block, kv head) tile
  const uint32_t ring = static_cast<uint32_t>(__cvta_generic_to_shared(ring_smem16)) + (threadIdx.x >> 5) * (R * kTileB);
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

    uint16_t* last_tile = kvh + last_blk * blk_stride;
    // start the copies of virtual tile v into ring slot v % R (one cp.async group per tile, empty past the end).
    // virtual tile v -> real tile: special ? (v == 0 ? n_blocks - 1 : v - 1) : v
    auto issue = [&](int v) {
      if (v < n_blocks) {
        const bool first_special = special && v == 0;
        const int t = first_special ? n_blocks - 1 : v - sp;
        const uint16_t* tile;
        if (first_special) {
          tile = last_tile;
        } else {
          if ((t & 31) == 0 && t > 0) ids = ids_next;
          if ((t & 31) == 8 && t + 24 + lane < n_blocks) ids_next = __ldg(bt + t + 24 + lane);
          tile = kvh + __shfl_sync(0xffffffffu, ids, t & 31) * blk_stride;
        }
        const uint32_t slot_addr = ring + (v % R) * kTileB;
        const int nv = n_tokens - t * kBlockSize;
        const int r_new = first_special ? nv - 1 : -1;           // fused append: that row comes from k_new / v_new
        const int64_t new_row = (static_cast<int64_t>(batch_idx) * p.num_kv_heads + h) * D;
        constexpr int kCh = D / 8;                                // 16-byte chunks per row
#pragma unroll
        for (int i = 0; i < 2 * kBlockSize * kCh / 32; ++i) {
          const int idx = lane + 32 * i, row32 = idx / kCh, ch = idx % kCh, row = row32 & (kBlockSize - 1);
          const uint16_t* srcp = tile + idx * 8;
          if (kAppend && row == r_new) srcp = ((row32 >> 4) ? p.v_new : p.k_new) + new_row + ch * 8;
          const int sz = row < nv ? 16 : 0;                       // zero-fill rows past the end
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(slot_addr + (row32 >> 4) * (kBlockSize * D * 2) +
                                                                          ring_chunk_off16<D>(row, ch)),
                       "l"(srcp), "r"(sz) : "memory");
        }
        if (kAppend && first_special) {                           // a3: the new row goes into the pool (global -> global)
          if (lane < 2 * kCh) {
            const int cc = lane / kCh, ch = lane % kCh;
            const uint4 x = ldg_stream((cc ? p.v_new : p.k_new) + new_row + ch * 8);
            *reinterpret_cast<uint4*>(last_tile + cc * (kBlockSize * D) + r_new * D + ch * 8) = x;
          }
          if (h == 0 && lane == 0) p.block_table[static_cast<int64_t>(slot) * p.bt_stride + blk_begin + n_blocks - 1] = last_blk;
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    };

    auto consume = [&](int v) {
      const int t = (special && v == 0) ? n_blocks - 1 : v - sp;
      KVTile<D> T;                                               // fragments of ring slot v % R
      {
        const uint32_t slot_addr = ring + (v % R) * kTileB;
#pragma unroll
        for (int rs = 0; rs < 2; ++rs)
#pragma unroll
          for (int j = 0; j < KJ; ++j) T.k[rs][j] = lds128_16(slot_addr + ring_chunk_off16<D>(g + 8 * rs, c + 4 * j));
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int cs = 0; cs < D / 64; ++cs)
            T.v[i][cs] = lds128_16(slot_addr + kBlockSize * D * 2 + ring_chunk_off16<D>(2 * c + (i & 1) + 8 * (i >> 1), g + 8 * cs));
      }
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

#pragma unroll
    for (int v = 0; v < R - 1; ++v) issue(v);                    // R - 1 tiles ahead
    for (int v = 0; v < n_blocks; ++v) {
      asm volatile("cp.async.wait_group %0;" ::"n"(R - 2) : "memory");   // tile v has landed (this lane's copies)
      __syncwarp();                                              // ... everyone's; and slot (v - 1) % R is free
      issue(v + R - 1);
      consume(v);
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();

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

}  // namespace kvp
