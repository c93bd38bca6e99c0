// kv_fp8.cuh — NEXT-2: the FP8 (e4m3) KV pool.  The paper's models are FP8 and the KV
// bytes per token are the denominator of Eq. 13: an FP8 pool holds and streams twice the
// tokens per byte.  Quantisation (C1-C4; the paper fixes none): per token row of one
// (layer, kv head, K|V)   amax = max |x_j|,  scale = fl32(amax / 448),  inv = fl32(448 / amax)
// (both 1 when amax = 0),  code_j = RNE_e4m3(fl32(x_j * inv)),  x^_j = e4m3(code_j) * scale.
// Per-TOKEN scales (not per block): a decode step appends one token to a partly filled block, and a
// block-wide scale would have to re-quantise the block's older tokens.
//
// Tile of one (layer, block, kv head), 32 D + 128 bytes:  K8[16][D] | V8[16][D] | sc[16] {ks_t, vs_t} fp32.
//
//   ingest_fp8_kernel<D>                          quantising scatter (a2 / a3 for an FP8 pool)
//   attn_fp8_ring_kernel<D, R, kAppend, kVarQ>    split-KV paged attention over an FP8 pool (a4 + a5 [+ a3], NEXT-1 rows):
//                                                 the default — tiles staged through a per-warp cp.async shared-memory ring
//   attn_fp8_kernel<D>                            the first version (option fp8_ring = 0): tiles in register buffers, decode only
//
// Both attention kernels keep the fragment mapping of the bf16 kernels (16 tokens on M, the <= 8 heads of the
// group on N, a fragment register is a plain 16-byte piece of a K or V row, turned into f16x2 by one
// F2FP.F16.E4M3.UNPACK per code pair) and run the MMAs in f16: e4m3 -> f16 is exact and one instruction.
//   * q rows are pre-scaled by a power of two so their largest element lies in [1, 2) and converted to
//     f16 (exact for every element within 2^-14 of the row maximum); the factor returns through the
//     per-column score scale.
//   * the score of token t is (K8_t . q~) * ks_t * scale; the V scale is folded into the softmax
//     REFERENCE rather than into the weights: the running maximum m' is taken over s_t + log2(vs_t),
//     so the weights fed to the PV MMA, p'_t = 2^(s_t + log2 vs_t - m') = p_t * vs_t, lie in (0, 1]
//     whatever the magnitude of V — no f16 overflow or underflow to manage — while l accumulates
//     p'_t / vs_t.  O and l share the reference m', so O / l and the LSE merge are unchanged.
#pragma once

#include <cuda_fp16.h>

#include "kv_kernels.cuh"

namespace kvp {

__device__ __forceinline__ uint2 ldg_stream8_pred(const void* ptr, bool pred) {
  uint2 r = make_uint2(0u, 0u);
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\t"
      "@p ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];\n\t}"
      : "+r"(r.x), "+r"(r.y)
      : "l"(ptr), "r"(static_cast<int>(pred)));
  return r;
}

__device__ __forceinline__ uint4 lds128(uint32_t smem_addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(smem_addr));
  return r;
}

// two e4m3 codes (low 16 bits / high 16 bits of w) -> f16x2, exact
__device__ __forceinline__ uint32_t e4m3x2_lo_to_f16x2(uint32_t w) {
  uint32_t d;
  asm("{\n\t.reg .b16 lo, hi;\n\tmov.b32 {lo, hi}, %1;\n\tcvt.rn.f16x2.e4m3x2 %0, lo;\n\t}" : "=r"(d) : "r"(w));
  return d;
}
__device__ __forceinline__ uint32_t e4m3x2_hi_to_f16x2(uint32_t w) {
  uint32_t d;
  asm("{\n\t.reg .b16 lo, hi;\n\tmov.b32 {lo, hi}, %1;\n\tcvt.rn.f16x2.e4m3x2 %0, hi;\n\t}" : "=r"(d) : "r"(w));
  return d;
}

// fl32 pair -> two e4m3 codes, RNE, saturating: low byte = code(lo), high byte = code(hi)
__device__ __forceinline__ uint32_t f32x2_to_e4m3x2(float lo, float hi) {
  uint16_t d;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(d) : "f"(hi), "f"(lo));
  return d;
}

__device__ __forceinline__ uint32_t pack_f16x2(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

__device__ __forceinline__ float fast_log2(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// D(16x8, f32) += A(16x16, f16, row) * B(16x8, f16, col)
__device__ __forceinline__ void mma_f16_m16n8k16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                                 uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

template <int D>
__host__ __device__ constexpr int64_t fp8_tile_bytes() { return 32 * D + 128; }

// ---------------------------------------------------------------------------------------------
// quantising scatter: same units, same descriptors as ingest_kernel (IngestParams::kv = the FP8 region),
// but one warp per (unit, K|V): the quantisation arithmetic sits between a warp's loads and its stores,
// so the kernel wants many light warps (4 KiB in flight each, ~50 registers) rather than few heavy ones.
// Launch with 2 * total_units warps.
// ---------------------------------------------------------------------------------------------
constexpr int kIngest8Threads = 64;   // small CTAs: an SM slot frees as soon as two warps are done (one-shot warps of uneven length)
constexpr int kIngest8Warps = kIngest8Threads / 32;
template <int D>
__global__ void __launch_bounds__(kIngest8Threads) ingest_fp8_kernel(const IngestParams p) {
  constexpr int kPiecesPerRow = D / 8;                          // 16-byte source pieces (8 bf16) per token row
  constexpr int kMaxPerLane = kBlockSize * kPiecesPerRow / 32;  // 8 at D=128, 4 at D=64
  const int lane = threadIdx.x & 31;
  const int64_t u2 = static_cast<int64_t>(blockIdx.x) * kIngest8Warps + (threadIdx.x >> 5);
  const int64_t u = u2 >> 1;
  const int c = static_cast<int>(u2 & 1);                        // 0: the K rows of the unit, 1: the V rows
  if (u >= p.total_units) return;

  // request of this unit: last i with unit_begin <= u.  The lanes test 32 candidates at a time (independent
  // loads, one ballot each) instead of walking a binary search of dependent loads: the warp's few-hundred-cycle
  // quantisation already sits between its loads and its stores, so its prologue should not add more dead time.
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
  const int lb = r.blk0 + jj;                                   // logical block
  const int row0 = (jj == 0) ? (r.start_pos & (kBlockSize - 1)) : 0;
  const int row1 = min(kBlockSize, r.start_pos + r.n_tokens - lb * kBlockSize);
  const int t0 = lb * kBlockSize + row0 - r.start_pos;          // first source token of this unit
  const int pieces = (row1 - row0) * kPiecesPerRow;

  const int64_t src_off = ((static_cast<int64_t>(ll) * p.src_kv_heads + p.src_head_begin + h) * r.n_tokens + t0) * D;
  const uint4* lin = reinterpret_cast<const uint4*>(reinterpret_cast<const uint16_t*>(c ? r.v_src : r.k_src) + src_off);
  uint8_t* tile = reinterpret_cast<uint8_t*>(p.kv) +
                  ((static_cast<int64_t>(p.layer_begin + ll) * p.num_blocks + blk) * p.num_kv_heads + h) * fp8_tile_bytes<D>();

  uint4 buf[kMaxPerLane];
#pragma unroll
  for (int i = 0; i < kMaxPerLane; ++i) buf[i] = ldg_copy_pred(lin + lane + 32 * i, lane + 32 * i < pieces);   // all loads first
#pragma unroll
  for (int i = 0; i < kMaxPerLane; ++i) {
    const int idx = lane + 32 * i;
    const bool ok = idx < pieces;
    const int row = row0 + idx / kPiecesPerRow, cp = idx % kPiecesPerRow;
    const uint4 x = buf[i];
    // row amax: bf16 magnitudes compare like unsigned integers
    uint32_t mx = __vmaxu2(__vmaxu2(x.x & 0x7fff7fffu, x.y & 0x7fff7fffu), __vmaxu2(x.z & 0x7fff7fffu, x.w & 0x7fff7fffu));
    mx = max(mx & 0xffffu, mx >> 16);
#pragma unroll
    for (int off = kPiecesPerRow / 2; off > 0; off >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    const float amax = __uint_as_float(mx << 16);
    const float scale = mx == 0 ? 1.f : __fdiv_rn(amax, 448.f);
    const float inv = mx == 0 ? 1.f : __fdiv_rn(448.f, amax);
    uint32_t w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t e = u4_get(x, k);
      w[k] = f32x2_to_e4m3x2(__fmul_rn(__uint_as_float(e << 16), inv), __fmul_rn(__uint_as_float(e & 0xffff0000u), inv));
    }
    if (ok) {
      uint8_t* dst = tile + c * (kBlockSize * D) + row * D + cp * 8;
      *reinterpret_cast<uint2*>(dst) = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
      if (cp == 0) *reinterpret_cast<float*>(tile + 2 * kBlockSize * D + row * 8 + c * 4) = scale;
    }
  }
  if (c == 0 && ll == 0 && h == 0 && lane == 0)                 // device block_table mirror (a1, device half)
    p.block_table[static_cast<int64_t>(r.slot) * p.bt_stride + lb] = blk;
}

// ---------------------------------------------------------------------------------------------
// split-KV paged decode attention over an FP8 pool
// ---------------------------------------------------------------------------------------------

template <int D>
struct KV8Tile {
  uint4 k[2][D / 64];      // rows g, g+8; 16 codes at column chunk c + 4j: word w of vector j = k-step 4j + w
  uint32_t v[4][D / 32];   // rows 2c, 2c+1, 2c+8, 2c+9; the lane's D/8 columns g*(D/8) ...
  float2 sc[2];            // (ks, vs) of tokens g, g+8
};

template <int D>
__device__ __forceinline__ void load_tile8(KV8Tile<D>& T, const uint8_t* tile, int nv, int g, int c) {
#pragma unroll
  for (int rs = 0; rs < 2; ++rs) {
    const int row = g + 8 * rs;
    const bool ok = row < nv;
#pragma unroll
    for (int j = 0; j < D / 64; ++j) T.k[rs][j] = ldg_stream_pred(tile + row * D + (c + 4 * j) * 16, ok);
    const uint2 s = ldg_stream8_pred(tile + 2 * kBlockSize * D + row * 8, ok);
    T.sc[rs] = make_float2(__uint_as_float(s.x), __uint_as_float(s.y));
  }
  const uint8_t* vp = tile + kBlockSize * D + g * (D / 8);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = 2 * c + (i & 1) + 8 * (i >> 1);
    const bool ok = row < nv;
    if constexpr (D == 128) {
      const uint4 x = ldg_stream_pred(vp + row * D, ok);
      T.v[i][0] = x.x; T.v[i][1] = x.y; T.v[i][2] = x.z; T.v[i][3] = x.w;
    } else {
      const uint2 x = ldg_stream8_pred(vp + row * D, ok);
      T.v[i][0] = x.x; T.v[i][1] = x.y;
    }
  }
}

template <int D>
__global__ void __launch_bounds__(kAttnThreads, 2) attn_fp8_kernel(const AttnParams p) {
  constexpr int KS = D / 16;   // MMA k-steps of S^T = K q^T
  constexpr int MT = D / 16;   // MMA m-tiles of O^T = V^T P^T
  constexpr int NE = D / 8;    // d columns owned per lane: g * NE + e
  constexpr int64_t kTile = fp8_tile_bytes<D>();
  constexpr unsigned kFull = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int g = lane >> 2, c = lane & 3;
  const int G = p.group;
  const int64_t blk_stride = static_cast<int64_t>(p.num_kv_heads) * kTile;
  const uint8_t* kv8 = reinterpret_cast<const uint8_t*>(p.kv_layer);

  const int n_warps = gridDim.x * kAttnWarps;
  for (int item = blockIdx.x * kAttnWarps + (threadIdx.x >> 5);;) {
    if (item >= p.n_units) break;
    const int h = item % p.num_kv_heads;
    const int4* wi = reinterpret_cast<const int4*>(p.items) + (item / p.num_kv_heads) * 2;
    const int4 w0 = __ldg(wi);
    const int4 w1 = __ldg(wi + 1);
    const int batch_idx = w0.x, slot = w0.y, blk_begin = w0.z, n_blocks = w0.w;
    const int n_tokens = w1.x;
    const int n_chunks = w1.z >> 16, chunk_idx = w1.z & 0xffff;
    const int pbase = w1.y < 0 ? -1 : w1.y + h * n_chunks;     // first partial slot of (request, kv head)
    const int pidx = w1.y < 0 ? -1 : pbase + chunk_idx;

    // q^T as f16 B fragments: lane (g, c) holds head g, d columns (c + 4j) * 16 + [0, 16), scaled by a
    // power of two so that the row maximum lies in [1, 2); cs0 / cs1 give the factor back to the scores
    uint32_t qf[KS][2];
    float cs0, cs1;
    {
      const bool ok = g < G;
      const uint16_t* qp = p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + (ok ? g : 0)) * D + c * 16;
      uint4 raw[D / 64][2];
      uint32_t mx = 0;
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          raw[j][k] = ldg_stream_pred(qp + j * 64 + k * 8, ok);
          mx = __vmaxu2(mx, __vmaxu2(__vmaxu2(raw[j][k].x & 0x7fff7fffu, raw[j][k].y & 0x7fff7fffu),
                                     __vmaxu2(raw[j][k].z & 0x7fff7fffu, raw[j][k].w & 0x7fff7fffu)));
        }
      mx = max(mx & 0xffffu, mx >> 16);
      mx = max(mx, __shfl_xor_sync(kFull, mx, 1));
      mx = max(mx, __shfl_xor_sync(kFull, mx, 2));
      const uint32_t eb = min(max(mx >> 7, 1u), 253u);           // biased exponent of the row maximum
      const float sf = __uint_as_float((254u - eb) << 23);        // 2^(127 - eb)
      const float back = __uint_as_float(eb << 23) * p.scale_log2;
      cs0 = __shfl_sync(kFull, back, (2 * c) * 4);
      cs1 = __shfl_sync(kFull, back, (2 * c + 1) * 4);
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
          for (int w = 0; w < 4; w += 2) {                       // words (w, w+1) = 4 bf16 = one k-step's (b0, b1)
            const uint32_t e0 = u4_get(raw[j][k], w), e1 = u4_get(raw[j][k], w + 1);
            qf[4 * j + 2 * k + w / 2][0] = pack_f16x2(__uint_as_float(e0 << 16) * sf, __uint_as_float(e0 & 0xffff0000u) * sf);
            qf[4 * j + 2 * k + w / 2][1] = pack_f16x2(__uint_as_float(e1 << 16) * sf, __uint_as_float(e1 & 0xffff0000u) * sf);
          }
    }

    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // heads 2c, 2c+1 (l: this lane's rows only)
    float o[MT][4];
#pragma unroll
    for (int i = 0; i < MT; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;

    const int32_t* bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
    const uint8_t* kvh = kv8 + static_cast<int64_t>(h) * kTile;
    int32_t ids = lane < n_blocks ? __ldg(bt + lane) : 0;       // physical ids of blocks [32k, 32k+32)
    int32_t ids_next = 0;

    auto issue = [&](KV8Tile<D>& T, int t) {                    // start the loads of tile t
      if ((t & 31) == 0 && t > 0) ids = ids_next;
      if ((t & 31) == 8 && t + 24 + lane < n_blocks) ids_next = __ldg(bt + t + 24 + lane);
      const int blk = __shfl_sync(kFull, ids, t & 31);
      load_tile8<D>(T, kvh + blk * blk_stride, n_tokens - t * kBlockSize, g, c);
    };

    auto consume = [&](const KV8Tile<D>& T, int t) {
      // ---- S^T = K8 q~^T : word w of vector j feeds k-step 4j + w; two accumulation chains ----
      float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          const uint32_t r0 = u4_get(T.k[0][j], w), r1 = u4_get(T.k[1][j], w);
          mma_f16_m16n8k16((w & 1) ? sb : sa, e4m3x2_lo_to_f16x2(r0), e4m3x2_lo_to_f16x2(r1), e4m3x2_hi_to_f16x2(r0),
                           e4m3x2_hi_to_f16x2(r1), qf[4 * j + w][0], qf[4 * j + w][1]);
        }
      // s[0], s[1]: token g, heads 2c, 2c+1;  s[2], s[3]: token g+8   (log2 units)
      float s[4];
      s[0] = (sa[0] + sb[0]) * (T.sc[0].x * cs0);
      s[1] = (sa[1] + sb[1]) * (T.sc[0].x * cs1);
      s[2] = (sa[2] + sb[2]) * (T.sc[1].x * cs0);
      s[3] = (sa[3] + sb[3]) * (T.sc[1].x * cs1);
      const int nv = n_tokens - t * kBlockSize;
      const bool ok0 = g < nv, ok1 = g + 8 < nv;                 // ragged last block: mask by index, not value
      // ---- online softmax with the V scale folded into the reference: t = s + log2(vs) ----
      const float lv0 = ok0 ? fast_log2(T.sc[0].y) : -INFINITY, lv1 = ok1 ? fast_log2(T.sc[1].y) : -INFINITY;
      const float iv0 = ok0 ? __frcp_rn(T.sc[0].y) : 0.f, iv1 = ok1 ? __frcp_rn(T.sc[1].y) : 0.f;
      const float t0 = s[0] + lv0, t1 = s[1] + lv0, t2 = s[2] + lv1, t3 = s[3] + lv1;
      float mx0 = fmaxf(t0, t2), mx1 = fmaxf(t1, t3);
#pragma unroll
      for (int off = 4; off < 32; off <<= 1) {
        mx0 = fmaxf(mx0, __shfl_xor_sync(kFull, mx0, off));
        mx1 = fmaxf(mx1, __shfl_xor_sync(kFull, mx1, off));
      }
      const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);   // finite: every tile has >= 1 valid token
      const bool moved = mn0 != m0 || mn1 != m1;
      const float a0 = fast_exp2(m0 - mn0), a1 = fast_exp2(m1 - mn1);
      m0 = mn0; m1 = mn1;
      const float p0 = fast_exp2(t0 - mn0), p1 = fast_exp2(t1 - mn1);   // p'_t = p_t * vs_t  in (0, 1]
      const float p2 = fast_exp2(t2 - mn0), p3 = fast_exp2(t3 - mn1);
      l0 = l0 * a0 + (p0 * iv0 + p2 * iv1);
      l1 = l1 * a1 + (p1 * iv0 + p3 * iv1);
      if (__any_sync(kFull, moved)) {                            // the running maximum settles after a few tiles
#pragma unroll
        for (int i = 0; i < MT; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
      }
      // ---- P'^T as the f16 B fragment (11-bit weights in (0, 1]: 2^-12 relative, below the final bf16 rounding) ----
      const uint32_t b0 = movmatrix_trans(pack_f16x2(p0, p1));  // tokens 2c, 2c+1   of head g
      const uint32_t b1 = movmatrix_trans(pack_f16x2(p2, p3));  // tokens 2c+8, 2c+9 of head g
      // ---- O^T += V8^T P'^T : m-tile i takes the lane's column e = i (row g) and e = i + NE/2 (row g+8);
      // one PRMT pairs the codes of two tokens for two neighbouring columns, one F2FP per pair ----
#pragma unroll
      for (int i = 0; i < MT; i += 2) {                          // columns (i, i+1) and (i + NE/2, i + 1 + NE/2)
        const int e1 = i, e2 = i + NE / 2;
        const uint32_t sel = (e1 & 2) ? 0x7362u : 0x5140u;      // bytes (b, b+1) of both rows: [A.b, B.b, A.b+1, B.b+1]
        const uint32_t x01 = __byte_perm(T.v[0][e1 >> 2], T.v[1][e1 >> 2], sel);   // tokens 2c, 2c+1; columns e1, e1+1
        const uint32_t x23 = __byte_perm(T.v[2][e1 >> 2], T.v[3][e1 >> 2], sel);   // tokens 2c+8, 2c+9
        const uint32_t y01 = __byte_perm(T.v[0][e2 >> 2], T.v[1][e2 >> 2], sel);   // columns e2, e2+1
        const uint32_t y23 = __byte_perm(T.v[2][e2 >> 2], T.v[3][e2 >> 2], sel);
        mma_f16_m16n8k16(o[i], e4m3x2_lo_to_f16x2(x01), e4m3x2_lo_to_f16x2(y01), e4m3x2_lo_to_f16x2(x23),
                         e4m3x2_lo_to_f16x2(y23), b0, b1);
        mma_f16_m16n8k16(o[i + 1], e4m3x2_hi_to_f16x2(x01), e4m3x2_hi_to_f16x2(y01), e4m3x2_hi_to_f16x2(x23),
                         e4m3x2_hi_to_f16x2(y23), b0, b1);
      }
    };

    KV8Tile<D> A, B, C, E;
    issue(A, 0);
    if (n_blocks > 1) issue(B, 1);
    if (n_blocks > 2) issue(C, 2);
    for (int v = 0; v < n_blocks; v += 4) {
      if (v + 3 < n_blocks) issue(E, v + 3);
      consume(A, v);
      if (v + 1 < n_blocks) {
        if (v + 4 < n_blocks) issue(A, v + 4);
        consume(B, v + 1);
      }
      if (v + 2 < n_blocks) {
        if (v + 5 < n_blocks) issue(B, v + 5);
        consume(C, v + 2);
      }
      if (v + 3 < n_blocks) {
        if (v + 6 < n_blocks) issue(C, v + 6);
        consume(E, v + 3);
      }
    }

    // ---- epilogue: finish l over the token lanes, then store ----
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {
      l0 += __shfl_xor_sync(kFull, l0, off);
      l1 += __shfl_xor_sync(kFull, l1, off);
    }
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
      const int head = 2 * c + hh;
      if (head >= G) continue;
      const float l = hh ? l1 : l0, m = hh ? m1 : m0;
      // element e of this lane: d column g * NE + e, register o[e % (NE/2)][2*(e/(NE/2)) + hh]
      if (pidx < 0) {
        const float inv = 1.f / l;
        uint16_t* op = p.out + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + head) * D + g * NE;
#pragma unroll
        for (int e = 0; e < NE; e += 8) {
          uint32_t w[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int ea = e + 2 * k, eb2 = ea + 1;
            w[k] = pack_bf16x2(o[ea % (NE / 2)][2 * (ea / (NE / 2)) + hh] * inv, o[eb2 % (NE / 2)][2 * (eb2 / (NE / 2)) + hh] * inv);
          }
          *reinterpret_cast<uint4*>(op + e) = make_uint4(w[0], w[1], w[2], w[3]);
        }
      } else {
        float* po = p.part_o + (static_cast<int64_t>(pidx) * G + head) * D + g * NE;
#pragma unroll
        for (int e = 0; e < NE; e += 4) {
          float f[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) f[k] = o[(e + k) % (NE / 2)][2 * ((e + k) / (NE / 2)) + hh];
          *reinterpret_cast<float4*>(po + e) = make_float4(f[0], f[1], f[2], f[3]);
        }
        if (g == 0) *reinterpret_cast<float2*>(p.part_ml + (static_cast<int64_t>(pidx) * G + head) * 2) = make_float2(m, l);
      }
    }
    // ---- fused a5: the unit that completes its (request, kv head) merges the partials ----
    if (pidx >= 0 && p.fuse_combine) {
      __threadfence();
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
    if (lane == 0) item = n_warps + atomicAdd(&p.counters[0], 1);
    item = __shfl_sync(kFull, item, 0);
  }

  // Last CTA out rewinds the work counter for the next launch
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned prev = atomicInc(reinterpret_cast<unsigned*>(&p.counters[1]), gridDim.x - 1);
    if (prev == gridDim.x - 1) p.counters[0] = 0;
  }
}

// Shared-memory ring variant.  ncu on attn_fp8_kernel (profiles/r01) shows what half-size tiles do to the
// register-direct design: the warp spends as long computing a 4 KiB tile as the memory system needs to
// deliver it, four tile buffers (144 registers) are all the prefetch depth 254 registers can pay for, and
// 8 warps per SM cannot cover the rest — 0.88 of the copy ceiling where a load-only version of the same
// kernel reaches 1.02.  Here the tiles wait in shared memory instead: every warp owns a private ring of R
// tile slots filled by 16-byte cp.async (zero-filled for rows past the request's end), so the prefetch depth
// costs no registers, the kernel fits 3 CTAs = 12 warps per SM, and a tile is pulled into fragment
// registers only when it is consumed.  Slot layout = tile layout with the 16-byte chunks of every 128-byte
// row XOR-swizzled, chunk' = chunk ^ (row bit 1) << 1 ^ (row bit 2 ^ row bit 0) << 2, which makes both
// fragment access patterns bank-conflict free: K reads (rows g, g+1 x chunks c + 4j) and V reads
// (rows 2c + const x chunks g).  No block-wide barrier: a ring is private to its warp (cp.async groups +
// __syncwarp).
template <int D>
__device__ __forceinline__ uint32_t ring_chunk_off(int row, int chunk) {   // byte offset of a 16-byte chunk of a code row
  if constexpr (D == 128) return row * 128 + ((chunk ^ (((row >> 1) & 1) << 1) ^ ((((row >> 2) ^ row) & 1) << 2)) << 4);
  else return row * 64 + ((chunk ^ ((row >> 1) & 3)) << 4);               // 4 chunks per row: rows pair up per 128 bytes
}

// kVarQ: the variable-q-length causal call on an FP8 pool — columns are (query token, head) pairs, 48-byte items,
// causal mask per column, -inf guards (see attn_splitkv_kernel, kVarQ).
template <int D, int R, bool kAppend, bool kVarQ = false>
__global__ void __launch_bounds__(kAttnThreads, 3) attn_fp8_ring_kernel(const AttnParams p) {
  extern __shared__ __align__(128) unsigned char ring_smem[];
  const uint32_t ring = static_cast<uint32_t>(__cvta_generic_to_shared(ring_smem)) +
                        (threadIdx.x >> 5) * static_cast<uint32_t>(R * fp8_tile_bytes<D>());
  constexpr int KS = D / 16;   // MMA k-steps of S^T = K q^T
  constexpr int MT = D / 16;   // MMA m-tiles of O^T = V^T P^T
  constexpr int NE = D / 8;    // d columns owned per lane: g * NE + e
  constexpr int64_t kTile = fp8_tile_bytes<D>();
  constexpr unsigned kFull = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int g = lane >> 2, c = lane & 3;
  const int G = p.group;
  const int64_t blk_stride = static_cast<int64_t>(p.num_kv_heads) * kTile;
  const uint8_t* kv8 = reinterpret_cast<const uint8_t*>(p.kv_layer);

  const int n_warps = gridDim.x * kAttnWarps;
  for (int item = blockIdx.x * kAttnWarps + (threadIdx.x >> 5);;) {
    if (item >= p.n_units) break;
    const int h = item % p.num_kv_heads;
    const int4* wi = reinterpret_cast<const int4*>(p.items) + (item / p.num_kv_heads) * (kVarQ ? 3 : 2);
    const int4 w0 = __ldg(wi);
    const int4 w1 = __ldg(wi + 1);
    const int batch_idx = w0.x, slot = w0.y, blk_begin = w0.z, n_blocks = w0.w;
    const int n_tokens = w1.x;
    const int n_chunks = w1.z >> 16, chunk_idx = w1.z & 0xffff;
    const int pbase = w1.y < 0 ? -1 : w1.y + h * n_chunks;     // first partial slot of (request, kv head)
    const int pidx = w1.y < 0 ? -1 : pbase + chunk_idx;
    // Fused append (a3 inside a4): the unit that owns the request's last block takes that tile FIRST; the new
    // token's K / V rows are quantised here exactly as ingest_fp8_kernel does (same fp32 roundings, same codes),
    // written into the pool, and patched into the ring slot once the tile's stale bytes have landed.
    const bool special = kAppend && chunk_idx == n_chunks - 1;
    const int sp = special ? 1 : 0;
    const int last_blk = w1.w;
    uint2 new_codes = make_uint2(0u, 0u);
    float new_scale = 0.f;
    // kVarQ: tokens in the tile, and the last visible token of columns 2c, 2c+1 relative to the chunk start
    int n_qtok = 1, rel0 = 0, rel1 = 0;
    if constexpr (kVarQ) {
      const int4 w2 = __ldg(wi + 2);
      n_qtok = w2.y;
      const int t0 = (2 * c) / G, t1 = (2 * c + 1) / G;
      rel0 = t0 < n_qtok ? w2.x + t0 - blk_begin * kBlockSize : 0x3fffffff;   // unused columns: q = 0, never stored
      rel1 = t1 < n_qtok ? w2.x + t1 - blk_begin * kBlockSize : 0x3fffffff;
    }

    // q^T as f16 B fragments: lane (g, c) holds head g, d columns (c + 4j) * 16 + [0, 16), scaled by a
    // power of two so that the row maximum lies in [1, 2); cs0 / cs1 give the factor back to the scores
    uint32_t qf[KS][2];
    float cs0, cs1;
    {
      bool ok = g < G;
      const uint16_t* qp = p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + (ok ? g : 0)) * D + c * 16;
      if constexpr (kVarQ) {                                     // column g = (query token g / G, head g % G)
        const int qt = g / G;
        ok = qt < n_qtok;
        qp = p.q + (static_cast<int64_t>(batch_idx + (ok ? qt : 0)) * p.num_q_heads + h * G + (ok ? g - qt * G : 0)) * D + c * 16;
      }
      uint4 raw[D / 64][2];
      uint32_t mx = 0;
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          raw[j][k] = ldg_stream_pred(qp + j * 64 + k * 8, ok);
          mx = __vmaxu2(mx, __vmaxu2(__vmaxu2(raw[j][k].x & 0x7fff7fffu, raw[j][k].y & 0x7fff7fffu),
                                     __vmaxu2(raw[j][k].z & 0x7fff7fffu, raw[j][k].w & 0x7fff7fffu)));
        }
      mx = max(mx & 0xffffu, mx >> 16);
      mx = max(mx, __shfl_xor_sync(kFull, mx, 1));
      mx = max(mx, __shfl_xor_sync(kFull, mx, 2));
      const uint32_t eb = min(max(mx >> 7, 1u), 253u);           // biased exponent of the row maximum
      const float sf = __uint_as_float((254u - eb) << 23);        // 2^(127 - eb)
      const float back = __uint_as_float(eb << 23) * p.scale_log2;
      cs0 = __shfl_sync(kFull, back, (2 * c) * 4);
      cs1 = __shfl_sync(kFull, back, (2 * c + 1) * 4);
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
          for (int w = 0; w < 4; w += 2) {                       // words (w, w+1) = 4 bf16 = one k-step's (b0, b1)
            const uint32_t e0 = u4_get(raw[j][k], w), e1 = u4_get(raw[j][k], w + 1);
            qf[4 * j + 2 * k + w / 2][0] = pack_f16x2(__uint_as_float(e0 << 16) * sf, __uint_as_float(e0 & 0xffff0000u) * sf);
            qf[4 * j + 2 * k + w / 2][1] = pack_f16x2(__uint_as_float(e1 << 16) * sf, __uint_as_float(e1 & 0xffff0000u) * sf);
          }
    }

    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // heads 2c, 2c+1 (l: this lane's rows only)
    float o[MT][4];
#pragma unroll
    for (int i = 0; i < MT; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;

    const int32_t* bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
    const uint8_t* kvh = kv8 + static_cast<int64_t>(h) * kTile;
    int32_t ids = lane < n_blocks ? __ldg(bt + lane) : 0;       // physical ids of blocks [32k, 32k+32)
    int32_t ids_next = 0;

    // start the copies of tile t into ring slot t % R (one cp.async group per tile, empty past the unit's end)
    // virtual tile v -> real tile: special ? (v == 0 ? n_blocks - 1 : v - 1) : v
    auto issue = [&](int v) {
      if (v < n_blocks) {
        const bool first_special = special && v == 0;
        const int t = first_special ? n_blocks - 1 : v - sp;
        const uint8_t* tile;
        if (first_special) {
          tile = kvh + last_blk * blk_stride;
        } else {
          if ((t & 31) == 0 && t > 0) ids = ids_next;
          if ((t & 31) == 8 && t + 24 + lane < n_blocks) ids_next = __ldg(bt + t + 24 + lane);
          tile = kvh + __shfl_sync(kFull, ids, t & 31) * blk_stride;
        }
        const uint32_t sl = ring + (v % R) * static_cast<uint32_t>(kTile);
        const int nv = n_tokens - t * kBlockSize;
        constexpr int kChunksPerRow = D / 16;
#pragma unroll
        for (int i = 0; i < 2 * kBlockSize * kChunksPerRow / 32; ++i) {          // the K8 | V8 code rows
          const int idx = lane + 32 * i, row32 = idx / kChunksPerRow, ch = idx % kChunksPerRow;
          const int row = row32 & (kBlockSize - 1);
          const uint32_t dst = sl + (row32 >> 4) * (kBlockSize * D) + ring_chunk_off<D>(row, ch);
          const int sz = row < nv ? 16 : 0;                                      // zero-fill rows past the end
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(tile + idx * 16), "r"(sz) : "memory");
        }
        if (lane < 8) {                                                           // sc[16] {ks, vs}: 8 chunks of 2 rows
          const int sz = 2 * lane < nv ? (2 * lane + 1 < nv ? 16 : 8) : 0;
          asm volatile("cp.async.ca.shared.global [%0], [%1], 16, %2;" ::"r"(sl + 2 * kBlockSize * D + lane * 16),
                       "l"(tile + 2 * kBlockSize * D + lane * 16), "r"(sz) : "memory");
        }
        if constexpr (kAppend) {
          if (first_special) {                                    // quantise the new row: lanes [0, D/8) K pieces, [D/8, D/4) V pieces
            constexpr int kP = D / 8;
            const int cc = lane / kP, cp = lane % kP, r_new = nv - 1;
            const bool on = lane < 2 * kP;
            const uint16_t* srow = (cc ? p.v_new : p.k_new) + (static_cast<int64_t>(batch_idx) * p.num_kv_heads + h) * D;
            const uint4 x = ldg_stream_pred(srow + cp * 8, on);
            uint32_t mx = __vmaxu2(__vmaxu2(x.x & 0x7fff7fffu, x.y & 0x7fff7fffu), __vmaxu2(x.z & 0x7fff7fffu, x.w & 0x7fff7fffu));
            mx = max(mx & 0xffffu, mx >> 16);
#pragma unroll
            for (int off = kP / 2; off > 0; off >>= 1) mx = max(mx, __shfl_xor_sync(kFull, mx, off));
            const float amax = __uint_as_float(mx << 16);
            new_scale = mx == 0 ? 1.f : __fdiv_rn(amax, 448.f);
            const float inv = mx == 0 ? 1.f : __fdiv_rn(448.f, amax);
            uint32_t w[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const uint32_t e = u4_get(x, k);
              w[k] = f32x2_to_e4m3x2(__fmul_rn(__uint_as_float(e << 16), inv), __fmul_rn(__uint_as_float(e & 0xffff0000u), inv));
            }
            new_codes = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
            if (on) {
              uint8_t* wt = const_cast<uint8_t*>(tile);
              *reinterpret_cast<uint2*>(wt + cc * (kBlockSize * D) + r_new * D + cp * 8) = new_codes;
              if (cp == 0) *reinterpret_cast<float*>(wt + 2 * kBlockSize * D + r_new * 8 + cc * 4) = new_scale;
            }
            if (h == 0 && lane == 0) p.block_table[static_cast<int64_t>(slot) * p.bt_stride + blk_begin + n_blocks - 1] = last_blk;
          }
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    };

    auto consume = [&](int v) {
      const int t = (special && v == 0) ? n_blocks - 1 : v - sp;
      KV8Tile<D> T;                                              // fragments of ring slot v % R
      {
        const uint32_t slot = ring + (v % R) * static_cast<uint32_t>(kTile);
        if constexpr (kAppend) {
          if (special && v == 0) {                               // the tile's stale row r_new has landed: patch in the new row
            constexpr int kP = D / 8;
            const int cc = lane / kP, cp = lane % kP, r_new = n_tokens - t * kBlockSize - 1;
            if (lane < 2 * kP) {
              asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(slot + cc * (kBlockSize * D) + ring_chunk_off<D>(r_new, cp >> 1) + (cp & 1) * 8),
                           "r"(new_codes.x), "r"(new_codes.y) : "memory");
              if (cp == 0) asm volatile("st.shared.f32 [%0], %1;" ::"r"(slot + 2 * kBlockSize * D + r_new * 8 + cc * 4), "f"(new_scale) : "memory");
            }
            __syncwarp();
          }
        }
#pragma unroll
        for (int rs = 0; rs < 2; ++rs) {
          const int row = g + 8 * rs;
#pragma unroll
          for (int j = 0; j < D / 64; ++j) T.k[rs][j] = lds128(slot + ring_chunk_off<D>(row, c + 4 * j));
          asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(T.sc[rs].x), "=f"(T.sc[rs].y) : "r"(slot + 2 * kBlockSize * D + row * 8));
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int row = 2 * c + (i & 1) + 8 * (i >> 1);
          if constexpr (D == 128) {
            const uint4 x = lds128(slot + kBlockSize * D + ring_chunk_off<D>(row, g));
            T.v[i][0] = x.x; T.v[i][1] = x.y; T.v[i][2] = x.z; T.v[i][3] = x.w;
          } else {
            asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(T.v[i][0]), "=r"(T.v[i][1])
                         : "r"(slot + kBlockSize * D + ring_chunk_off<D>(row, g >> 1) + (g & 1) * 8));
          }
        }
      }
      // ---- S^T = K8 q~^T : word w of vector j feeds k-step 4j + w; two accumulation chains ----
      float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          const uint32_t r0 = u4_get(T.k[0][j], w), r1 = u4_get(T.k[1][j], w);
          mma_f16_m16n8k16((w & 1) ? sb : sa, e4m3x2_lo_to_f16x2(r0), e4m3x2_lo_to_f16x2(r1), e4m3x2_hi_to_f16x2(r0),
                           e4m3x2_hi_to_f16x2(r1), qf[4 * j + w][0], qf[4 * j + w][1]);
        }
      // s[0], s[1]: token g, heads 2c, 2c+1;  s[2], s[3]: token g+8   (log2 units)
      float s[4];
      s[0] = (sa[0] + sb[0]) * (T.sc[0].x * cs0);
      s[1] = (sa[1] + sb[1]) * (T.sc[0].x * cs1);
      s[2] = (sa[2] + sb[2]) * (T.sc[1].x * cs0);
      s[3] = (sa[3] + sb[3]) * (T.sc[1].x * cs1);
      const int nv = n_tokens - t * kBlockSize;
      const bool ok0 = g < nv, ok1 = g + 8 < nv;                 // ragged last block: mask by index, not value
      // ---- online softmax with the V scale folded into the reference: t = s + log2(vs) ----
      const float lv0 = ok0 ? fast_log2(T.sc[0].y) : -INFINITY, lv1 = ok1 ? fast_log2(T.sc[1].y) : -INFINITY;
      const float iv0 = ok0 ? __frcp_rn(T.sc[0].y) : 0.f, iv1 = ok1 ? __frcp_rn(T.sc[1].y) : 0.f;
      float t0 = s[0] + lv0, t1 = s[1] + lv0, t2 = s[2] + lv1, t3 = s[3] + lv1;
      if constexpr (kVarQ) {                                    // causal: a column sees tokens <= its own position
        const int tok = t * kBlockSize + g;
        if (tok > rel0) t0 = -INFINITY;
        if (tok > rel1) t1 = -INFINITY;
        if (tok + 8 > rel0) t2 = -INFINITY;
        if (tok + 8 > rel1) t3 = -INFINITY;
      }
      float mx0 = fmaxf(t0, t2), mx1 = fmaxf(t1, t3);
#pragma unroll
      for (int off = 4; off < 32; off <<= 1) {
        mx0 = fmaxf(mx0, __shfl_xor_sync(kFull, mx0, off));
        mx1 = fmaxf(mx1, __shfl_xor_sync(kFull, mx1, off));
      }
      const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);   // finite: every tile has >= 1 valid token ...
      const bool moved = mn0 != m0 || mn1 != m1;
      float ms0 = mn0, ms1 = mn1;
      if constexpr (kVarQ) {                                    // ... except for a column that sees nothing yet
        ms0 = mn0 == -INFINITY ? 0.f : mn0;
        ms1 = mn1 == -INFINITY ? 0.f : mn1;
      }
      const float a0 = fast_exp2(m0 - ms0), a1 = fast_exp2(m1 - ms1);
      m0 = mn0; m1 = mn1;
      const float p0 = fast_exp2(t0 - ms0), p1 = fast_exp2(t1 - ms1);   // p'_t = p_t * vs_t  in (0, 1]
      const float p2 = fast_exp2(t2 - ms0), p3 = fast_exp2(t3 - ms1);
      l0 = l0 * a0 + (p0 * iv0 + p2 * iv1);
      l1 = l1 * a1 + (p1 * iv0 + p3 * iv1);
      if (__any_sync(kFull, moved)) {                            // the running maximum settles after a few tiles
#pragma unroll
        for (int i = 0; i < MT; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
      }
      // ---- P'^T as the f16 B fragment (11-bit weights in (0, 1]: 2^-12 relative, below the final bf16 rounding) ----
      const uint32_t b0 = movmatrix_trans(pack_f16x2(p0, p1));  // tokens 2c, 2c+1   of head g
      const uint32_t b1 = movmatrix_trans(pack_f16x2(p2, p3));  // tokens 2c+8, 2c+9 of head g
      // ---- O^T += V8^T P'^T : m-tile i takes the lane's column e = i (row g) and e = i + NE/2 (row g+8);
      // one PRMT pairs the codes of two tokens for two neighbouring columns, one F2FP per pair ----
#pragma unroll
      for (int i = 0; i < MT; i += 2) {                          // columns (i, i+1) and (i + NE/2, i + 1 + NE/2)
        const int e1 = i, e2 = i + NE / 2;
        const uint32_t sel = (e1 & 2) ? 0x7362u : 0x5140u;      // bytes (b, b+1) of both rows: [A.b, B.b, A.b+1, B.b+1]
        const uint32_t x01 = __byte_perm(T.v[0][e1 >> 2], T.v[1][e1 >> 2], sel);   // tokens 2c, 2c+1; columns e1, e1+1
        const uint32_t x23 = __byte_perm(T.v[2][e1 >> 2], T.v[3][e1 >> 2], sel);   // tokens 2c+8, 2c+9
        const uint32_t y01 = __byte_perm(T.v[0][e2 >> 2], T.v[1][e2 >> 2], sel);   // columns e2, e2+1
        const uint32_t y23 = __byte_perm(T.v[2][e2 >> 2], T.v[3][e2 >> 2], sel);
        mma_f16_m16n8k16(o[i], e4m3x2_lo_to_f16x2(x01), e4m3x2_lo_to_f16x2(y01), e4m3x2_lo_to_f16x2(x23),
                         e4m3x2_lo_to_f16x2(y23), b0, b1);
        mma_f16_m16n8k16(o[i + 1], e4m3x2_hi_to_f16x2(x01), e4m3x2_hi_to_f16x2(y01), e4m3x2_hi_to_f16x2(x23),
                         e4m3x2_hi_to_f16x2(y23), b0, b1);
      }
    };

#pragma unroll
    for (int t = 0; t < R - 1; ++t) issue(t);                    // R - 1 tiles ahead
    for (int t = 0; t < n_blocks; ++t) {
      asm volatile("cp.async.wait_group %0;" ::"n"(R - 2) : "memory");   // tile t has landed (this lane's copies)
      __syncwarp();                                              // ... everyone's; and slot (t - 1) % R is free
      issue(t + R - 1);
      consume(t);
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();

    // ---- epilogue: finish l over the token lanes, then store ----
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {
      l0 += __shfl_xor_sync(kFull, l0, off);
      l1 += __shfl_xor_sync(kFull, l1, off);
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
      // element e of this lane: d column g * NE + e, register o[e % (NE/2)][2*(e/(NE/2)) + hh]
      if (pidx < 0) {
        const float inv = 1.f / l;
        uint16_t* op = p.out + out_row * D + g * NE;
#pragma unroll
        for (int e = 0; e < NE; e += 8) {
          uint32_t w[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int ea = e + 2 * k, eb2 = ea + 1;
            w[k] = pack_bf16x2(o[ea % (NE / 2)][2 * (ea / (NE / 2)) + hh] * inv, o[eb2 % (NE / 2)][2 * (eb2 / (NE / 2)) + hh] * inv);
          }
          *reinterpret_cast<uint4*>(op + e) = make_uint4(w[0], w[1], w[2], w[3]);
        }
      } else {
        float* po = p.part_o + (static_cast<int64_t>(pidx) * PG + head) * D + g * NE;
#pragma unroll
        for (int e = 0; e < NE; e += 4) {
          float f[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) f[k] = o[(e + k) % (NE / 2)][2 * ((e + k) / (NE / 2)) + hh];
          *reinterpret_cast<float4*>(po + e) = make_float4(f[0], f[1], f[2], f[3]);
        }
        if (g == 0) *reinterpret_cast<float2*>(p.part_ml + (static_cast<int64_t>(pidx) * PG + head) * 2) = make_float2(m, l);
      }
    }
    // ---- fused a5: the unit that completes its (request, kv head) merges the partials ----
    if (pidx >= 0 && (kVarQ || p.fuse_combine)) {
      __threadfence();
      __syncwarp();
      int last = 0;
      if (lane == 0) {
        last = atomicAdd(&p.arrive[pbase], 1) == n_chunks - 1;
        if (last) p.arrive[pbase] = 0;                           // ready for the next launch
      }
      last = __shfl_sync(kFull, last, 0);
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
    item = __shfl_sync(kFull, item, 0);
  }

  // Last CTA out rewinds the work counter for the next launch
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned prev = atomicInc(reinterpret_cast<unsigned*>(&p.counters[1]), gridDim.x - 1);
    if (prev == gridDim.x - 1) p.counters[0] = 0;
  }
}

}  // namespace kvp
