// kv_attn.cuh — a4 (+ a3, a5): split-KV paged decode attention, ONE kernel body for both pool formats.
//
//   attn_kernel<Bf16Tiles<D>, kAppend, kVarQ, R, kCtas>   bf16 pool
//   attn_kernel<Fp8Tiles<D>,  kAppend, kVarQ, R, kCtas>   FP8 (e4m3) pool, NEXT-2
//
// One warp per work unit = (request chunk, kv head); 4 independent warps per CTA, dynamic work claiming from a
// global counter, largest units first.  Fragment mapping (both formats): the 16 tokens of a block sit on the MMA M
// axis and the (<= 8) query heads of the GQA group on N:
//     S^T[16 tok x 8 heads] = K[16 x D] . q^T[D x 8]            D/16 MMAs (m16n8k16), A = K rows
//     O^T[D x 8 heads]     += V^T[D x 16 tok] . P^T[16 x 8]     D/16 MMAs, B = P^T via movmatrix
// A dot product does not care in which order the contraction index is visited, so a lane feeds the k-slots of its
// A fragment from ANY d columns as long as the q fragment uses the same ones; likewise the d columns of O^T are
// permuted freely and un-permuted at the store.  A fragment register is therefore always a plain 16-byte piece of
// a K or V row: no ldmatrix, no transposes beyond a few PRMT per V m-tile.
// Staging: a per-warp shared-memory ring of R tile slots filled by 16-byte cp.async (SASS LDGSTS), zero-filled
// past the request's end, one commit group per tile, cp.async.wait_group + __syncwarp before a tile is consumed —
// no block-wide barrier: a ring is private to its warp.  The 16-byte chunks of every row are XOR-swizzled so that
// both fragment read patterns are bank-conflict free.
// What the two formats do differently is confined to the tile providers below: the bytes of a tile and their
// copy, the query fragments, fragments -> scores, weights -> O (PV), and the append of the new token's row.
// Everything else — work-item decode, the block-id stream, the tile pipeline, masks, the online softmax, the
// epilogue, the fused log-sum-exp merge (a5), work claiming, programmatic dependent launch — is written once.
#pragma once

#include "kv_common.cuh"

namespace kvp {

// =============================================================================================
// bf16 tiles: K[16][D] | V[16][D] bf16, 4 D bytes per token... 64 D bytes per tile (8 KiB at D = 128)
// =============================================================================================
// kTmaL = true (D = 128 only): the ring slot has the layout the TMA unit writes for a [64 rows][128 B] box with
// CU_TENSOR_MAP_SWIZZLE_128B — 128-byte row rho of the tile (token t's K row = rows 2t, 2t+1; V rows follow at 32 + ...)
// at rho * 128 with its 16-byte chunks XORed with rho & 7 — so that full tiles can be fetched by ONE
// cp.async.bulk.tensor instruction (SASS UTMALDG) issued by one lane, completion on an mbarrier.  That swizzle is not
// the one this kernel would choose (the fragment reads of MMA rows g, g+1 would collide), so the TOKENS are permuted
// over the MMA rows instead: row r of S^T holds token tok(r) — an online softmax does not care — which makes both
// fragment read patterns conflict-free again.  Ragged and fused-append tiles still go through LDGSTS (same layout).
template <int D_, bool kTmaL = false>
struct Bf16Tiles {
  static constexpr int D = D_;
  static_assert(!kTmaL || D_ == 128, "the TMA layout is built for 256-byte rows");
  static constexpr bool kTma = kTmaL;
  static constexpr int KJ = D / 32;                             // K vectors per row per lane
  static constexpr int KS = D / 16, MT = D / 16, NE = D / 8;
  static constexpr uint32_t kSlotBytes = 2 * kBlockSize * D * 2;
  static constexpr int64_t kPoolTileBytes = kSlotBytes;
  static constexpr uint32_t kSlotStride = kSlotBytes;           // ring slot pitch (a multiple of 1 KiB at D = 128)
  template <int R> static __host__ __device__ constexpr uint32_t warp_ring_bytes() { return R * kSlotStride; }
  template <int R> static __device__ __forceinline__ uint32_t scales_addr(uint32_t, int) { return 0; }
  // TMA: one tensor copy per tile
  static __device__ __forceinline__ void tma_tile(uint32_t slot_addr, uint32_t, const void* tmap, uint32_t bar, int64_t row,
                                                  const unsigned char*) {
    mbar_arrive_expect_tx(bar, kSlotBytes);
    tma_load_2d(slot_addr, tmap, bar, 0, static_cast<int32_t>(row));
  }

  // token held by MMA row r (r in [0, 8); rows r + 8 hold token tok(r) + 8)
  static __device__ __forceinline__ int tok(int r) { return kTmaL ? static_cast<int>((0x57463120u >> (4 * r)) & 7u) : r; }
  static constexpr bool kVScaled = false;                       // no per-token V scale in the softmax reference
  static constexpr bool kLazyRescale = false;
  static constexpr bool kPatchNewRow = false;                   // the fused append sources the new row in copy_tile

  struct Query { uint32_t f[KS][2]; };
  struct NewRow {};
  struct Frag {
    uint4 k[2][KJ];        // rows g, g+8; column chunks c + 4j
    uint4 v[4][D / 64];    // rows 2c, 2c+1, 2c+8, 2c+9; column chunks g + 8cs
  };

  // byte offset of 16-byte chunk `chunk` of row `row` inside a K or V half of a slot:
  // chunk' = chunk ^ (row bit 1) << 1 ^ (row bit 2 ^ row bit 0) << 2
  static __device__ __forceinline__ uint32_t chunk_off(int row, int chunk) {
    if constexpr (kTmaL) {
      const int rho = 2 * row + (chunk >> 3);
      return rho * 128 + (((chunk & 7) ^ (rho & 7)) << 4);
    } else {
      return row * (D * 2) + ((chunk ^ (((row >> 1) & 1) << 1) ^ ((((row >> 2) ^ row) & 1) << 2)) << 4);
    }
  }

  // q^T as B fragments: lane (g, c) holds MMA column g, d columns of chunk c + 4j (zero if !ok)
  static __device__ __forceinline__ void load_query(Query& Q, const uint16_t* qrow, bool ok, int c, float scale_log2,
                                                    float& cs0, float& cs1) {
#pragma unroll
    for (int j = 0; j < KJ; ++j) {
      const uint4 v = ldg_stream_pred(qrow + c * 8 + j * 32, ok);
      Q.f[2 * j][0] = v.x; Q.f[2 * j][1] = v.y; Q.f[2 * j + 1][0] = v.z; Q.f[2 * j + 1][1] = v.w;
    }
    cs0 = cs1 = scale_log2;
  }

  // start the copies of one tile into a ring slot; row r_new (>= 0 only for the fused append's tile) comes from
  // the new token's rows instead of the pool
  template <bool kAppend>
  static __device__ __forceinline__ void copy_tile(uint32_t slot_addr, uint32_t, const unsigned char* tile, int nv, int lane, int r_new,
                                                   const uint16_t* knew_row, const uint16_t* vnew_row) {
    constexpr int kCh = D / 8;                                  // 16-byte chunks per row
#pragma unroll
    for (int i = 0; i < 2 * kBlockSize * kCh / 32; ++i) {
      const int idx = lane + 32 * i, row32 = idx / kCh, ch = idx % kCh, row = row32 & (kBlockSize - 1);
      const void* srcp = tile + idx * 16;
      if (kAppend && row == r_new) srcp = ((row32 >> 4) ? vnew_row : knew_row) + ch * 8;
      cp_async16(slot_addr + (row32 >> 4) * (kBlockSize * D * 2) + chunk_off(row, ch), srcp, row < nv ? 16 : 0);
    }
  }

  // a3 inside a4: the new token's K and V rows go into the pool tile (global -> global)
  static __device__ __forceinline__ void append_row(unsigned char* tile, int r_new, const uint16_t* knew_row,
                                                    const uint16_t* vnew_row, int lane, NewRow&) {
    constexpr int kCh = D / 8;
    if (lane < 2 * kCh) {
      const int cc = lane / kCh, ch = lane % kCh;
      const uint4 x = ldg_stream((cc ? vnew_row : knew_row) + ch * 8);
      *reinterpret_cast<uint4*>(tile + cc * (kBlockSize * D * 2) + r_new * (D * 2) + ch * 16) = x;
    }
  }
  static __device__ __forceinline__ void patch_slot(uint32_t, uint32_t, int, int, const NewRow&) {}

  static __device__ __forceinline__ void load_frags(Frag& T, uint32_t slot_addr, uint32_t, int g, int c) {
#pragma unroll
    for (int rs = 0; rs < 2; ++rs)
#pragma unroll
      for (int j = 0; j < KJ; ++j) T.k[rs][j] = lds128(slot_addr + chunk_off(tok(g) + 8 * rs, c + 4 * j));
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int cs = 0; cs < D / 64; ++cs)
        T.v[i][cs] = lds128(slot_addr + kBlockSize * D * 2 + chunk_off(tok(2 * c + (i & 1)) + 8 * (i >> 1), g + 8 * cs));
  }

  // s[0], s[1]: token g, MMA columns 2c, 2c+1;  s[2], s[3]: token g+8   (log2 units)
  static __device__ __forceinline__ void scores(const Frag& T, const Query& Q, float cs0, float cs1, float (&s)[4],
                                                float (&vs)[2]) {
    float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};   // two independent accumulation chains
#pragma unroll
    for (int j = 0; j < KJ; ++j) {
      mma_bf16_m16n8k16(sa, T.k[0][j].x, T.k[1][j].x, T.k[0][j].y, T.k[1][j].y, Q.f[2 * j][0], Q.f[2 * j][1]);
      mma_bf16_m16n8k16(sb, T.k[0][j].z, T.k[1][j].z, T.k[0][j].w, T.k[1][j].w, Q.f[2 * j + 1][0], Q.f[2 * j + 1][1]);
    }
    s[0] = (sa[0] + sb[0]) * cs0; s[1] = (sa[1] + sb[1]) * cs1;
    s[2] = (sa[2] + sb[2]) * cs0; s[3] = (sa[3] + sb[3]) * cs1;
    vs[0] = vs[1] = 1.f;
  }

  // O^T += V^T P^T.  P is fed to the tensor core as bf16 hi + bf16 lo (p = hi + lo up to 2^-17 p), so the weights
  // keep ~16 mantissa bits and the only bf16-sized error left in the result is the final rounding of `out`.
  // m-tile i takes the lane's d column e = i (row g) and e = i + NE/2 (row g+8).
  static __device__ __forceinline__ void pv(const Frag& T, float p0, float p1, float p2, float p3, float (&o)[MT][4]) {
    const uint32_t ph01 = pack_bf16x2(p0, p1), ph23 = pack_bf16x2(p2, p3);
    const uint32_t pl01 = pack_bf16x2(p0 - __uint_as_float(ph01 << 16), p1 - __uint_as_float(ph01 & 0xffff0000u));
    const uint32_t pl23 = pack_bf16x2(p2 - __uint_as_float(ph23 << 16), p3 - __uint_as_float(ph23 & 0xffff0000u));
    const uint32_t b0 = movmatrix_trans(ph01);                   // tokens 2c, 2c+1   of column g
    const uint32_t b1 = movmatrix_trans(ph23);                   // tokens 2c+8, 2c+9 of column g
    const uint32_t c0 = movmatrix_trans(pl01);
    const uint32_t c1 = movmatrix_trans(pl23);
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
  }

  // first d column of the lane's 8-element group cs (element e = 8 cs + k lives in o[e % (NE/2)][2 (e / (NE/2)) + hh])
  static __device__ __forceinline__ int col0(int g, int cs) { return (g + 8 * cs) * 8; }
};

// =============================================================================================
// FP8 tiles (NEXT-2): K8[16][D] | V8[16][D] e4m3 codes | sc[16]{ks_t, vs_t} fp32 — 32 D + 128 bytes (4224 at D = 128).
// The MMAs run in f16: e4m3 -> f16 is exact and one instruction per code pair (F2FP.F16.E4M3.UNPACK_B).
//   * q rows are pre-scaled by a power of two so their largest element lies in [1, 2) and converted to f16 (exact
//     for every element within 2^-14 of the row maximum); the factor returns through the per-column score scale.
//   * the score of token t is (K8_t . q~) * ks_t * scale; the V scale is folded into the softmax REFERENCE rather
//     than into the weights: the running maximum m' is taken over s_t + log2(vs_t), so the weights fed to the PV
//     MMA, p'_t = 2^(s_t + log2 vs_t - m') = p_t * vs_t, lie in (0, 1] whatever the magnitude of V — no f16
//     overflow or underflow to manage — while l accumulates p'_t / vs_t.  O and l share the reference m', so O / l
//     and the LSE merge are unchanged.
// =============================================================================================
// kTmaL = true (D = 128): the codes of a tile (32 rows of 128 B) arrive by one cp.async.bulk.tensor into a 1 KiB-aligned
// 4 KiB slot in the hardware's 128-byte swizzle, the 128 bytes of scales by a second (1-D) bulk copy into a small ring
// behind the code slots, both completing on the slot's mbarrier; tokens are permuted over the MMA rows (tok) so that the
// fragment reads stay conflict-free under that swizzle.  This is where TMA pays: the FP8 loop spends 9 LDGSTS + ~45
// integer instructions per 4 KiB tile on copies, on a warp that is issue-limited.
template <int D_, bool kTmaL = false>
struct Fp8Tiles {
  static constexpr int D = D_;
  static_assert(!kTmaL || D_ == 128, "the TMA layout is built for 128-byte code rows");
  static constexpr int KS = D / 16, MT = D / 16, NE = D / 8;
  static constexpr uint32_t kSlotBytes = 32 * D + 128;          // bytes of a tile (what a copy moves)
  static constexpr int64_t kPoolTileBytes = kSlotBytes;
  static constexpr bool kTma = kTmaL;
  static constexpr uint32_t kSlotStride = kTmaL ? 32 * D : kSlotBytes;
  // per-warp ring: R slots (+ R x 128 B of scales behind them in the TMA layout), padded to a multiple of 1 KiB
  template <int R> static __host__ __device__ constexpr uint32_t warp_ring_bytes() {
    return kTmaL ? (R * kSlotStride + R * 128 + 1023u) / 1024u * 1024u : R * kSlotStride;
  }
  template <int R> static __device__ __forceinline__ uint32_t scales_addr(uint32_t ring, int s) {
    return kTmaL ? ring + R * kSlotStride + s * 128 : ring + s * kSlotStride + 2 * kBlockSize * D;
  }
  static __device__ __forceinline__ int tok(int r) { return kTmaL ? static_cast<int>((0x37156240u >> (4 * r)) & 7u) : r; }
  static __device__ __forceinline__ void tma_tile(uint32_t slot_addr, uint32_t sc_addr, const void* tmap, uint32_t bar, int64_t row,
                                                  const unsigned char* tile) {
    mbar_arrive_expect_tx(bar, kSlotBytes);
    tma_load_2d(slot_addr, tmap, bar, 0, static_cast<int32_t>(row));
    bulk_load_1d(sc_addr, tile + 2 * kBlockSize * D, 128, bar);
  }
  static constexpr bool kVScaled = true;
  static constexpr bool kLazyRescale = true;                    // rescale O only when some running maximum moved
  static constexpr bool kPatchNewRow = true;                    // the quantised new row is patched into the slot after it landed

  struct Query { uint32_t f[KS][2]; };
  struct NewRow { uint2 codes; float scale; };
  struct Frag {
    uint4 k[2][D / 64];      // rows g, g+8; 16 codes at column chunk c + 4j: word w of vector j = k-step 4j + w
    uint32_t v[4][D / 32];   // rows 2c, 2c+1, 2c+8, 2c+9; the lane's D/8 columns g*(D/8) ...
    float2 sc[2];            // (ks, vs) of tokens g, g+8
  };

  static __device__ __forceinline__ uint32_t chunk_off(int row, int chunk) {   // byte offset of a 16-byte chunk of a code row
    if constexpr (kTmaL) return row * 128 + ((chunk ^ (row & 7)) << 4);
    else if constexpr (D == 128) return row * 128 + ((chunk ^ (((row >> 1) & 1) << 1) ^ ((((row >> 2) ^ row) & 1) << 2)) << 4);
    else return row * 64 + ((chunk ^ ((row >> 1) & 3)) << 4);                 // 4 chunks per row: rows pair up per 128 bytes
  }

  // q^T as f16 B fragments: lane (g, c) holds MMA column g, d columns (c + 4j) * 16 + [0, 16)
  static __device__ __forceinline__ void load_query(Query& Q, const uint16_t* qrow, bool ok, int c, float scale_log2,
                                                    float& cs0, float& cs1) {
    uint4 raw[D / 64][2];
    uint32_t mx = 0;
#pragma unroll
    for (int j = 0; j < D / 64; ++j)
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        raw[j][k] = ldg_stream_pred(qrow + c * 16 + j * 64 + k * 8, ok);
        mx = max(mx, amax_bits8(raw[j][k]));
      }
    mx = max(mx, __shfl_xor_sync(kFull, mx, 1));
    mx = max(mx, __shfl_xor_sync(kFull, mx, 2));
    const uint32_t eb = min(max(mx >> 7, 1u), 253u);             // biased exponent of the row maximum
    const float sf = __uint_as_float((254u - eb) << 23);          // 2^(127 - eb)
    const float back = __uint_as_float(eb << 23) * scale_log2;
    cs0 = __shfl_sync(kFull, back, (2 * c) * 4);
    cs1 = __shfl_sync(kFull, back, (2 * c + 1) * 4);
#pragma unroll
    for (int j = 0; j < D / 64; ++j)
#pragma unroll
      for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int w = 0; w < 4; w += 2) {                         // words (w, w+1) = 4 bf16 = one k-step's (b0, b1)
          const uint32_t e0 = u4_get(raw[j][k], w), e1 = u4_get(raw[j][k], w + 1);
          Q.f[4 * j + 2 * k + w / 2][0] = pack_f16x2(__uint_as_float(e0 << 16) * sf, __uint_as_float(e0 & 0xffff0000u) * sf);
          Q.f[4 * j + 2 * k + w / 2][1] = pack_f16x2(__uint_as_float(e1 << 16) * sf, __uint_as_float(e1 & 0xffff0000u) * sf);
        }
  }

  template <bool kAppend>
  static __device__ __forceinline__ void copy_tile(uint32_t slot_addr, uint32_t sc_addr, const unsigned char* tile, int nv, int lane, int,
                                                   const uint16_t*, const uint16_t*) {
    constexpr int kChunksPerRow = D / 16;
#pragma unroll
    for (int i = 0; i < 2 * kBlockSize * kChunksPerRow / 32; ++i) {          // the K8 | V8 code rows
      const int idx = lane + 32 * i, row32 = idx / kChunksPerRow, ch = idx % kChunksPerRow;
      const int row = row32 & (kBlockSize - 1);
      cp_async16(slot_addr + (row32 >> 4) * (kBlockSize * D) + chunk_off(row, ch), tile + idx * 16, row < nv ? 16 : 0);
    }
    if (lane < 8) {                                                           // sc[16] {ks, vs}: 8 chunks of 2 rows
      const int sz = 2 * lane < nv ? (2 * lane + 1 < nv ? 16 : 8) : 0;
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16, %2;" ::"r"(sc_addr + lane * 16),
                   "l"(tile + 2 * kBlockSize * D + lane * 16), "r"(sz) : "memory");
    }
  }

  // a3 inside a4: quantise the new token's K and V rows exactly as ingest_fp8_kernel does (same fp32 roundings, same
  // codes) and write codes and scales into the pool tile: lanes [0, D/8) hold the K pieces, [D/8, D/4) the V pieces.
  // Two halves, so that a caller may issue the load early: append_load (the lane's 16-byte piece of the new rows) and
  // append_store (quantise + store).
  static __device__ __forceinline__ uint4 append_load(const uint16_t* knew_row, const uint16_t* vnew_row, int lane) {
    constexpr int kP = D / 8;
    return ldg_stream_pred((lane / kP ? vnew_row : knew_row) + (lane % kP) * 8, lane < 2 * kP);
  }
  static __device__ __forceinline__ void append_store(unsigned char* tile, int r_new, const uint4& x, int lane, NewRow& nr) {
    constexpr int kP = D / 8;
    const int cc = lane / kP, cp = lane % kP;
    uint32_t mx = amax_bits8(x);
#pragma unroll
    for (int off = kP / 2; off > 0; off >>= 1) mx = max(mx, __shfl_xor_sync(kFull, mx, off));
    nr.codes = quantise_piece(x, mx, &nr.scale);
    if (lane < 2 * kP) {
      *reinterpret_cast<uint2*>(tile + cc * (kBlockSize * D) + r_new * D + cp * 8) = nr.codes;
      if (cp == 0) *reinterpret_cast<float*>(tile + 2 * kBlockSize * D + r_new * 8 + cc * 4) = nr.scale;
    }
  }
  static __device__ __forceinline__ void append_row(unsigned char* tile, int r_new, const uint16_t* knew_row,
                                                    const uint16_t* vnew_row, int lane, NewRow& nr) {
    append_store(tile, r_new, append_load(knew_row, vnew_row, lane), lane, nr);
  }
  // ... and, once the tile's stale bytes have landed in the slot, the same row goes on top of them
  static __device__ __forceinline__ void patch_slot(uint32_t slot_addr, uint32_t sc_addr, int r_new, int lane, const NewRow& nr) {
    constexpr int kP = D / 8;
    const int cc = lane / kP, cp = lane % kP;
    if (lane < 2 * kP) {
      asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(slot_addr + cc * (kBlockSize * D) + chunk_off(r_new, cp >> 1) + (cp & 1) * 8),
                   "r"(nr.codes.x), "r"(nr.codes.y) : "memory");
      if (cp == 0) asm volatile("st.shared.f32 [%0], %1;" ::"r"(sc_addr + r_new * 8 + cc * 4), "f"(nr.scale) : "memory");
    }
  }

  static __device__ __forceinline__ void load_frags(Frag& T, uint32_t slot, uint32_t sc_addr, int g, int c) {
#pragma unroll
    for (int rs = 0; rs < 2; ++rs) {
      const int row = tok(g) + 8 * rs;
#pragma unroll
      for (int j = 0; j < D / 64; ++j) T.k[rs][j] = lds128(slot + chunk_off(row, c + 4 * j));
      asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(T.sc[rs].x), "=f"(T.sc[rs].y) : "r"(sc_addr + row * 8));
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int row = tok(2 * c + (i & 1)) + 8 * (i >> 1);
      if constexpr (D == 128) {
        const uint4 x = lds128(slot + kBlockSize * D + chunk_off(row, g));
        T.v[i][0] = x.x; T.v[i][1] = x.y; T.v[i][2] = x.z; T.v[i][3] = x.w;
      } else {
        asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(T.v[i][0]), "=r"(T.v[i][1])
                     : "r"(slot + kBlockSize * D + chunk_off(row, g >> 1) + (g & 1) * 8));
      }
    }
  }

  // S^T = K8 q~^T : word w of vector j feeds k-step 4j + w; two accumulation chains.  vs = V scales of tokens g, g+8.
  static __device__ __forceinline__ void scores(const Frag& T, const Query& Q, float cs0, float cs1, float (&s)[4],
                                                float (&vs)[2]) {
    float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < D / 64; ++j)
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          const uint32_t r0 = u4_get(T.k[0][j], w), r1 = u4_get(T.k[1][j], w);
          mma_f16_m16n8k16((w & 1) ? sb : sa, e4m3x2_lo_to_f16x2(r0), e4m3x2_lo_to_f16x2(r1), e4m3x2_hi_to_f16x2(r0),
                           e4m3x2_hi_to_f16x2(r1), Q.f[4 * j + w][0], Q.f[4 * j + w][1]);
        }
    s[0] = (sa[0] + sb[0]) * (T.sc[0].x * cs0);
    s[1] = (sa[1] + sb[1]) * (T.sc[0].x * cs1);
    s[2] = (sa[2] + sb[2]) * (T.sc[1].x * cs0);
    s[3] = (sa[3] + sb[3]) * (T.sc[1].x * cs1);
    vs[0] = T.sc[0].y; vs[1] = T.sc[1].y;
  }

  // O^T += V8^T P'^T with P' as one f16 (11-bit weights in (0, 1]: 2^-12 relative, below the final bf16 rounding).
  // m-tile i takes the lane's column e = i (row g) and e = i + NE/2 (row g+8); one PRMT pairs the codes of two
  // tokens for two neighbouring columns, one F2FP per pair.
  static __device__ __forceinline__ void pv(const Frag& T, float p0, float p1, float p2, float p3, float (&o)[MT][4]) {
    const uint32_t b0 = movmatrix_trans(pack_f16x2(p0, p1));     // tokens 2c, 2c+1   of column g
    const uint32_t b1 = movmatrix_trans(pack_f16x2(p2, p3));     // tokens 2c+8, 2c+9 of column g
#pragma unroll
    for (int i = 0; i < MT; i += 2) {                            // columns (i, i+1) and (i + NE/2, i + 1 + NE/2)
      const int e1 = i, e2 = i + NE / 2;
      const uint32_t sel = (e1 & 2) ? 0x7362u : 0x5140u;        // bytes (b, b+1) of both rows: [A.b, B.b, A.b+1, B.b+1]
      const uint32_t x01 = __byte_perm(T.v[0][e1 >> 2], T.v[1][e1 >> 2], sel);   // tokens 2c, 2c+1; columns e1, e1+1
      const uint32_t x23 = __byte_perm(T.v[2][e1 >> 2], T.v[3][e1 >> 2], sel);   // tokens 2c+8, 2c+9
      const uint32_t y01 = __byte_perm(T.v[0][e2 >> 2], T.v[1][e2 >> 2], sel);   // columns e2, e2+1
      const uint32_t y23 = __byte_perm(T.v[2][e2 >> 2], T.v[3][e2 >> 2], sel);
      mma_f16_m16n8k16(o[i], e4m3x2_lo_to_f16x2(x01), e4m3x2_lo_to_f16x2(y01), e4m3x2_lo_to_f16x2(x23),
                       e4m3x2_lo_to_f16x2(y23), b0, b1);
      mma_f16_m16n8k16(o[i + 1], e4m3x2_hi_to_f16x2(x01), e4m3x2_hi_to_f16x2(y01), e4m3x2_hi_to_f16x2(x23),
                       e4m3x2_hi_to_f16x2(y23), b0, b1);
    }
  }

  static __device__ __forceinline__ int col0(int g, int cs) { return g * NE + 8 * cs; }
};

// =============================================================================================
// the kernel
//
// kVarQ (in-place prefill of ultra-short requests merged with decoding): the 8
// MMA columns of a unit are (query token, head) pairs of ONE kv head — column j = query token j / G of the tile,
// head j % G of the group — instead of the G heads of one token.  A work item is then a QUERY TILE of 8 / G
// consecutive query tokens of one request (48-byte item: words 8..9 = pos0, the absolute position of the tile's
// first query token, and n_qtok), `batch_idx` is the tile's first row in q / out, and the mask is causal: column j
// sees tokens 0 .. pos0 + j / G.  A column may see nothing of a later chunk: its running max stays -inf, handled
// by the guards below (chunk 0 always holds token 0, visible to every column).
//
// Programmatic dependent launch: the kernel may be launched with the programmatic-stream-serialization attribute,
// in which case its CTAs start while the stream's previous kernel drains.  Nothing that kernel may have produced
// is touched before griddepcontrol.wait: q, k_new, v_new, out, the partials, the work and arrival counters and
// (unless p.chained) the work items and the block table are all accessed after it.
// =============================================================================================
template <class TP, bool kAppend, bool kVarQ, int R, int kCtas>
__global__ void __launch_bounds__(kAttnThreads, kCtas) attn_kernel(const __grid_constant__ AttnParams p) {
  extern __shared__ __align__(128) unsigned char ring_smem[];
  constexpr int D = TP::D, MT = TP::MT, NE = TP::NE;
  const int lane = threadIdx.x & 31;
  uint32_t smem0 = static_cast<uint32_t>(__cvta_generic_to_shared(ring_smem));
  if constexpr (TP::kTma) smem0 = (smem0 + 1023u) & ~1023u;     // the 128-byte swizzle is a function of the address
  const uint32_t ring = smem0 + (threadIdx.x >> 5) * TP::template warp_ring_bytes<R>();
  // TMA variants: one mbarrier per ring slot of this warp (behind the rings), and the parity each is next waited on
  const uint32_t bars = smem0 + kAttnWarps * TP::template warp_ring_bytes<R>() + (threadIdx.x >> 5) * (R * 8);
  uint32_t bar_parity = 0;
  if constexpr (TP::kTma) {
    if (lane == 0) {
#pragma unroll
      for (int s = 0; s < R; ++s) mbar_init(bars + s * 8, 1);
      mbar_init_fence();
    }
    __syncwarp();
  }
  const int g = lane >> 2, c = lane & 3;
  const int tg = TP::tok(g);                                     // the token (of a block's first 8) on MMA row g
  const int G = p.group;
  const int64_t blk_stride = static_cast<int64_t>(p.num_kv_heads) * TP::kPoolTileBytes;
  unsigned char* const kv = reinterpret_cast<unsigned char*>(p.kv_layer);

  if (!p.chained) pdl_wait();
  bool waited = !p.chained;
  pdl_launch_dependents();

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
    const int n_chunks = static_cast<int>(static_cast<uint32_t>(w1.z) >> 16), chunk_idx = w1.z & 0xffff, last_blk = w1.w;
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
    const int32_t* bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
    int32_t ids = lane < n_blocks ? __ldg(bt + lane) : 0;       // physical ids of blocks [32k, 32k+32)
    int32_t ids_next = 0;
    if (!waited) { pdl_wait(); waited = true; }

    // q^T as B fragments: lane (g, c) holds MMA column g (zero for unused columns)
    typename TP::Query Q;
    float cs0, cs1;                                              // score scale of columns 2c, 2c+1 (log2 units)
    {
      bool ok = g < G;
      const uint16_t* qrow = p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + (ok ? g : 0)) * D;
      if constexpr (kVarQ) {                                     // column g = (query token g / G, head g % G)
        const int qt = g / G;
        ok = qt < n_qtok;
        qrow = p.q + (static_cast<int64_t>(batch_idx + (ok ? qt : 0)) * p.num_q_heads + h * G + (ok ? g - qt * G : 0)) * D;
      }
      TP::load_query(Q, qrow, ok, c, p.scale_log2, cs0, cs1);
    }

    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // columns 2c, 2c+1 (l: this lane's rows only)
    float o[MT][4];
#pragma unroll
    for (int i = 0; i < MT; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;

    unsigned char* const kvh = kv + static_cast<int64_t>(h) * TP::kPoolTileBytes;
    unsigned char* const last_tile = kvh + last_blk * blk_stride;
    const int64_t new_row = (static_cast<int64_t>(batch_idx) * p.num_kv_heads + h) * D;
    typename TP::NewRow nr;

    // start the copies of virtual tile v into ring slot v % R (one cp.async group per tile, empty past the end).
    // virtual tile v -> real tile: special ? (v == 0 ? n_blocks - 1 : v - 1) : v
    auto issue = [&](int v) {
      if (v < n_blocks) {
        const bool first_special = special && v == 0;
        const int t = first_special ? n_blocks - 1 : v - sp;
        const unsigned char* tile;
        if (first_special) {
          tile = last_tile;
        } else {
          if ((t & 31) == 0 && t > 0) ids = ids_next;
          if ((t & 31) == 8 && t + 24 + lane < n_blocks) ids_next = __ldg(bt + t + 24 + lane);
          tile = kvh + __shfl_sync(kFull, ids, t & 31) * blk_stride;
        }
        const int nv = n_tokens - t * kBlockSize;
        bool by_tma = false;
        if constexpr (TP::kTma) by_tma = nv >= kBlockSize && !first_special;   // full tiles: one bulk tensor copy
        const uint32_t dst = ring + (v % R) * TP::kSlotStride, dst_sc = TP::template scales_addr<R>(ring, v % R);
        if (by_tma) {
          if (lane == 0) {
            fence_proxy_async();                                 // the slot's last readers used the generic proxy
            TP::tma_tile(dst, dst_sc, p.tmap, bars + (v % R) * 8, p.tma_row0 + (tile - kv) / 128, tile);
          }
        } else {
          TP::template copy_tile<kAppend>(dst, dst_sc, tile, nv, lane, first_special ? nv - 1 : -1,
                                          p.k_new + new_row, p.v_new + new_row);
        }
        if constexpr (kAppend) {
          if (first_special) {                                   // a3: the new row goes into the pool
            TP::append_row(last_tile, nv - 1, p.k_new + new_row, p.v_new + new_row, lane, nr);
            if (h == 0 && lane == 0) p.block_table[static_cast<int64_t>(slot) * p.bt_stride + blk_begin + n_blocks - 1] = last_blk;
          }
        }
      }
      if constexpr (!TP::kTma) cp_async_commit();
    };

    auto consume = [&](int v) {
      const int t = (special && v == 0) ? n_blocks - 1 : v - sp;
      const int nv = n_tokens - t * kBlockSize;
      const uint32_t slot_addr = ring + (v % R) * TP::kSlotStride, sc_addr = TP::template scales_addr<R>(ring, v % R);
      if constexpr (TP::kTma) {                                  // wait for the tile: mbarrier (TMA) or this warp's LDGSTS
        if (nv >= kBlockSize && !(special && v == 0)) {
          mbar_wait(bars + (v % R) * 8, (bar_parity >> (v % R)) & 1u);
          bar_parity ^= 1u << (v % R);
        } else {
          cp_async_commit();
          cp_async_wait<0>();
          __syncwarp();
        }
      }
      if constexpr (kAppend && TP::kPatchNewRow) {
        if (special && v == 0) {
          TP::patch_slot(slot_addr, sc_addr, nv - 1, lane, nr);
          __syncwarp();
        }
      }
      typename TP::Frag T;
      TP::load_frags(T, slot_addr, sc_addr, g, c);
      float s[4], vs[2];
      TP::scores(T, Q, cs0, cs1, s, vs);
      float iv0 = 1.f, iv1 = 1.f;
      if constexpr (TP::kVScaled) {                              // t = s + log2(vs); ragged last block masked by index
        const bool ok0 = tg < nv, ok1 = tg + 8 < nv;
        const float lv0 = ok0 ? fast_log2(vs[0]) : -INFINITY, lv1 = ok1 ? fast_log2(vs[1]) : -INFINITY;
        iv0 = ok0 ? fast_rcp(vs[0]) : 0.f;
        iv1 = ok1 ? fast_rcp(vs[1]) : 0.f;
        s[0] += lv0; s[1] += lv0; s[2] += lv1; s[3] += lv1;
      } else if (nv < kBlockSize) {                              // ragged last block: mask by index, not value
        if (tg >= nv) s[0] = s[1] = -INFINITY;
        if (tg + 8 >= nv) s[2] = s[3] = -INFINITY;
      }
      if constexpr (kVarQ) {                                    // causal: column sees tokens <= its own position
        const int tok = t * kBlockSize + tg;
        if (tok > rel0) s[0] = -INFINITY;
        if (tok > rel1) s[1] = -INFINITY;
        if (tok + 8 > rel0) s[2] = -INFINITY;
        if (tok + 8 > rel1) s[3] = -INFINITY;
      }
      // ---- online softmax over the token axis (= across the 8 lanes sharing c) ----
      float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
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
      const float p0 = fast_exp2(s[0] - ms0), p1 = fast_exp2(s[1] - ms1);
      const float p2 = fast_exp2(s[2] - ms0), p3 = fast_exp2(s[3] - ms1);
      if constexpr (TP::kVScaled) {
        l0 = l0 * a0 + (p0 * iv0 + p2 * iv1);
        l1 = l1 * a1 + (p1 * iv0 + p3 * iv1);
      } else {
        l0 = l0 * a0 + (p0 + p2);
        l1 = l1 * a1 + (p1 + p3);
      }
      if (!TP::kLazyRescale || __any_sync(kFull, moved)) {       // the running maximum settles after a few tiles
#pragma unroll
        for (int i = 0; i < MT; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
      }
      TP::pv(T, p0, p1, p2, p3, o);
    };

#pragma unroll
    for (int v = 0; v < R - 1; ++v) issue(v);                    // R - 1 tiles ahead
    for (int v = 0; v < n_blocks; ++v) {
      if constexpr (!TP::kTma) cp_async_wait<R - 2>();           // tile v has landed (this lane's copies)
      __syncwarp();                                              // ... everyone's; and slot (v - 1) % R is free
      issue(v + R - 1);
      consume(v);
    }
    if constexpr (!TP::kTma) cp_async_wait<0>();
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
      // element e = 8 cs + k of this lane: d column col0(g, cs) + k, register o[e % (NE/2)][2*(e/(NE/2)) + hh]
      if (pidx < 0) {
        const float inv = 1.f / l;
        uint16_t* op = p.out + out_row * D;
#pragma unroll
        for (int cs = 0; cs < NE / 8; ++cs) {
          uint32_t w[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int e = cs * 8 + 2 * k;
            w[k] = pack_bf16x2(o[e % (NE / 2)][2 * (e / (NE / 2)) + hh] * inv,
                               o[(e + 1) % (NE / 2)][2 * ((e + 1) / (NE / 2)) + hh] * inv);
          }
          *reinterpret_cast<uint4*>(op + TP::col0(g, cs)) = make_uint4(w[0], w[1], w[2], w[3]);
        }
      } else {
        float* po = p.part_o + (static_cast<int64_t>(pidx) * PG + head) * D;
#pragma unroll
        for (int cs = 0; cs < NE / 8; ++cs) {
          float f[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const int e = cs * 8 + k;
            f[k] = o[e % (NE / 2)][2 * (e / (NE / 2)) + hh];
          }
          float4* dst = reinterpret_cast<float4*>(po + TP::col0(g, cs));
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
      last = __shfl_sync(kFull, last, 0);
      if (last) {
        __threadfence();
        if constexpr (kVarQ) {
          for (int qt = 0; qt < n_qtok; ++qt)
            combine_cols<D>(p.part_o, p.part_ml, pbase, n_chunks, 8, qt * G, G,
                            p.out + (static_cast<int64_t>(batch_idx + qt) * p.num_q_heads + h * G) * D, lane);
        } else {
          combine_cols<D>(p.part_o, p.part_ml, pbase, n_chunks, G, 0, G,
                          p.out + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G) * D, lane);
        }
      }
    }
    if (lane == 0) item = n_warps + atomicAdd(&p.counters[0], 1);
    item = __shfl_sync(kFull, item, 0);
  }
  if (!waited) pdl_wait();                                       // a warp without work still orders the rewind below

  // Last CTA out rewinds the work counter for the next launch (attention launches of one pool are ordered on one
  // stream — enforced by the host; counters[1] wraps to 0 by itself).
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned prev = atomicInc(reinterpret_cast<unsigned*>(&p.counters[1]), gridDim.x - 1);
    if (prev == gridDim.x - 1) p.counters[0] = 0;
  }
}

}  // namespace kvp
