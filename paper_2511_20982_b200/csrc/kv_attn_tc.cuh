// kv_attn_tc.cuh — a4 (+ a3, a5) on the 5th-generation tensor cores: split-KV paged decode attention over an FP8
// (e4m3) pool with head_dim 128, written for tcgen05 / TMEM / TMA.   attn_tc_kernel<kAppend>
//
// Why a second formulation.  The mma.sync kernel (kv_attn.cuh) has to UNPACK every e4m3 code to f16 in registers
// (one F2FP per code pair) before an HMMA can eat it: 341 warp instructions per 4 KiB tile, ALU pipe 51 % busy, and
// on short launches the warp's dependent chain, not HBM, sets the pace (profiles/README.md r02).  tcgen05.mma
// kind::f8f6f4 reads e4m3 operands straight from shared memory, so here NO thread ever touches a K or V byte:
//
//   tile  = 128 tokens (8 blocks) of one (request chunk, kv head): K8[128][128 B] | V8[128][128 B] | sc[128]{ks, vs}
//   GEMM1   S^T[128 tok x 16]  = K8[128 x 128] . Q8^T     M = tokens, K = d, N = 2 e4m3 terms x 8 heads
//   GEMM2   O^T[128 d  x 32] += V8^T[128 x 128 tok] . P^T  M = d, K = tokens, N = 4 e5m2 terms x 8 heads
//
// Both A operands are the tile exactly as TMA lays it down with the 128-byte swizzle: rows of 128 bytes = one token's
// codes.  For GEMM1 that is the canonical K-major layout (contraction index d contiguous); for GEMM2 the SAME bytes
// are the canonical MN-major layout (M = d contiguous, contraction index = token row) — the instruction descriptor's
// a_major bit does the transpose that the mma.sync kernel does with PRMTs.
//   * q (bf16) is scaled by a power of two so that its row maximum lies in [128, 256) and split into two e4m3 terms
//     q = a1 + a2 (exact for every element within 2^-9 of the row maximum; absolute error <= 2^-17 max|q| below);
//     the two terms occupy 16 N-columns and are summed after the TMEM load.
//   * the weights p' = 2^(s + log2 vs - m_ref) are rounded to f16 (as in the mma.sync kernel) and that f16 is split
//     EXACTLY into four e5m2 terms by masking its top byte three times (f16 and e5m2 share sign and exponent, and
//     x - (x & 0xff00) is exact); a token's 32 bytes [term][head] go into the B operand of GEMM2 with two 16-byte
//     stores (MN-major, un-swizzled: kTcPByToken below); the four column groups of O^T are summed after the TMEM
//     load.  Numerics are those of the mma.sync kernel.
//   * m_ref is a LAZY reference: it moves only when some score of a tile exceeds it by more than 2^8 (p' <= 256; times the
//     bias 2^7 below, 2^15 fits f16 and e5m2), so the rescale of O^T in TMEM (tcgen05.ld / st) runs a handful of times per unit.
//
// Roles (256 threads, 2 CTAs per SM, 112.5 KiB of shared memory each):
//   warps 0-3  softmax + epilogue: thread i owns token i of a tile (TMEM lane i of S^T) and column d = i of O^T
//   warp 4     lead producer: claims units, stages Q8, appends the new row (a3), publishes each unit's descriptor to
//              the two helper warps, issues the scale copies of the 3-stage tile ring
//   warp 5     MMA issuer (one lane) + TMEM allocation
//   warp 6, 7  helper producers: the K-code and the V-code copies of every tile.  A tile is 24 bulk copies (8 blocks x
//              {K codes, V codes, scales}) and ONE warp issues a copy every ~45 ns: 1.1 us per tile, at which point the
//              producer, not HBM, paces the CTA (profiles/README.md r02) — so the issue is spread over three warps.
//   The producers run ahead ACROSS unit boundaries (they own no registers worth mentioning).
//   The fused append never waits for a global store to reach the TMA unit: the lead producer writes the quantised row to
//   the pool AND to shared memory, the tile holding its slot is fetched like any other, and the MMA warp patches the
//   row into the stage before that tile's GEMM1 (the softmax thread of that token takes its two scales from the copy).
// All hand-offs are mbarriers; the only block-wide barrier is at start-up and tear-down.
#pragma once

#include <cuda_fp16.h>

#include "kv_attn.cuh"

namespace kvp {

constexpr int kTcThreads = 256;
constexpr int kTcSoftmaxThreads = 128;
constexpr int kTcStages = 3;
constexpr int kTcTileBlocks = 8, kTcTileTokens = kTcTileBlocks * kBlockSize;
constexpr uint32_t kTcStageBytes = 2 * kTcTileTokens * 128 + kTcTileTokens * 8;   // 33792 = 33 KiB
constexpr uint32_t kTcQBytes = 16 * 128, kTcPBytes = 32 * 128;
constexpr uint32_t kTcMiscOff = kTcStages * kTcStageBytes + 2 * kTcQBytes + 2 * kTcPBytes;
constexpr uint32_t kTcSmemBytes = kTcMiscOff + 1664;                              // 115328 = 112.6 KiB
constexpr uint32_t kTcTmemCols = 128;       // S^T: 2 x 16 columns, O^T: 2 x 32 columns
constexpr float kTcLazyLog2 = 8.f;          // m_ref moves when a score exceeds it by more than this (log2 units)
// The weights are fed as 2^(s - m_ref + kTcWeightBias): the four e5m2 terms of a weight bottom out at e5m2's smallest
// subnormal, 2^-16, whereas the f16 they split has 2^-24 — so the weights sit as high as the formats allow (<= 2^15 with the
// lazy reference, below e5m2's 57344 and f16's 65504) and keep all 11 bits down to 2^-13 of the reference.  O and l
// carry the same factor; it cancels in O / l and in the merge of partials.
constexpr float kTcWeightBias = 7.f;

// ---- tcgen05 / TMEM wrappers ---------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// all tcgen05.mma issued so far by this thread arrive (once) on `bar` when they have completed
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem desc] . B[smem desc], 8-bit float operands (formats and majors in idesc), K = 32 per instruction
__device__ __forceinline__ void tc_mma_f8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
               "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
                 "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
                 "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
               : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float (&v)[32]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
               "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
               ::"r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])),
                 "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])),
                 "r"(__float_as_uint(v[7])), "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])),
                 "r"(__float_as_uint(v[11])), "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])),
                 "r"(__float_as_uint(v[15])), "r"(__float_as_uint(v[16])), "r"(__float_as_uint(v[17])), "r"(__float_as_uint(v[18])),
                 "r"(__float_as_uint(v[19])), "r"(__float_as_uint(v[20])), "r"(__float_as_uint(v[21])), "r"(__float_as_uint(v[22])),
                 "r"(__float_as_uint(v[23])), "r"(__float_as_uint(v[24])), "r"(__float_as_uint(v[25])), "r"(__float_as_uint(v[26])),
                 "r"(__float_as_uint(v[27])), "r"(__float_as_uint(v[28])), "r"(__float_as_uint(v[29])), "r"(__float_as_uint(v[30])),
                 "r"(__float_as_uint(v[31]))
               : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// the 128 softmax threads only (warps 4 and 5 never take part)
__device__ __forceinline__ void softmax_barrier() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
__device__ __forceinline__ void sts8(uint32_t addr, uint32_t v) { asm volatile("st.shared.u8 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// Shared-memory matrix descriptor of a [rows][128 B] operand in the 128-byte swizzle (what TMA writes with
// CU_TENSOR_MAP_SWIZZLE_128B and what the producer / softmax threads write by hand): 8-row groups 1 KiB apart.
//   K-major  (rows = M or N index, the 128 bytes = contraction index):  SBO = 1024, LBO unused (1)
//   MN-major (the 128 bytes = M index, rows = contraction index):       SBO = 1024 between 8-row groups, one 128-element
//                                                                       atom along M so LBO is unused
// bits [0,14) start >> 4 | [16,30) LBO >> 4 | [32,46) SBO >> 4 | [46,48) version = 1 | [61,64) layout = 2 (SWIZZLE_128B)
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t addr) {
  return static_cast<uint64_t>((addr & 0x3ffffu) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptors (kind::f8f6f4): D = f32 (bits 4-5 = 1), A format bits 7-9, B format bits 10-12 (0 e4m3, 1 e5m2),
// a_major bit 15 (1 = MN-major), b_major bit 16, N >> 3 at bits 17-22, M >> 4 at bits 24-28
constexpr uint32_t kTcIdescQK = (1u << 4) | (0u << 7) | (0u << 10) | (0u << 15) | ((16u >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t kTcIdescPV = (1u << 4) | (0u << 7) | (1u << 10) | (1u << 15) | ((32u >> 3) << 17) | ((128u >> 4) << 24);
// P^T, the B operand of GEMM2 (N = 32 (term, head) columns, K = 128 tokens).  kTcPByToken = true: MN-major and
// un-swizzled — core matrices of 8 tokens x 16 N-bytes (128 contiguous bytes, a token's 16 bytes per row), the two
// N-halves 2 KiB apart (SBO), 8-token groups 128 B apart (LBO) — so that the thread that owns a token writes its 32
// weight bytes with TWO 16-byte stores; a warp's stores are 512 contiguous bytes, no bank conflict.  false: K-major in
// the 128-byte swizzle (rows = (term, head), a token = one byte of each of 32 rows: 32 one-byte stores per thread, four
// lanes to a word — 2.5-8.4 M bank conflicts per launch, profiles/README.md r02).
constexpr bool kTcPByToken = true;
constexpr uint32_t kTcIdescPVt = kTcIdescPV | (1u << 16);
__device__ __forceinline__ uint64_t tc_smem_desc_p(uint32_t addr) {   // layout type 0 (no swizzle), version 1
  return static_cast<uint64_t>((addr & 0x3ffffu) >> 4) | ((128ull >> 4) << 16) | ((2048ull >> 4) << 32) | (1ull << 46);
}

struct TcUnit {            // what the producer hands to the MMA and softmax warps for one unit (shared memory, 64 bytes)
  int32_t n_tiles;         // 0: no more work
  int32_t n_tokens;        // valid tokens of the chunk
  int32_t batch_idx, h;
  int32_t pidx, pbase, n_chunks;
  int32_t new_row;         // fused append: row of the unit's LAST tile that holds the token being appended, else -1
  float qs[8];             // per head: 2^(eb - 134) * sm_scale * log2(e), the factor that turns K8 . q8 * ks into log2 scores
};
static_assert(sizeof(TcUnit) == 64, "TcUnit");

struct TcDesc {            // what the lead producer hands to the helper producers for one unit (shared memory, 160 bytes)
  int32_t n_blocks;        // 0: no more work
  int32_t row_h;           // first 128-byte row of (layer, block 0, this kv head) in the tensor map
  int32_t slot, blk_begin; // where the chunk's block ids continue in the device block table
  int32_t owns_last;       // the chunk ends with the request's last block ...
  int32_t last_blk;        // ... whose physical id is this (the device block table may not hold it yet)
  int32_t pad[2];
  int32_t ids[32];         // physical ids of the chunk's first 32 blocks
};
static_assert(sizeof(TcDesc) == 160, "TcDesc");

template <bool kAppend>
__global__ void __launch_bounds__(kTcThreads, 2) attn_tc_kernel(const __grid_constant__ AttnParams p) {
  extern __shared__ __align__(1024) unsigned char tc_smem[];
  constexpr int D = 128;
  using TP = Fp8Tiles<128>;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem0 = static_cast<uint32_t>(__cvta_generic_to_shared(tc_smem));
  const uint32_t q_smem = smem0 + kTcStages * kTcStageBytes;
  const uint32_t p_smem = q_smem + 2 * kTcQBytes;
  const uint32_t misc = smem0 + kTcMiscOff;
  // mbarriers
  const uint32_t b_full = misc, b_empty = misc + 24, b_d1_full = misc + 48, b_d1_empty = misc + 64, b_p_full = misc + 80,
                 b_p_free = misc + 96, b_o_full = misc + 112, b_o_empty = misc + 128, b_u_full = misc + 144, b_u_empty = misc + 160,
                 b_dsc_full = misc + 192, b_dsc_empty = misc + 208;
  const uint32_t tmem_slot = misc + 176, merge_flag = misc + 180;
  TcUnit* const units = reinterpret_cast<TcUnit*>(tc_smem + kTcMiscOff + 256);
  const uint32_t flags_smem = misc + 384;   // [2][4] int
  const uint32_t wmax_smem = misc + 416;    // [2][4][8] float
  const uint32_t lsum_smem = misc + 672;    // [4][8] float
  const uint32_t desc_smem = misc + 800;    // [2] TcDesc
  const uint32_t stash_smem = misc + 1120;  // [2] the appended row as the pool stores it: K codes[128] | V codes[128] | ks, vs | pad (272 B)

  if (threadIdx.x == 0) {
    if (smem0 & 1023u) __trap();            // the 128-byte swizzle is a function of the shared-memory address
    for (int s = 0; s < kTcStages; ++s) { mbar_init(b_full + 8 * s, 3); mbar_init(b_empty + 8 * s, 1); }   // three issuing warps
    for (int i = 0; i < 2; ++i) {
      mbar_init(b_d1_full + 8 * i, 1); mbar_init(b_d1_empty + 8 * i, kTcSoftmaxThreads);
      mbar_init(b_p_full + 8 * i, kTcSoftmaxThreads); mbar_init(b_p_free + 8 * i, 1);
      mbar_init(b_o_full + 8 * i, 1); mbar_init(b_o_empty + 8 * i, kTcSoftmaxThreads);
      mbar_init(b_u_full + 8 * i, 1); mbar_init(b_u_empty + 8 * i, kTcSoftmaxThreads);
      mbar_init(b_dsc_full + 8 * i, 1); mbar_init(b_dsc_empty + 8 * i, 2);
    }
    mbar_init_fence();
  }
  if (warp == 5) {
    tmem_alloc(tmem_slot, kTcTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = lds32(tmem_slot);

  pdl_launch_dependents();
  const int G = p.group;

  if (warp == 4) {
    // ===================================== producer =====================================
    // A unit costs a chain of dependent global loads before its first tile can be asked for (claim -> work item ->
    // block ids; q and the new rows hang off the work item).  With two CTAs per SM there are no other warps to hide
    // that chain behind, so it is software-pipelined: while the last three tiles of unit u are being issued the warp
    // claims unit u + 1, fetches its work item, then its block ids, its q rows and its new K / V row — one link per
    // tile, each link's loads in flight while the warp waits for a free stage anyway.  At the unit switch the first
    // tile goes out before anything else; Q8 is staged and the new row appended while it is in flight.
    bool waited = !p.chained;
    if (waited) pdl_wait();
    unsigned char* const kv = reinterpret_cast<unsigned char*>(p.kv_layer);
    const int64_t blk_stride = static_cast<int64_t>(p.num_kv_heads) * TP::kPoolTileBytes;
    const int b = lane & (kTcTileBlocks - 1);
    const int qhead = lane >> 2, quarter = lane & 3;                 // Q8 staging: head of the group, 32 d columns
    const bool qok = qhead < G;
    uint32_t g_tile = 0, u_seq = 0;

    // what is known of a unit before it starts
    struct Desc { int32_t unit; int4 w0, w1; int32_t ids; uint4 q[4]; uint4 nrow; };
    auto fetch_item = [&](Desc& d) {                                 // link 2: the work item
      if (d.unit < p.n_units) {
        const int4* wi = reinterpret_cast<const int4*>(p.items) + (d.unit / p.num_kv_heads) * 2;
        d.w0 = __ldg(wi);
        d.w1 = __ldg(wi + 1);
      }
    };
    auto fetch_rows = [&](Desc& d, bool with_inputs) {               // link 3: block ids (+ q rows, new K / V row)
      if (d.unit >= p.n_units) return;
      const int h = d.unit % p.num_kv_heads;
      const int batch_idx = d.w0.x, slot = d.w0.y, blk_begin = d.w0.z, n_blocks = d.w0.w;
      const int32_t* bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
      d.ids = lane < n_blocks ? __ldg(bt + lane) : 0;                // physical ids of blocks [0, 32) of the chunk
      if (with_inputs) {
        const uint16_t* qrow = p.q + (static_cast<int64_t>(batch_idx) * p.num_q_heads + h * G + (qok ? qhead : 0)) * D + quarter * 32;
#pragma unroll
        for (int k = 0; k < 4; ++k) d.q[k] = ldg_stream_pred(qrow + k * 8, qok);
        if constexpr (kAppend) {
          const int n_chunks = static_cast<int>(static_cast<uint32_t>(d.w1.z) >> 16), chunk_idx = d.w1.z & 0xffff;
          if (chunk_idx == n_chunks - 1) {
            const int64_t new_row = (static_cast<int64_t>(batch_idx) * p.num_kv_heads + h) * D;
            d.nrow = TP::append_load(p.k_new + new_row, p.v_new + new_row, lane);
          }
        }
      }
    };

    Desc cur{};
    cur.unit = blockIdx.x;
    fetch_item(cur);
    fetch_rows(cur, waited);                                         // q, k_new, v_new only after griddepcontrol.wait
    if (!waited) {
      pdl_wait();
      waited = true;
      if (cur.unit < p.n_units) {                                    // (the block ids are re-read: harmless)
        fetch_rows(cur, true);
      }
    }

    for (;; ++u_seq) {
      const int e = u_seq & 1;
      TcUnit* const U = units + e;
      TcDesc* const Dsc = reinterpret_cast<TcDesc*>(tc_smem + kTcMiscOff + 800) + e;
      mbar_wait(b_dsc_empty + 8 * e, ((u_seq >> 1) & 1u) ^ 1u);       // both helpers have read the descriptor two units back
      if (cur.unit >= p.n_units) {
        mbar_wait(b_u_empty + 8 * e, ((u_seq >> 1) & 1u) ^ 1u);
        if (lane == 0) {
          U->n_tiles = 0;
          Dsc->n_blocks = 0;
          mbar_arrive(b_u_full + 8 * e);
          mbar_arrive(b_dsc_full + 8 * e);
        }
        break;
      }
      const int h = cur.unit % p.num_kv_heads;
      const int batch_idx = cur.w0.x, slot = cur.w0.y, blk_begin = cur.w0.z, n_blocks = cur.w0.w;
      const int n_tokens = cur.w1.x;
      const int n_chunks = static_cast<int>(static_cast<uint32_t>(cur.w1.z) >> 16), chunk_idx = cur.w1.z & 0xffff, last_blk = cur.w1.w;
      const int pbase = cur.w1.y < 0 ? -1 : cur.w1.y + h * n_chunks;
      const int n_tiles = (n_blocks + kTcTileBlocks - 1) / kTcTileBlocks;
      const bool owns_last = chunk_idx == n_chunks - 1;
      const int32_t* bt = p.block_table + static_cast<int64_t>(slot) * p.bt_stride + blk_begin;
      int32_t ids = cur.ids, ids_next = 0;
      const unsigned char* const sc_h = kv + static_cast<int64_t>(h) * TP::kPoolTileBytes + 4096;
      const bool append = kAppend && owns_last;
      // ---- the unit's descriptor goes to the helper producers before anything else ----
      Dsc->ids[lane] = ids;
      if (lane == 0) {
        Dsc->n_blocks = n_blocks; Dsc->row_h = static_cast<int32_t>(p.tma_row0) + h * 33; Dsc->slot = slot; Dsc->blk_begin = blk_begin;
        Dsc->owns_last = owns_last ? 1 : 0; Dsc->last_blk = last_blk;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(b_dsc_full + 8 * e);

      Desc nxt{};
      nxt.unit = p.n_units;
      int link = 0;                                                  // links of the next unit's chain already started
      for (int t = 0; t < n_tiles; ++t, ++g_tile) {
        const int left = n_tiles - t;                                // tiles of this unit not yet issued
        if (left <= 3 && link == 0) {                                // link 1: claim
          int32_t c = 0;
          if (lane == 0) c = gridDim.x + atomicAdd(&p.counters[0], 1);
          nxt.unit = c;
          link = 1;
        }
        if (left <= 2 && link == 1) {
          nxt.unit = __shfl_sync(kFull, nxt.unit, 0);
          fetch_item(nxt);
          link = 2;
        }
        // ---- tile t, this warp's share: the scales of its (up to) 8 blocks, lane b < 8 owns block b ----
        {
          const uint32_t s = g_tile % kTcStages;
          const int blk0 = t * kTcTileBlocks;
          if ((blk0 & 31) == 0 && blk0 > 0) ids = ids_next;
          if ((blk0 & 31) == 8 && blk0 + 24 + lane < n_blocks) ids_next = __ldg(bt + blk0 + 24 + lane);
          int32_t id = __shfl_sync(kFull, ids, (blk0 + b) & 31);
          if (owns_last && blk0 + b == n_blocks - 1) id = last_blk;   // see TcDesc::last_blk
          const int nb = min(kTcTileBlocks, n_blocks - blk0);
          const uint32_t st = smem0 + s * kTcStageBytes, bar = b_full + 8 * s;
          mbar_wait(b_empty + 8 * s, ((g_tile / kTcStages) & 1u) ^ 1u);
          if (lane == 0) mbar_arrive_expect_tx(bar, static_cast<uint32_t>(nb) * 128u);
          __syncwarp();
          if (lane < nb) bulk_load_1d(st + 32768 + b * 128, sc_h + id * blk_stride, 128, bar);
        }
        if (t == 0) {
          // ---- Q8 (while tile 0 is in flight): two e4m3 terms of this lane's 32 d columns, rows term * 8 + head ----
          mbar_wait(b_u_empty + 8 * e, ((u_seq >> 1) & 1u) ^ 1u);
          uint32_t mx = 0;
#pragma unroll
          for (int k = 0; k < 4; ++k) mx = max(mx, amax_bits8(cur.q[k]));
          mx = max(mx, __shfl_xor_sync(kFull, mx, 1));
          mx = max(mx, __shfl_xor_sync(kFull, mx, 2));
          const uint32_t eb = min(max(mx >> 7, 8u), 253u);          // biased exponent of the row maximum
          const float sf = __uint_as_float((261u - eb) << 23);       // 2^(134 - eb): row maximum -> [128, 256)
          if (quarter == 0) U->qs[qhead] = qok ? __uint_as_float((eb - 7u) << 23) * p.scale_log2 : 0.f;
          uint32_t t1[8], t2[8];                                     // 32 codes per term = 8 words
#pragma unroll
          for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int w = 0; w < 4; w += 2) {
              uint32_t c1[2], c2[2];
#pragma unroll
              for (int ww = 0; ww < 2; ++ww) {
                const uint32_t e2 = u4_get(cur.q[k], w + ww);
                const float x0 = __uint_as_float(e2 << 16) * sf, x1 = __uint_as_float(e2 & 0xffff0000u) * sf;
                c1[ww] = f32x2_to_e4m3x2(x0, x1);
                const uint32_t hb = e4m3x2_lo_to_f16x2(c1[ww]);     // what the first term holds, exactly
                const float2 back = __half22float2(*reinterpret_cast<const __half2*>(&hb));
                c2[ww] = f32x2_to_e4m3x2(x0 - back.x, x1 - back.y);
              }
              t1[2 * k + w / 2] = c1[0] | (c1[1] << 16);
              t2[2 * k + w / 2] = c2[0] | (c2[1] << 16);
            }
          const uint32_t qb = q_smem + e * kTcQBytes;
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            const int chunk = quarter * 2 + half;
            sts128(qb + qhead * 128 + ((chunk ^ qhead) << 4), make_uint4(t1[4 * half], t1[4 * half + 1], t1[4 * half + 2], t1[4 * half + 3]));
            sts128(qb + (8 + qhead) * 128 + ((chunk ^ qhead) << 4), make_uint4(t2[4 * half], t2[4 * half + 1], t2[4 * half + 2], t2[4 * half + 3]));
          }
          // a3 inside a4: the unit that owns the request's last block quantises the new row (ingest's arithmetic, ingest's
          // bytes), writes it to the pool for the steps to come, and leaves a copy in shared memory: the tile that holds
          // its slot is fetched like any other (stale bytes in that row) and the MMA warp patches the row in before it
          // issues the tile's GEMM1.  Nothing waits for a global store to become visible to the TMA unit.
          if constexpr (kAppend) {
            if (append) {
              unsigned char* const last_tile = kv + static_cast<int64_t>(h) * TP::kPoolTileBytes + last_blk * blk_stride;
              typename TP::NewRow nr;
              TP::append_store(last_tile, n_tokens - (n_blocks - 1) * kBlockSize - 1, cur.nrow, lane, nr);
              if (h == 0 && lane == 0) p.block_table[static_cast<int64_t>(slot) * p.bt_stride + blk_begin + n_blocks - 1] = last_blk;
              const uint32_t sa = stash_smem + e * 272u;
              asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(sa + lane * 8), "r"(nr.codes.x), "r"(nr.codes.y) : "memory");
              if ((lane & 15) == 0) sts32(sa + 256 + (lane >> 4) * 4, __float_as_uint(nr.scale));
            }
          }
          fence_proxy_async();                                        // Q8 in shared memory -> visible to the tensor core
          __syncwarp();
          if (lane == 0) {
            U->n_tiles = n_tiles; U->n_tokens = n_tokens; U->batch_idx = batch_idx; U->h = h;
            U->pidx = cur.w1.y < 0 ? -1 : pbase + chunk_idx; U->pbase = pbase; U->n_chunks = n_chunks;
            U->new_row = append ? n_tokens - 1 - (n_tiles - 1) * kTcTileTokens : -1;
            mbar_arrive(b_u_full + 8 * e);
          }
        }
        if (left <= 1 && link == 2) {                                // link 3 (after this unit's q registers are dead)
          fetch_rows(nxt, true);
          link = 3;
        }
      }
      cur = nxt;
    }
  } else if (warp >= 6) {
    // ===================================== helper producers: K codes (warp 6), V codes (warp 7) =====================================
    if (!p.chained) pdl_wait();                                      // they read the block table beyond a chunk's first 32 ids
    const int b = lane & (kTcTileBlocks - 1);
    const uint32_t part = warp == 6 ? 0u : 16384u;                   // offset of this warp's codes inside a stage ...
    const int32_t part_row = warp == 6 ? 0 : 16;                     // ... and inside a pool tile (128-byte rows)
    const int32_t row_blk = 33 * p.num_kv_heads;
    uint32_t g_tile = 0, u_seq = 0;
    for (;; ++u_seq) {
      const int e = u_seq & 1;
      mbar_wait(b_dsc_full + 8 * e, (u_seq >> 1) & 1u);
      const uint32_t da = desc_smem + e * static_cast<uint32_t>(sizeof(TcDesc));
      const uint4 d0 = lds128(da), d1 = lds128(da + 16);
      int32_t ids = static_cast<int32_t>(lds32(da + 32 + lane * 4)), ids_next = 0;
      __syncwarp();
      if (lane == 0) mbar_arrive(b_dsc_empty + 8 * e);
      const int n_blocks = static_cast<int>(d0.x);
      if (n_blocks == 0) break;
      const int32_t row_h = static_cast<int32_t>(d0.y) + part_row;
      const int32_t* bt = p.block_table + static_cast<int64_t>(static_cast<int32_t>(d0.z)) * p.bt_stride + static_cast<int32_t>(d0.w);
      const bool owns_last = d1.x != 0;
      const int32_t last_blk = static_cast<int32_t>(d1.y);
      const int n_tiles = (n_blocks + kTcTileBlocks - 1) / kTcTileBlocks;
      for (int t = 0; t < n_tiles; ++t, ++g_tile) {
        const uint32_t s = g_tile % kTcStages;
        const int blk0 = t * kTcTileBlocks;
        if ((blk0 & 31) == 0 && blk0 > 0) ids = ids_next;
        if ((blk0 & 31) == 8 && blk0 + 24 + lane < n_blocks) ids_next = __ldg(bt + blk0 + 24 + lane);
        int32_t id = __shfl_sync(kFull, ids, (blk0 + b) & 31);
        if (owns_last && blk0 + b == n_blocks - 1) id = last_blk;
        const int nb = min(kTcTileBlocks, n_blocks - blk0);
        const uint32_t st = smem0 + s * kTcStageBytes + part, bar = b_full + 8 * s;
        mbar_wait(b_empty + 8 * s, ((g_tile / kTcStages) & 1u) ^ 1u);
        if (lane == 0) mbar_arrive_expect_tx(bar, static_cast<uint32_t>(nb) * 2048u);
        __syncwarp();
        if (lane < nb) tma_load_2d(st + b * 2048, p.tmap, bar, 0, row_h + id * row_blk);
      }
    }
  } else if (warp == 5) {
    // ===================================== MMA issuer: one thread =====================================
    if (lane == 0) {
      uint32_t g1 = 0, g2 = 0, u_seq = 0;                          // GEMM1 / GEMM2 / unit sequence numbers of this CTA
      for (;; ++u_seq) {
        const int e = u_seq & 1;
        mbar_wait(b_u_full + 8 * e, (u_seq >> 1) & 1u);
        const int n_tiles = static_cast<int>(lds32(misc + 256 + e * 64));
        if (n_tiles == 0) break;
        const int new_row = kAppend ? static_cast<int>(lds32(misc + 256 + e * 64 + 28)) : -1;
        mbar_wait(b_o_empty + 8 * e, ((u_seq >> 1) & 1u) ^ 1u);    // O^T buffer e: the unit two back has been read out
        const uint64_t qdesc = tc_smem_desc(q_smem + e * kTcQBytes);
        const uint32_t o_tmem = tmem + 32 + e * 32;
        // GEMM1 runs up to two tiles ahead of GEMM2 (S^T is double-buffered).  Whichever of "the next tile has landed"
        // and "the weights of the oldest open tile are ready" happens first is issued first, so a stage goes back to
        // the producer as soon as its GEMM2 can run, whether or not the next tile is there yet.
        int t1 = 0, t2 = 0;                                        // tiles of this unit whose GEMM1 / GEMM2 has been issued
        while (t2 < n_tiles) {
          const bool may1 = t1 < n_tiles && t1 < t2 + 2;
          if (may1) {
            const uint32_t s1 = g1 % kTcStages, db = g1 & 1u;
            const bool must = t1 == t2;                            // nothing else to do: wait for the tile
            if (must) {
              mbar_wait(b_full + 8 * s1, (g1 / kTcStages) & 1u);
              mbar_wait(b_d1_empty + 8 * db, ((g1 >> 1) & 1u) ^ 1u);
            }
            if (must || (mbar_try_wait(b_full + 8 * s1, (g1 / kTcStages) & 1u) &&
                         mbar_try_wait(b_d1_empty + 8 * db, ((g1 >> 1) & 1u) ^ 1u))) {
              tc_fence_after();
              if (kAppend && new_row >= 0 && t1 == n_tiles - 1) {
                // a3 inside a4: the appended row goes on top of the stale bytes the tile brought for its slot (row
                // `new_row` of the K and of the V codes, 16-byte chunks in the 128-byte swizzle, and its two scales)
                const uint32_t st = smem0 + s1 * kTcStageBytes, sa = stash_smem + e * 272u;
                const uint32_t row = static_cast<uint32_t>(new_row);
#pragma unroll
                for (uint32_t c = 0; c < 8; ++c) {
                  sts128(st + row * 128 + ((c ^ (row & 7u)) << 4), lds128(sa + c * 16));
                  sts128(st + 16384 + row * 128 + ((c ^ (row & 7u)) << 4), lds128(sa + 128 + c * 16));
                }
                fence_proxy_async();                               // ... before the tensor core reads them
              }
              const uint64_t kdesc = tc_smem_desc(smem0 + s1 * kTcStageBytes);
#pragma unroll
              for (int k = 0; k < 4; ++k) tc_mma_f8(tmem + db * 16, kdesc + 2 * k, qdesc + 2 * k, kTcIdescQK, k > 0);
              tc_commit(b_d1_full + 8 * db);
              ++g1; ++t1;
              continue;
            }
          }
          const uint32_t s = g2 % kTcStages, pb = g2 & 1u;
          if (may1) {                                              // poll: weights of tile t2 / arrival of tile t1
            if (!mbar_try_wait(b_p_full + 8 * pb, (g2 >> 1) & 1u)) continue;
          } else {
            mbar_wait(b_p_full + 8 * pb, (g2 >> 1) & 1u);
          }
          tc_fence_after();
          const uint64_t vdesc = tc_smem_desc(smem0 + s * kTcStageBytes + 16384);
          if constexpr (kTcPByToken) {
            const uint64_t pdesc = tc_smem_desc_p(p_smem + pb * kTcPBytes);
#pragma unroll
            for (int k = 0; k < 4; ++k) tc_mma_f8(o_tmem, vdesc + 256 * k, pdesc + 32 * k, kTcIdescPVt, (t2 > 0 || k > 0) ? 1u : 0u);
          } else {
            const uint64_t pdesc = tc_smem_desc(p_smem + pb * kTcPBytes);
#pragma unroll
            for (int k = 0; k < 4; ++k) tc_mma_f8(o_tmem, vdesc + 256 * k, pdesc + 2 * k, kTcIdescPV, (t2 > 0 || k > 0) ? 1u : 0u);
          }
          tc_commit(b_empty + 8 * s);                              // the stage goes back to the producer
          tc_commit(b_p_free + 8 * pb);
          if (t2 == n_tiles - 1) tc_commit(b_o_full + 8 * e);
          ++g2; ++t2;
        }
      }
    }
  } else {
    // ===================================== softmax + epilogue =====================================
    pdl_wait();
    const int tid = threadIdx.x;                                   // token of a tile / d column of O^T
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
    uint32_t g = 0, u_seq = 0;                                     // tile and unit sequence numbers of this CTA
    uint32_t p_off[8];                                             // byte offset of (term 0, head, token tid) in a P buffer
#pragma unroll
    for (int hh = 0; hh < 8; ++hh) p_off[hh] = hh * 128 + (((tid >> 4) ^ hh) << 4) + (tid & 15);
    for (;; ++u_seq) {
      const int e = u_seq & 1;
      mbar_wait(b_u_full + 8 * e, (u_seq >> 1) & 1u);
      TcUnit U;
      {
        const uint32_t ua = misc + 256 + e * 64;
        const uint4 a = lds128(ua), b = lds128(ua + 16), c = lds128(ua + 32), d = lds128(ua + 48);
        U.n_tiles = static_cast<int32_t>(a.x); U.n_tokens = static_cast<int32_t>(a.y);
        U.batch_idx = static_cast<int32_t>(a.z); U.h = static_cast<int32_t>(a.w);
        U.pidx = static_cast<int32_t>(b.x); U.pbase = static_cast<int32_t>(b.y); U.n_chunks = static_cast<int32_t>(b.z);
        U.new_row = static_cast<int32_t>(b.w);
        U.qs[0] = __uint_as_float(c.x); U.qs[1] = __uint_as_float(c.y); U.qs[2] = __uint_as_float(c.z); U.qs[3] = __uint_as_float(c.w);
        U.qs[4] = __uint_as_float(d.x); U.qs[5] = __uint_as_float(d.y); U.qs[6] = __uint_as_float(d.z); U.qs[7] = __uint_as_float(d.w);
      }
      if (U.n_tiles == 0) break;
      const uint32_t o_tmem = tmem + 32 + e * 32 + lane_base;
      float m_ref[8], l[8];
#pragma unroll
      for (int hh = 0; hh < 8; ++hh) { m_ref[hh] = -INFINITY; l[hh] = 0.f; }

      for (int t = 0; t < U.n_tiles; ++t, ++g) {
        const uint32_t s = g % kTcStages, db = g & 1u, pb = g & 1u;
        const uint32_t st = smem0 + s * kTcStageBytes;
        mbar_wait(b_full + 8 * s, (g / kTcStages) & 1u);           // the tile's scales (and V rows, below) are readable
        float ks, vs;
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(ks), "=f"(vs) : "r"(st + 32768 + tid * 8) : "memory");
        if (kAppend && t == U.n_tiles - 1 && tid == U.new_row)       // the appended row's scales: the tile brought stale ones
          asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(ks), "=f"(vs) : "r"(stash_smem + e * 272u + 256u) : "memory");
        const bool valid = t * kTcTileTokens + tid < U.n_tokens;
        if (t == U.n_tiles - 1) {                                  // rows past the chunk's end: no stale V byte reaches GEMM2
          // the warp zeroes its invalid rows (a suffix of its 32) four rows per store: lane -> (row r + lane / 8, 16-byte
          // chunk lane % 8), 512 contiguous bytes per instruction (a thread zeroing its own 128-byte row is a 32-way
          // bank conflict: 0.94 M excess wavefronts per launch on config 3, ncu source page)
          const int first = max(U.n_tokens - t * kTcTileTokens, warp * 32);   // first invalid row of the tile, within this warp's
          const uint4 z = make_uint4(0u, 0u, 0u, 0u);
          for (int r = first & ~3; r < warp * 32 + 32; r += 4) {
            const int row = r + (lane >> 3);
            if (row >= first) sts128(st + 16384 + row * 128 + (lane & 7) * 16, z);
          }
        }
        mbar_wait(b_d1_full + 8 * db, (g >> 1) & 1u);
        tc_fence_after();
        float d1[16];
        tmem_ld16(tmem + db * 16 + lane_base, d1);
        tc_fence_before();
        mbar_arrive(b_d1_empty + 8 * db);

        const float lv = fast_log2(vs), iv = valid ? fast_rcp(vs) : 0.f;
        float sc[8];
        bool over = false;
#pragma unroll
        for (int hh = 0; hh < 8; ++hh) {
          const float x = (d1[hh] + d1[8 + hh]) * (ks * U.qs[hh]) + lv;
          sc[hh] = valid ? x : -INFINITY;                           // masked by index, never by value
          over |= sc[hh] > m_ref[hh] + kTcLazyLog2;
        }
        const uint32_t par = g & 1u;
        const bool warp_over = __any_sync(kFull, over);
        if (warp_over) {                                           // rare: publish this warp's maxima
#pragma unroll
          for (int hh = 0; hh < 8; ++hh) {
            float mx = sc[hh];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, off));
            if (lane == 0) sts32(wmax_smem + ((par * 4 + warp) * 8 + hh) * 4, __float_as_uint(mx));
          }
        }
        if (lane == 0) sts32(flags_smem + (par * 4 + warp) * 4, warp_over ? 1u : 0u);
        softmax_barrier();
        const uint4 fl = lds128(flags_smem + par * 16);
        if (fl.x | fl.y | fl.z | fl.w) {
          // ---- the reference moves: m_new = max(m_ref, published maxima); O^T and l follow ----
          float alpha[8];
#pragma unroll
          for (int hh = 0; hh < 8; ++hh) {
            float mn = m_ref[hh];
#pragma unroll
            for (int w = 0; w < 4; ++w)
              if (u4_get(fl, w)) mn = fmaxf(mn, __uint_as_float(lds32(wmax_smem + ((par * 4 + w) * 8 + hh) * 4)));
            alpha[hh] = m_ref[hh] == -INFINITY ? 0.f : fast_exp2(m_ref[hh] - mn);
            l[hh] *= alpha[hh];
            m_ref[hh] = mn;
          }
          if (t > 0) {                                             // GEMM2 of the previous tile has to be in O^T first
            mbar_wait(b_p_free + 8 * ((g - 1) & 1u), ((g - 1) >> 1) & 1u);
            tc_fence_after();
            float o[32];
            tmem_ld32(o_tmem, o);
#pragma unroll
            for (int c = 0; c < 32; ++c) o[c] *= alpha[c & 7];
            tmem_st32(o_tmem, o);
            tc_fence_before();
          }
        }
        // ---- weights: f16, split exactly into four e5m2 terms; bytes P^T[term][head][token] ----
        if (g >= 2) mbar_wait(b_p_free + 8 * pb, ((g >> 1) - 1) & 1u);   // GEMM2 of tile g - 2 has read this buffer
        const uint32_t pbuf = p_smem + pb * kTcPBytes;
        if constexpr (kTcPByToken) {
          uint32_t x[4], wt[8];                                     // x[j]: f16 weights of heads 2j, 2j+1; wt: [term][head] bytes
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float p0 = fast_exp2(sc[2 * j] - m_ref[2 * j] + kTcWeightBias), p1 = fast_exp2(sc[2 * j + 1] - m_ref[2 * j + 1] + kTcWeightBias);
            l[2 * j] += p0 * iv;
            l[2 * j + 1] += p1 * iv;
            x[j] = pack_f16x2(p0, p1);
          }
#pragma unroll
          for (int term = 0; term < 4; ++term) {
            wt[2 * term] = __byte_perm(x[0], x[1], 0x7531);         // the top bytes (e5m2 terms) of heads 0..3
            wt[2 * term + 1] = __byte_perm(x[2], x[3], 0x7531);     //                          ... of heads 4..7
            if (term < 3) {
#pragma unroll
              for (int j = 0; j < 4; ++j) {
                const uint32_t top = x[j] & 0xff00ff00u;
                const __half2 r = __hsub2(*reinterpret_cast<const __half2*>(&x[j]), *reinterpret_cast<const __half2*>(&top));
                x[j] = *reinterpret_cast<const uint32_t*>(&r);
              }
            }
          }
          const uint32_t prow = pbuf + (tid >> 3) * 128 + (tid & 7) * 16;
          sts128(prow, make_uint4(wt[0], wt[1], wt[2], wt[3]));          // N = 0..15: terms 0, 1
          sts128(prow + 2048, make_uint4(wt[4], wt[5], wt[6], wt[7]));   // N = 16..31: terms 2, 3
        } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float p0 = fast_exp2(sc[2 * j] - m_ref[2 * j] + kTcWeightBias), p1 = fast_exp2(sc[2 * j + 1] - m_ref[2 * j + 1] + kTcWeightBias);
          l[2 * j] += p0 * iv;
          l[2 * j + 1] += p1 * iv;
          uint32_t x = pack_f16x2(p0, p1);
#pragma unroll
          for (int term = 0; term < 4; ++term) {
            const uint32_t top = x & 0xff00ff00u;
            sts8(pbuf + term * 1024 + p_off[2 * j], top >> 8);
            sts8(pbuf + term * 1024 + p_off[2 * j + 1], top >> 24);
            if (term < 3) {
              const __half2 r = __hsub2(*reinterpret_cast<const __half2*>(&x), *reinterpret_cast<const __half2*>(&top));
              x = *reinterpret_cast<const uint32_t*>(&r);
            }
          }
        }
        }
        fence_proxy_async();                                       // P^T (and zeroed V rows) -> visible to the tensor core
        mbar_arrive(b_p_full + 8 * pb);
      }

      // ---- epilogue: l over the 128 tokens lanes, O^T out of TMEM, store / partial + fused merge (a5) ----
#pragma unroll
      for (int hh = 0; hh < 8; ++hh) {
        float x = l[hh];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(kFull, x, off);
        if (lane == 0) sts32(lsum_smem + (warp * 8 + hh) * 4, __float_as_uint(x));
      }
      softmax_barrier();
#pragma unroll
      for (int hh = 0; hh < 8; ++hh) {
        float x = 0.f;
#pragma unroll
        for (int w = 0; w < 4; ++w) x += __uint_as_float(lds32(lsum_smem + (w * 8 + hh) * 4));
        l[hh] = x;
      }
      mbar_wait(b_o_full + 8 * e, (u_seq >> 1) & 1u);
      tc_fence_after();
      float o[32];
      tmem_ld32(o_tmem, o);
      tc_fence_before();
      mbar_arrive(b_o_empty + 8 * e);
      const int64_t out_row0 = static_cast<int64_t>(U.batch_idx) * p.num_q_heads + U.h * G;
      if (U.pidx < 0) {
#pragma unroll
        for (int hh = 0; hh < 8; ++hh)
          if (hh < G) {
            const float v = (o[hh] + o[8 + hh] + o[16 + hh] + o[24 + hh]) / l[hh];
            p.out[(out_row0 + hh) * D + tid] = static_cast<uint16_t>(pack_bf16x2(v, 0.f) & 0xffffu);
          }
      } else {
#pragma unroll
        for (int hh = 0; hh < 8; ++hh)
          if (hh < G) {
            p.part_o[(static_cast<int64_t>(U.pidx) * G + hh) * D + tid] = o[hh] + o[8 + hh] + o[16 + hh] + o[24 + hh];
            if (tid == hh) *reinterpret_cast<float2*>(p.part_ml + (static_cast<int64_t>(U.pidx) * G + hh) * 2) = make_float2(m_ref[hh], l[hh]);
          }
        if (p.fuse_combine) {                                      // the unit that completes its (request, kv head) merges
          __threadfence();
          softmax_barrier();
          if (tid == 0) {
            const int last = atomicAdd(&p.arrive[U.pbase], 1) == U.n_chunks - 1;
            if (last) p.arrive[U.pbase] = 0;
            sts32(merge_flag, static_cast<uint32_t>(last));
          }
          softmax_barrier();
          if (lds32(merge_flag)) {
            __threadfence();
            for (int hh = warp; hh < G; hh += 4)
              combine_heads<D, 1>(p.part_o, p.part_ml, U.pbase, U.n_chunks, G, hh, p.out + (out_row0 + hh) * D, lane);
          }
        }
      }
      softmax_barrier();                                           // lsum / merge_flag are free again; the unit is done
      mbar_arrive(b_u_empty + 8 * e);
    }
  }

  // ---- tear-down ----
  tc_fence_before();
  __syncthreads();
  if (warp == 5) {
    tc_fence_after();
    tmem_dealloc(tmem, kTcTmemCols);
  }
  // Last CTA out rewinds the work counter for the next launch (as attn_kernel does).
  if (threadIdx.x == 0) {
    const unsigned prev = atomicInc(reinterpret_cast<unsigned*>(&p.counters[1]), gridDim.x - 1);
    if (prev == gridDim.x - 1) p.counters[0] = 0;
  }
}

}  // namespace kvp
