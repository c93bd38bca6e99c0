// kv_common.cuh — what every sm_100a kernel of the D-instance KV path shares: geometry constants, small PTX
// wrappers, the launch-parameter structs (their layouts are also written by the host serialisers in kv_pool.cu)
// and the log-sum-exp merge of split-KV partials (a5), which runs both inside the attention kernel (last-arriver
// merge) and as the stand-alone combine_kernel.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace kvp {

constexpr int kBlockSize = 16;     // tokens per KV block (BASELINE.json: block size 16)
constexpr int kAttnThreads = 128;  // 4 warps per CTA, each an independent split-KV worker
constexpr int kAttnWarps = kAttnThreads / 32;
constexpr unsigned kFull = 0xffffffffu;

// bytes of one (layer, block, kv head) tile: bf16 K[16][D] | V[16][D];  FP8 K8[16][D] | V8[16][D] | sc[16]{ks, vs} fp32
template <int D>
__host__ __device__ constexpr int64_t bf16_tile_bytes() { return 2 * kBlockSize * D * 2; }
template <int D>
__host__ __device__ constexpr int64_t fp8_tile_bytes() { return 32 * D + 128; }

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

__device__ __forceinline__ uint2 ldg_copy8_pred(const void* ptr, bool pred) {
  uint2 r = make_uint2(0u, 0u);
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\t"
      "@p ld.global.L1::no_allocate.v2.u32 {%0, %1}, [%2];\n\t}"
      : "+r"(r.x), "+r"(r.y)
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

__device__ __forceinline__ void stg_stream8_pred(void* ptr, const uint2& v, bool pred) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %3, 0;\n\t"
      "@p st.global.L1::no_allocate.v2.u32 [%0], {%1, %2};\n\t}"
      :
      : "l"(ptr), "r"(v.x), "r"(v.y), "r"(static_cast<int>(pred))
      : "memory");
}

__device__ __forceinline__ uint4 lds128(uint32_t smem_addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(smem_addr));
  return r;
}

// 16-byte cp.async (SASS LDGSTS), L2 only; bytes past src_bytes (0 or 16 here) are zero-filled
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gptr), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- TMA (cp.async.bulk.tensor, SASS UTMALDG) + mbarrier --------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
// make freshly initialised barriers visible to the async proxy (the TMA unit completes transactions on them)
__device__ __forceinline__ void mbar_init_fence() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// order this thread's earlier generic-proxy accesses to shared memory before later async-proxy (TMA) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// 2-D tiled tensor copy global -> shared; completion (bytes) is signalled on `bar`.  `tmap` is the generic address of a
// CUtensorMap living in kernel parameter space (__grid_constant__).
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void* tmap, uint32_t bar, int32_t c0, int32_t c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar), "r"(c0), "r"(c1) : "memory");
}

// 1-D bulk copy global -> shared (SASS UBLKCP), 16-byte aligned, size a multiple of 16; completion on `bar`
__device__ __forceinline__ void bulk_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// Programmatic dependent launch (PDL).  wait: block until every grid this launch depends on has completed and its
// memory is visible (a no-op for a launch without the programmatic attribute).  launch_dependents: allow the next
// launch of the stream, if it carries the attribute, to start its CTAs as SM resources free up.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// D(16x8, f32) += A(16x16, bf16, row) * B(16x8, bf16, col)
__device__ __forceinline__ void mma_bf16_m16n8k16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                                  uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
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

__device__ __forceinline__ uint32_t pack_f16x2(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// 1 / x to ~1 ulp, subnormal inputs handled (not flushed)
__device__ __forceinline__ float fast_rcp(float x) {
  float y;
  asm("rcp.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ float fast_log2(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// (a.lo16, b.lo16) / (a.hi16, b.hi16): pair up one bf16 from each of two registers
__device__ __forceinline__ uint32_t pair_lo(uint32_t a, uint32_t b) { return __byte_perm(a, b, 0x5410); }
__device__ __forceinline__ uint32_t pair_hi(uint32_t a, uint32_t b) { return __byte_perm(a, b, 0x7632); }

__device__ __forceinline__ uint32_t u4_get(const uint4& v, int i) {
  return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w));
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

// max |x| over the 8 bf16 of a 16-byte piece, as a bf16 bit pattern (bf16 magnitudes order like unsigned integers)
__device__ __forceinline__ uint32_t amax_bits8(const uint4& x) {
  const uint32_t m = __vmaxu2(__vmaxu2(x.x & 0x7fff7fffu, x.y & 0x7fff7fffu), __vmaxu2(x.z & 0x7fff7fffu, x.w & 0x7fff7fffu));
  return max(m & 0xffffu, m >> 16);
}

// The FP8 pool's quantisation of one 16-byte piece of a row whose |max| has bf16 bits `mx` (C1-C4; every
// rounding in fp32, decided the same way by the oracle): scale = fl32(amax / 448), inv = fl32(448 / amax) (1 if
// amax = 0), code = RNE_e4m3_satfinite(fl32(x * inv)).  Returns the 8 codes; *scale receives the row scale.
__device__ __forceinline__ uint2 quantise_piece(const uint4& x, uint32_t mx, float* scale) {
  const float amax = __uint_as_float(mx << 16);
  *scale = mx == 0 ? 1.f : __fdiv_rn(amax, 448.f);
  const float inv = mx == 0 ? 1.f : __fdiv_rn(448.f, amax);
  uint32_t w[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint32_t e = u4_get(x, k);
    w[k] = f32x2_to_e4m3x2(__fmul_rn(__uint_as_float(e << 16), inv), __fmul_rn(__uint_as_float(e & 0xffff0000u), inv));
  }
  return make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
}

// ---------------------------------------------------------------------------------------------
// launch parameters
// ---------------------------------------------------------------------------------------------

// One request of an ingest / gather / transfer launch.  Units of request i are
// [unit_begin, unit_begin + n_touched * layer_count * Hkv), ordered (layer, head, touched block)
// with the touched block fastest, so consecutive warps stream consecutive source runs.
struct IngestReq {
  uint64_t k_src, v_src;  // device addresses of the contiguous [layer_count][Hkv][n_tokens][D] tensors (transfer: unused)
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
  uint16_t* kv;              // KV region base (the pool written by ingest / transfer, read by gather)
  int32_t* block_table;      // device mirror [max_requests][bt_stride]
  int32_t bt_stride;
  int32_t layer_begin, layer_count, num_kv_heads;
  int64_t num_blocks;
  // KV-head sharding: the contiguous side is [layer_count][src_kv_heads][n][D] and this
  // pool's head h is its head src_head_begin + h.  Unsharded: src_kv_heads = num_kv_heads, src_head_begin = 0.
  int32_t src_kv_heads, src_head_begin;
  // transfer (NEXT-4): the producer pool's KV region and block count; request i's producer block ids follow its
  // consumer block ids in blk_ids (at blk_off + n_touched)
  const uint16_t* src_kv;
  int64_t src_num_blocks;
};

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
  int32_t chained;             // 1: the stream's previous kernel is an attention launch of the same plan, so work items,
                               //    block ids and this layer's KV may be read before griddepcontrol.wait
  float scale_log2;            // sm_scale * log2(e)
  int64_t tma_row0;            // TMA variants: first 128-byte row of this layer's KV inside the tensor map
  alignas(64) unsigned char tmap[128];   // CUtensorMap over the KV region as [rows][128 B] (TMA variants; else unused)
};

// ---------------------------------------------------------------------------------------------
// a5: log-sum-exp merge of split-KV partials
// ---------------------------------------------------------------------------------------------

// Query heads [head0, head0 + NH) of one (request, kv head): out = sum_c 2^(m_c - M) O_c / sum_c 2^(m_c - M) l_c
// over the n_chunks partials starting at partial slot pb (one slot per chunk).  One warp; lane owns D/32 columns of
// every head.  The merge is a running (online) one so the loads of all heads and of several chunks are independent
// and in flight together — this code is pure latency, it runs on warps that would otherwise be streaming KV.  Loads
// bypass L1 (.cg): the partials were written by other SMs, possibly earlier in this same kernel.
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
      const float mn = fmaxf(M[hh], mlv[hh].x);                 // finite: chunk 0 is merged first and holds token 0
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

// Plan upload as a KERNEL (pinned host staging, read in place over PCIe -> the plan slot in the slab), so that the
// stream holds only kernels and programmatic dependent launch chains straight through a decode step's boundary: its
// copy overlaps the tail of the previous attention launch (a different plan slot), and it completes only after that
// launch has (griddepcontrol.wait), so the attention launch behind it inherits the ordering.
__global__ void __launch_bounds__(256) plan_upload_kernel(const uint4* __restrict__ host_src, uint4* __restrict__ dst, int n16) {
  pdl_launch_dependents();
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += gridDim.x * blockDim.x) dst[i] = host_src[i];
  pdl_wait();
}

struct CombineEntryDev { int32_t batch_idx, partial_begin, n_chunks, pad; };  // == kvp::CombineEntry

struct CombineParams {
  const CombineEntryDev* entries;
  int32_t n_entries;
  const float* part_o;
  const float* part_ml;
  uint16_t* out;
  int32_t num_q_heads, num_kv_heads, group;
};

// a5 stand-alone (option fuse_combine = 0): one warp per (combine entry, head of the group)
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
