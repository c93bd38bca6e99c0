/*
 * kv_oracle.c — the ORACLE: a plain, slow, fp64 CPU statement of what the D-instance KV
 * path computes.  TEST INFRASTRUCTURE ONLY: nothing outside tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it, and it shares no code,
 * header, table or helper with paper_2511_20982_b200/ (the CUDA path).
 *
 * What it states (citations are /root/reference/PAPER.md lines):
 *   - oracle_attention: PAPER.md:146 (§IV-A, Eq. 1) Output = softmax(Q K^T) V, in the decode
 *     form of PAPER.md:200 / :219 (one query token per in-flight request over that request's
 *     stored KV).  Readings: A1 the omitted 1/sqrt(d) scale is an
 *     explicit argument; A2 query head h reads KV head h / G; A3/A4 all n stored tokens are
 *     visible, no mask.  This is the DEFINITION written out: the CUDA path's paging,
 *     split-KV, online softmax and LSE combine reach the same value (up to rounding), so
 *     none of that appears here.
 *   - oracle_scatter / oracle_gather: the relocation of a prefill-completed request's
 *     contiguous KV ("prefill-completed requests (together with KV-cache)")
 *     into the consumer's KV-cache blocks, and its inverse.  Pure bit copies.
 *   - oracle_chunk / oracle_combine: the per-chunk (m, l, O) triple and the log-sum-exp
 *     merge, in fp64, so that tests can pin the merge identity.  Not used
 *     by oracle_attention.
 *
 * Slab layout is the one include/kv_pool.h documents for the caller-owned slab, restated
 * here independently (kv_index).  bf16 inputs are widened exactly: a bf16 is the top 16 bits
 * of an IEEE float.  Sums are plain left-to-right loops in double.
 *
 * Parity pins (tests/test_oracle_pins.py): n = 1 returns V_0; q = 0 gives the mean of V;
 * hand-computed weights (1/3, 2/3), (1/7, 2/7, 4/7), (1/6, 2/6, 3/6); weights sum to 1;
 * block-permutation invariance; GQA map; shift invariance / no overflow; agreement with
 * torch.nn.functional.scaled_dot_product_attention in fp64; an independent numpy
 * brute-force over gathered rows; chunk+combine == unsplit; scatter o gather == identity and
 * whole-slab equality with a numpy fancy-index scatter.  oracle_attention_varq
 * (tests/test_oracle_varq_pins.py): q_len = 1 equals oracle_attention; full and chunked
 * prefill equal torch SDPA with a causal (lower-right aligned) mask in fp64; first token of
 * a fresh prefill returns V_0; q = 0 gives running means; each query row equals decode over
 * the truncated sequence; future tokens do not matter.  oracle_capacity / oracle_pd_ratio
 * (tests/test_capacity_model.py): exact-fraction hand values; Eq. 14 with Table I's printed T_p
 * and T_d brackets the printed optimum 4.58.  FP8 functions
 * (tests/test_oracle_fp8_pins.py): the e4m3 decode table and the RNE encoder equal
 * torch.float8_e4m3fn on every code, every midpoint and a dense random sweep; the quantising
 * scatter equals an independent numpy/torch-float8 statement over the whole slab, a brute-force
 * nearest-code search and the |x - x^| <= 16 scale bound; attention over an FP8 pool equals
 * oracle_attention when the data is exactly representable and torch SDPA (fp64) on the
 * dequantised values otherwise; oracle_attention_varq_fp8 equals oracle_attention_fp8 at q_len = 1,
 * oracle_attention_varq on exactly representable rows and torch SDPA (causal, fp64) on the
 * dequantised values.  NEXT-4 functions (tests/test_oracle_transfer_pins.py): oracle_transfer into a
 * sentinel-filled pool B equals oracle_scatter of the ORIGINAL source through B's block list over the
 * whole slab (and an independent numpy fancy-index statement), A is untouched, slots past the
 * request's end keep the sentinel, gather(B) returns the source; oracle_transfer_fp8 likewise against
 * oracle_scatter_fp8 and a numpy byte-view statement; oracle_gather_fp8's codes x scales equal
 * oracle_dequant_fp8 and a numpy index statement of the tile layout.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif
#include <stdlib.h>
#include <string.h>

typedef struct {
  int32_t num_layers, num_kv_heads, head_dim, block_size;
  int64_t num_blocks;
} oracle_dims_t;

static double bf16_to_double(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return (double)f;
}

/* element index of kv[layer][block][kv_head][c][slot][j] (include/kv_pool.h, "Slab layout") */
static int64_t kv_index(const oracle_dims_t* D, int64_t layer, int64_t block, int64_t head,
                        int64_t c, int64_t slot, int64_t j) {
  return ((((layer * D->num_blocks + block) * D->num_kv_heads + head) * 2 + c) * D->block_size +
          slot) * D->head_dim + j;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/*
 * Reference scatter.  blocks[] is the request's block list (logical
 * block i -> physical id).  Copies tokens t in [0,n) of src (layout
 * [layer_count][num_kv_heads][n][head_dim]) to logical positions start_pos + t of layers
 * layer_begin .. layer_begin+layer_count-1.
 */
void oracle_scatter(uint16_t* kv, const oracle_dims_t* D, const int32_t* blocks,
                    int32_t start_pos, int32_t n, const uint16_t* k_src, const uint16_t* v_src,
                    int32_t layer_begin, int32_t layer_count) {
  for (int32_t ll = 0; ll < layer_count; ++ll)
    for (int32_t h = 0; h < D->num_kv_heads; ++h)
      for (int32_t t = 0; t < n; ++t) {
        int32_t pos = start_pos + t;
        int32_t blk = blocks[pos / D->block_size];
        int32_t slot = pos % D->block_size;
        int64_t s = (((int64_t)ll * D->num_kv_heads + h) * n + t) * D->head_dim;
        for (int32_t j = 0; j < D->head_dim; ++j) {
          kv[kv_index(D, layer_begin + ll, blk, h, 0, slot, j)] = k_src[s + j];
          kv[kv_index(D, layer_begin + ll, blk, h, 1, slot, j)] = v_src[s + j];
        }
      }
}

/* Reference gather: inverse of oracle_scatter over tokens [0,len), all layers.
 * k_dst / v_dst: [num_layers][num_kv_heads][len][head_dim]. */
void oracle_gather(const uint16_t* kv, const oracle_dims_t* D, const int32_t* blocks, int32_t len,
                   uint16_t* k_dst, uint16_t* v_dst) {
  for (int32_t l = 0; l < D->num_layers; ++l)
    for (int32_t h = 0; h < D->num_kv_heads; ++h)
      for (int32_t t = 0; t < len; ++t) {
        int32_t blk = blocks[t / D->block_size];
        int32_t slot = t % D->block_size;
        int64_t s = (((int64_t)l * D->num_kv_heads + h) * len + t) * D->head_dim;
        for (int32_t j = 0; j < D->head_dim; ++j) {
          k_dst[s + j] = kv[kv_index(D, l, blk, h, 0, slot, j)];
          v_dst[s + j] = kv[kv_index(D, l, blk, h, 1, slot, j)];
        }
      }
}

/*
 * Decode attention, the definition:
 *   for request r, query head h:  g = h / G;  n = seq_lens[r]
 *     s_t = scale * sum_j q[r][h][j] * K_t[j]        t in [0,n)
 *     m = max_t s_t;  w_t = exp(s_t - m);  Z = sum_t w_t
 *     out[r][h][:] = sum_t (w_t / Z) * V_t[:]         (fp64, not rounded)
 * Block lists are ragged: request r's list is bt[bt_off[r] .. bt_off[r+1]).
 * wsum (optional, may be NULL): wsum[r*Hq+h] = sum_t (w_t / Z), for the sum-to-1 invariant.
 * Returns 0, or -1 if some request has n < 1 (empty context is an error).
 */
int oracle_attention(const uint16_t* kv, const oracle_dims_t* D, int32_t layer, int32_t num_q_heads,
                     int32_t batch, const int32_t* bt, const int64_t* bt_off,
                     const int32_t* seq_lens, const uint16_t* q, double scale, double* out,
                     double* wsum) {
  const int32_t d = D->head_dim, Hq = num_q_heads, G = num_q_heads / D->num_kv_heads;
  for (int32_t r = 0; r < batch; ++r)
    if (seq_lens[r] < 1) return -1;
  int bad = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int32_t r = 0; r < batch; ++r)
    for (int32_t h = 0; h < Hq; ++h) {
      const int32_t g = h / G, n = seq_lens[r];
      const int32_t* blocks = bt + bt_off[r];
      const uint16_t* qv = q + ((int64_t)r * Hq + h) * d;
      double* s = (double*)malloc(sizeof(double) * (size_t)n);
      double* o = out + ((int64_t)r * Hq + h) * d;
      if (!s) { bad = 1; continue; }
      for (int32_t t = 0; t < n; ++t) {
        int64_t kb = kv_index(D, layer, blocks[t / D->block_size], g, 0, t % D->block_size, 0);
        double acc = 0.0;
        for (int32_t j = 0; j < d; ++j) acc += bf16_to_double(qv[j]) * bf16_to_double(kv[kb + j]);
        s[t] = scale * acc;
      }
      double m = s[0];
      for (int32_t t = 1; t < n; ++t)
        if (s[t] > m) m = s[t];
      double Z = 0.0;
      for (int32_t t = 0; t < n; ++t) {
        s[t] = exp(s[t] - m);
        Z += s[t];
      }
      for (int32_t j = 0; j < d; ++j) o[j] = 0.0;
      double ws = 0.0;
      for (int32_t t = 0; t < n; ++t) {
        int64_t vb = kv_index(D, layer, blocks[t / D->block_size], g, 1, t % D->block_size, 0);
        double w = s[t] / Z;
        ws += w;
        for (int32_t j = 0; j < d; ++j) o[j] += w * bf16_to_double(kv[vb + j]);
      }
      if (wsum) wsum[(int64_t)r * Hq + h] = ws;
      free(s);
    }
  return bad ? -2 : 0;
}

/*
 * Variable-q-length causal attention.  PAPER.md:443 (§V-E): "For
 * ultra-short requests we employ PD-aggregation: merging their prefill with other requests'
 * decoding on D-instances"; PAPER.md:94 (§II): such requests are executed "in-place (i.e.,
 * without remote prefill)".  So one batch holds decode rows (one query token) and in-place
 * prefill rows (q_len query tokens); Eq. 1 applies with Q = the LAST q_lens[r]
 * tokens of request r.  Readings (B1-B3): the mask is causal — query token i, at
 * absolute position P_i = seq_lens[r] - q_lens[r] + i, sees stored tokens 0..P_i inclusive (its
 * own K/V is already in the pool); q_lens[r] = 1 is exactly oracle_attention's decode row.
 *   q, out: [total_q][num_q_heads][head_dim], request r's rows start at q_off[r]
 *   (q_off[batch] = total_q).  out is fp64, not rounded.  wsum optional as in oracle_attention.
 * Returns 0; -1 if some request has q_lens[r] < 1 or q_lens[r] > seq_lens[r]; -2 out of memory.
 */
int oracle_attention_varq(const uint16_t* kv, const oracle_dims_t* D, int32_t layer,
                          int32_t num_q_heads, int32_t batch, const int32_t* bt,
                          const int64_t* bt_off, const int32_t* seq_lens, const int32_t* q_lens,
                          const int64_t* q_off, const uint16_t* q, double scale, double* out,
                          double* wsum) {
  const int32_t d = D->head_dim, Hq = num_q_heads, G = num_q_heads / D->num_kv_heads;
  for (int32_t r = 0; r < batch; ++r)
    if (q_lens[r] < 1 || q_lens[r] > seq_lens[r]) return -1;
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t r = 0; r < batch; ++r) {
    const int32_t* blocks = bt + bt_off[r];
    double* s = (double*)malloc(sizeof(double) * (size_t)seq_lens[r]);
    if (!s) { bad = 1; continue; }
    for (int32_t i = 0; i < q_lens[r]; ++i) {
      const int32_t n = seq_lens[r] - q_lens[r] + i + 1;   /* tokens 0 .. P_i visible */
      for (int32_t h = 0; h < Hq; ++h) {
        const int32_t g = h / G;
        const uint16_t* qv = q + ((q_off[r] + i) * Hq + h) * d;
        double* o = out + ((q_off[r] + i) * Hq + h) * d;
        for (int32_t t = 0; t < n; ++t) {
          int64_t kb = kv_index(D, layer, blocks[t / D->block_size], g, 0, t % D->block_size, 0);
          double acc = 0.0;
          for (int32_t j = 0; j < d; ++j) acc += bf16_to_double(qv[j]) * bf16_to_double(kv[kb + j]);
          s[t] = scale * acc;
        }
        double m = s[0];
        for (int32_t t = 1; t < n; ++t)
          if (s[t] > m) m = s[t];
        double Z = 0.0;
        for (int32_t t = 0; t < n; ++t) {
          s[t] = exp(s[t] - m);
          Z += s[t];
        }
        for (int32_t j = 0; j < d; ++j) o[j] = 0.0;
        double ws = 0.0;
        for (int32_t t = 0; t < n; ++t) {
          int64_t vb = kv_index(D, layer, blocks[t / D->block_size], g, 1, t % D->block_size, 0);
          double w = s[t] / Z;
          ws += w;
          for (int32_t j = 0; j < d; ++j) o[j] += w * bf16_to_double(kv[vb + j]);
        }
        if (wsum) wsum[(q_off[r] + i) * Hq + h] = ws;
      }
    }
    free(s);
  }
  return bad ? -2 : 0;
}

/*
 * D-instance capacity model, the formulas as printed:
 *   PAPER.md:206 Eq. 11  V_mem = (M_gpu - M') x TP - M_model
 *   PAPER.md:212 Eq. 12  V_BW  = t_d^SLO x alpha x TP x BW
 *   PAPER.md:216 Eq. 13  cc_d  = min(V_mem, V_BW) / ((ISL + OSL/2) x M_token)
 * out[0..2] = V_mem, V_BW, cc_d (cc_d = 0 if the smaller volume is not positive).
 */
void oracle_capacity(double M_gpu, double M_prime, double M_model, double TP, double BW, double alpha,
                     double t_d_slo, double ISL, double OSL, double M_token, double* out) {
  double V_mem = (M_gpu - M_prime) * TP - M_model;
  double V_BW = t_d_slo * alpha * TP * BW;
  double V = V_mem < V_BW ? V_mem : V_BW;
  out[0] = V_mem;
  out[1] = V_BW;
  out[2] = V > 0.0 ? V / ((ISL + OSL / 2.0) * M_token) : 0.0;
}

/* PAPER.md:223 Eq. 14  n_p x (t_d x OSL / t_p) = n_d x cc_d, solved for n_p / n_d (the closed form
 * announced at PAPER.md:225 is missing from the extraction; reading A10). */
double oracle_pd_ratio(double cc_d, double t_p, double t_d, double OSL) {
  double per_p = t_d * OSL / t_p; /* concurrency one P-instance can drive on a D-instance */
  return cc_d / per_p;
}

/*
 * One split-KV chunk in fp64: over tokens [t0, t1) of one request and
 * one query head,  m = max s_t,  l = sum exp(s_t - m),  O = sum exp(s_t - m) V_t.
 */
void oracle_chunk(const uint16_t* kv, const oracle_dims_t* D, int32_t layer, int32_t kv_head,
                  const int32_t* blocks, int32_t t0, int32_t t1, const uint16_t* qv, double scale,
                  double* m_out, double* l_out, double* O_out) {
  const int32_t d = D->head_dim;
  double m = -INFINITY;
  for (int32_t t = t0; t < t1; ++t) {
    int64_t kb = kv_index(D, layer, blocks[t / D->block_size], kv_head, 0, t % D->block_size, 0);
    double acc = 0.0;
    for (int32_t j = 0; j < d; ++j) acc += bf16_to_double(qv[j]) * bf16_to_double(kv[kb + j]);
    if (scale * acc > m) m = scale * acc;
  }
  double l = 0.0;
  for (int32_t j = 0; j < d; ++j) O_out[j] = 0.0;
  for (int32_t t = t0; t < t1; ++t) {
    int64_t kb = kv_index(D, layer, blocks[t / D->block_size], kv_head, 0, t % D->block_size, 0);
    int64_t vb = kv_index(D, layer, blocks[t / D->block_size], kv_head, 1, t % D->block_size, 0);
    double acc = 0.0;
    for (int32_t j = 0; j < d; ++j) acc += bf16_to_double(qv[j]) * bf16_to_double(kv[kb + j]);
    double w = exp(scale * acc - m);
    l += w;
    for (int32_t j = 0; j < d; ++j) O_out[j] += w * bf16_to_double(kv[vb + j]);
  }
  *m_out = m;
  *l_out = l;
}

/* LSE combine:  M = max_c m_c;  out = sum_c e^{m_c-M} O_c / sum_c e^{m_c-M} l_c */
void oracle_combine(int32_t n_chunks, int32_t d, const double* m, const double* l, const double* O,
                    double* out) {
  double M = m[0];
  for (int32_t c = 1; c < n_chunks; ++c)
    if (m[c] > M) M = m[c];
  double den = 0.0;
  for (int32_t j = 0; j < d; ++j) out[j] = 0.0;
  for (int32_t c = 0; c < n_chunks; ++c) {
    double a = exp(m[c] - M);
    den += a * l[c];
    for (int32_t j = 0; j < d; ++j) out[j] += a * O[(int64_t)c * d + j];
  }
  for (int32_t j = 0; j < d; ++j) out[j] /= den;
}

/* =============================================================================================
 * NEXT-2: FP8 (e4m3) KV pool.  The paper's models are FP8 and
 * the KV bytes per token M_token are the denominator of Eq. 13: halving them doubles
 * cc_d under both Eq. 11 and Eq. 12.  The paper fixes no KV quantisation; the reading taken
 * (C1-C4) is stated here step by step, in the precision both sides use (fp32 for the
 * two roundings that decide a code):
 *   per token row x[0..d) of one (layer, kv head, K|V):
 *     amax  = max_j |x_j|                          (exact: bf16 magnitudes)
 *     scale = amax == 0 ? 1 : fl32(amax / 448)     stored beside the row, fp32
 *     inv   = amax == 0 ? 1 : fl32(448 / amax)
 *     code_j = RNE_e4m3( fl32(x_j * inv) )         e4m3 "fn": 1-4-3 bits, bias 7, no infinities,
 *                                                  S.1111.111 = NaN, max finite 448; saturating
 *   dequantised value  x^_j = e4m3(code_j) * scale  (exact in fp64)
 * Attention over an FP8 pool is Eq. 1 on the dequantised values (oracle_attention_fp8, fp64).
 *
 * FP8 slab layout (restated independently from include/kv_pool.h): per (layer, block, kv head) one
 * tile of 32 d + 128 bytes:  K8[16][d] codes | V8[16][d] codes | sc[16][2] fp32 (ks_t, vs_t);
 * tiles ordered [layer][block][kv_head].
 * ============================================================================================= */

static double e4m3_decode(uint8_t c) {
  int sign = c >> 7, e = (c >> 3) & 15, m = c & 7;
  double v;
  if (e == 15 && m == 7) return NAN;
  if (e == 0) v = ldexp((double)m, -9);            /* subnormal: m/8 * 2^-6 */
  else v = ldexp(1.0 + m / 8.0, e - 7);
  return sign ? -v : v;
}

void oracle_e4m3_decode_table(double* out256) {
  for (int c = 0; c < 256; ++c) out256[c] = e4m3_decode((uint8_t)c);
}

/* Round-to-nearest-even onto the e4m3 grid, saturating at +-448; NaN -> 0x7f. */
uint8_t oracle_e4m3_encode(float yf) {
  double y = (double)yf;
  if (y != y) return 0x7f;
  uint8_t sign = (uint8_t)(signbit(y) ? 0x80 : 0);
  double a = fabs(y);
  if (a >= 448.0) return (uint8_t)(sign | 0x7e);   /* satfinite (also covers inf) */
  int e;
  (void)frexp(a, &e);                               /* a = f * 2^e, f in [0.5, 1)  ->  floor(log2 a) = e - 1 */
  int ex = a == 0.0 ? -6 : e - 1;
  if (ex < -6) ex = -6;                             /* subnormal range shares the quantum of 2^-6 */
  double quantum = ldexp(1.0, ex - 3);              /* spacing of the grid in [2^ex, 2^(ex+1)) */
  double n = nearbyint(a / quantum);                /* exact division by a power of two; ties to even */
  double r = n * quantum;                           /* may round up into the next binade: still on the grid */
  if (r > 448.0) r = 448.0;
  if (r == 0.0) return sign;
  (void)frexp(r, &e);
  ex = e - 1;
  if (ex < -6) return (uint8_t)(sign | (uint8_t)(r / ldexp(1.0, -9)));          /* subnormal: m = r / 2^-9 */
  int m = (int)((r / ldexp(1.0, ex) - 1.0) * 8.0);
  return (uint8_t)(sign | ((ex + 7) << 3) | m);
}

void oracle_e4m3_encode_many(const float* y, int64_t n, uint8_t* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = oracle_e4m3_encode(y[i]);
}

static int64_t kv8_tile_bytes(const oracle_dims_t* D) { return 32 * (int64_t)D->head_dim + 128; }
static int64_t kv8_tile(const oracle_dims_t* D, int64_t layer, int64_t block, int64_t head) {
  return ((layer * D->num_blocks + block) * D->num_kv_heads + head) * kv8_tile_bytes(D);
}

static float bf16_to_float(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return f;
}

/* one row: codes[d] and the fp32 scale, by the steps in the header comment */
static float quantise_row(const uint16_t* x, int32_t d, uint8_t* codes) {
  float amax = 0.0f;
  for (int32_t j = 0; j < d; ++j) {
    float a = fabsf(bf16_to_float(x[j]));
    if (a > amax) amax = a;
  }
  volatile float scale = amax == 0.0f ? 1.0f : amax / 448.0f;   /* volatile: force the fp32 rounding */
  volatile float inv = amax == 0.0f ? 1.0f : 448.0f / amax;
  for (int32_t j = 0; j < d; ++j) {
    volatile float y = bf16_to_float(x[j]) * inv;
    codes[j] = oracle_e4m3_encode(y);
  }
  return scale;
}

/* Quantising scatter: oracle_scatter's relocation with each row quantised on the way. */
void oracle_scatter_fp8(uint8_t* kv8, const oracle_dims_t* D, const int32_t* blocks, int32_t start_pos,
                        int32_t n, const uint16_t* k_src, const uint16_t* v_src, int32_t layer_begin,
                        int32_t layer_count) {
  const int32_t d = D->head_dim;
  for (int32_t ll = 0; ll < layer_count; ++ll)
    for (int32_t h = 0; h < D->num_kv_heads; ++h)
      for (int32_t t = 0; t < n; ++t) {
        int32_t pos = start_pos + t;
        int32_t slot = pos % D->block_size;
        uint8_t* tile = kv8 + kv8_tile(D, layer_begin + ll, blocks[pos / D->block_size], h);
        int64_t s = (((int64_t)ll * D->num_kv_heads + h) * n + t) * d;
        float ks = quantise_row(k_src + s, d, tile + (int64_t)slot * d);
        float vs = quantise_row(v_src + s, d, tile + 16 * (int64_t)d + (int64_t)slot * d);
        memcpy(tile + 32 * (int64_t)d + slot * 8, &ks, 4);
        memcpy(tile + 32 * (int64_t)d + slot * 8 + 4, &vs, 4);
      }
}

/* Dequantised row of one token as doubles: c = 0 K, 1 V. */
static void dequant_row(const uint8_t* kv8, const oracle_dims_t* D, int32_t layer, int32_t block, int32_t head,
                        int32_t c, int32_t slot, double* out) {
  const int32_t d = D->head_dim;
  const uint8_t* tile = kv8 + kv8_tile(D, layer, block, head);
  float sc;
  memcpy(&sc, tile + 32 * (int64_t)d + slot * 8 + 4 * c, 4);
  const uint8_t* codes = tile + (int64_t)c * 16 * d + (int64_t)slot * d;
  for (int32_t j = 0; j < d; ++j) out[j] = e4m3_decode(codes[j]) * (double)sc;
}

/* Gather + dequantise one request's layer: k_out / v_out fp64 [num_kv_heads][len][d] (test support). */
void oracle_dequant_fp8(const uint8_t* kv8, const oracle_dims_t* D, int32_t layer, const int32_t* blocks,
                        int32_t len, double* k_out, double* v_out) {
  const int32_t d = D->head_dim;
  for (int32_t h = 0; h < D->num_kv_heads; ++h)
    for (int32_t t = 0; t < len; ++t) {
      int64_t o = ((int64_t)h * len + t) * d;
      dequant_row(kv8, D, layer, blocks[t / D->block_size], h, 0, t % D->block_size, k_out + o);
      dequant_row(kv8, D, layer, blocks[t / D->block_size], h, 1, t % D->block_size, v_out + o);
    }
}

/* oracle_attention over an FP8 pool: the same definition on the dequantised values. */
int oracle_attention_fp8(const uint8_t* kv8, const oracle_dims_t* D, int32_t layer, int32_t num_q_heads,
                         int32_t batch, const int32_t* bt, const int64_t* bt_off, const int32_t* seq_lens,
                         const uint16_t* q, double scale, double* out, double* wsum) {
  const int32_t d = D->head_dim, Hq = num_q_heads, G = num_q_heads / D->num_kv_heads;
  for (int32_t r = 0; r < batch; ++r)
    if (seq_lens[r] < 1) return -1;
  int bad = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int32_t r = 0; r < batch; ++r)
    for (int32_t h = 0; h < Hq; ++h) {
      const int32_t g = h / G, n = seq_lens[r];
      const int32_t* blocks = bt + bt_off[r];
      const uint16_t* qv = q + ((int64_t)r * Hq + h) * d;
      double* s = (double*)malloc(sizeof(double) * (size_t)n);
      double* row = (double*)malloc(sizeof(double) * (size_t)d);
      double* o = out + ((int64_t)r * Hq + h) * d;
      if (!s || !row) { bad = 1; free(s); free(row); continue; }
      for (int32_t t = 0; t < n; ++t) {
        dequant_row(kv8, D, layer, blocks[t / D->block_size], g, 0, t % D->block_size, row);
        double acc = 0.0;
        for (int32_t j = 0; j < d; ++j) acc += bf16_to_double(qv[j]) * row[j];
        s[t] = scale * acc;
      }
      double m = s[0];
      for (int32_t t = 1; t < n; ++t)
        if (s[t] > m) m = s[t];
      double Z = 0.0;
      for (int32_t t = 0; t < n; ++t) {
        s[t] = exp(s[t] - m);
        Z += s[t];
      }
      for (int32_t j = 0; j < d; ++j) o[j] = 0.0;
      double ws = 0.0;
      for (int32_t t = 0; t < n; ++t) {
        dequant_row(kv8, D, layer, blocks[t / D->block_size], g, 1, t % D->block_size, row);
        double w = s[t] / Z;
        ws += w;
        for (int32_t j = 0; j < d; ++j) o[j] += w * row[j];
      }
      if (wsum) wsum[(int64_t)r * Hq + h] = ws;
      free(s);
      free(row);
    }
  return bad ? -2 : 0;
}

/* oracle_attention_varq over an FP8 pool: the variable-q-length causal definition (readings B1-B3) on the
 * dequantised values (readings C1-C4).  Same arguments as oracle_attention_varq. */
int oracle_attention_varq_fp8(const uint8_t* kv8, const oracle_dims_t* D, int32_t layer, int32_t num_q_heads,
                              int32_t batch, const int32_t* bt, const int64_t* bt_off, const int32_t* seq_lens,
                              const int32_t* q_lens, const int64_t* q_off, const uint16_t* q, double scale,
                              double* out, double* wsum) {
  const int32_t d = D->head_dim, Hq = num_q_heads, G = num_q_heads / D->num_kv_heads;
  for (int32_t r = 0; r < batch; ++r)
    if (q_lens[r] < 1 || q_lens[r] > seq_lens[r]) return -1;
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t r = 0; r < batch; ++r) {
    const int32_t* blocks = bt + bt_off[r];
    const int32_t len = seq_lens[r];
    /* dequantise the request's layer once: [kv head][token][d] */
    double* kd = (double*)malloc(sizeof(double) * (size_t)D->num_kv_heads * (size_t)len * (size_t)d);
    double* vd = (double*)malloc(sizeof(double) * (size_t)D->num_kv_heads * (size_t)len * (size_t)d);
    double* s = (double*)malloc(sizeof(double) * (size_t)len);
    if (!kd || !vd || !s) { bad = 1; free(kd); free(vd); free(s); continue; }
    oracle_dequant_fp8(kv8, D, layer, blocks, len, kd, vd);
    for (int32_t i = 0; i < q_lens[r]; ++i) {
      const int32_t n = len - q_lens[r] + i + 1;   /* tokens 0 .. P_i visible */
      for (int32_t h = 0; h < Hq; ++h) {
        const double* kh = kd + (int64_t)(h / G) * len * d;
        const double* vh = vd + (int64_t)(h / G) * len * d;
        const uint16_t* qv = q + ((q_off[r] + i) * Hq + h) * d;
        double* o = out + ((q_off[r] + i) * Hq + h) * d;
        for (int32_t t = 0; t < n; ++t) {
          double acc = 0.0;
          for (int32_t j = 0; j < d; ++j) acc += bf16_to_double(qv[j]) * kh[(int64_t)t * d + j];
          s[t] = scale * acc;
        }
        double m = s[0];
        for (int32_t t = 1; t < n; ++t)
          if (s[t] > m) m = s[t];
        double Z = 0.0;
        for (int32_t t = 0; t < n; ++t) {
          s[t] = exp(s[t] - m);
          Z += s[t];
        }
        for (int32_t j = 0; j < d; ++j) o[j] = 0.0;
        double ws = 0.0;
        for (int32_t t = 0; t < n; ++t) {
          double w = s[t] / Z;
          ws += w;
          for (int32_t j = 0; j < d; ++j) o[j] += w * vh[(int64_t)t * d + j];
        }
        if (wsum) wsum[(q_off[r] + i) * Hq + h] = ws;
      }
    }
    free(kd); free(vd); free(s);
  }
  return bad ? -2 : 0;
}

/* =============================================================================================
 * NEXT-4: producer -> consumer KV transfer.  PAPER.md:82 (§II): "KV-cache
 * transmission can add on the order of 15-80ms depending on block fragmentation and count";
 * PAPER.md:360 (§V-C): the KV-cache transmitter moves a prefill-completed request's KV out of the
 * producer's KV-cache blocks into KV-cache blocks registered on the consumer.  Both sides are
 * paged pools with their OWN block lists (and their own num_blocks), so the operation is, by
 * definition, "gather from pool A through A's block list, then scatter into pool B through B's":
 * token t of the request moves from A's block src_blocks[t / bs], slot t % bs, to B's block
 * dst_blocks[t / bs], slot t % bs, for every layer in [layer_begin, layer_begin + layer_count),
 * every kv head, K and V.  Pure bit copies; A is read-only; bytes of B outside the n written
 * token slots keep their contents (reading A5).  The two pools share layer count, kv heads,
 * head_dim and block_size (checked by the caller); num_blocks may differ.
 * ============================================================================================= */
void oracle_transfer(const uint16_t* src_kv, const oracle_dims_t* Ds, const int32_t* src_blocks,
                     uint16_t* dst_kv, const oracle_dims_t* Dd, const int32_t* dst_blocks, int32_t n,
                     int32_t layer_begin, int32_t layer_count) {
  for (int32_t l = layer_begin; l < layer_begin + layer_count; ++l)
    for (int32_t h = 0; h < Ds->num_kv_heads; ++h)
      for (int32_t t = 0; t < n; ++t) {
        int32_t slot = t % Ds->block_size;
        int32_t sb = src_blocks[t / Ds->block_size], db = dst_blocks[t / Dd->block_size];
        for (int32_t c = 0; c < 2; ++c)
          for (int32_t j = 0; j < Ds->head_dim; ++j)
            dst_kv[kv_index(Dd, l, db, h, c, slot, j)] = src_kv[kv_index(Ds, l, sb, h, c, slot, j)];
      }
}

/* The same relocation between two FP8 pools: a token's d codes of K, d codes of V and its two fp32
 * row scales (ks_t, vs_t) move verbatim — no re-quantisation (a code row and its scale are a pure
 * function of the token row, reading C2, so they mean the same in any pool). */
void oracle_transfer_fp8(const uint8_t* src_kv8, const oracle_dims_t* Ds, const int32_t* src_blocks,
                         uint8_t* dst_kv8, const oracle_dims_t* Dd, const int32_t* dst_blocks, int32_t n,
                         int32_t layer_begin, int32_t layer_count) {
  const int64_t d = Ds->head_dim;
  for (int32_t l = layer_begin; l < layer_begin + layer_count; ++l)
    for (int32_t h = 0; h < Ds->num_kv_heads; ++h)
      for (int32_t t = 0; t < n; ++t) {
        int32_t slot = t % 16;
        const uint8_t* st = src_kv8 + kv8_tile(Ds, l, src_blocks[t / 16], h);
        uint8_t* dt = dst_kv8 + kv8_tile(Dd, l, dst_blocks[t / 16], h);
        for (int64_t j = 0; j < d; ++j) {
          dt[slot * d + j] = st[slot * d + j];                       /* K codes */
          dt[16 * d + slot * d + j] = st[16 * d + slot * d + j];     /* V codes */
        }
        for (int32_t b = 0; b < 8; ++b) dt[32 * d + slot * 8 + b] = st[32 * d + slot * 8 + b];  /* ks_t, vs_t */
      }
}

/* Inverse of oracle_scatter_fp8's relocation (NOT of its quantisation): the stored codes and scales of
 * tokens [0, len), all layers, in contiguous form — the producer-side paged -> contiguous step on an FP8
 * pool.  k_codes / v_codes: [num_layers][num_kv_heads][len][d] bytes; k_scales / v_scales:
 * [num_layers][num_kv_heads][len] fp32. */
void oracle_gather_fp8(const uint8_t* kv8, const oracle_dims_t* D, const int32_t* blocks, int32_t len,
                       uint8_t* k_codes, float* k_scales, uint8_t* v_codes, float* v_scales) {
  const int64_t d = D->head_dim;
  for (int32_t l = 0; l < D->num_layers; ++l)
    for (int32_t h = 0; h < D->num_kv_heads; ++h)
      for (int32_t t = 0; t < len; ++t) {
        int32_t slot = t % 16;
        const uint8_t* tile = kv8 + kv8_tile(D, l, blocks[t / 16], h);
        int64_t row = ((int64_t)l * D->num_kv_heads + h) * len + t;
        for (int64_t j = 0; j < d; ++j) {
          k_codes[row * d + j] = tile[slot * d + j];
          v_codes[row * d + j] = tile[16 * d + slot * d + j];
        }
        memcpy(&k_scales[row], tile + 32 * d + slot * 8, 4);
        memcpy(&v_scales[row], tile + 32 * d + slot * 8 + 4, 4);
      }
}
