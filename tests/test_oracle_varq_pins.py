"""Pins of oracle_attention_varq (variable-q-length causal paged attention; SURVEY §8(f) NEXT-1,
PAPER.md:443 PD-aggregation of ultra-short requests) against things other than itself:

  V1  q_len = 1 everywhere      == oracle_attention (already pinned by P1-P13), bit for bit
  V2  fresh prefill (q_len = n) == torch SDPA(is_causal=True) in fp64           (library routine)
  V3  chunked prefill (p > 0)   == torch SDPA with an explicit lower-right-aligned mask, fp64
  V4  first token of a fresh prefill returns V_0 exactly                        (special case)
  V5  q = 0 -> running means of V over the visible prefix                       (closed form, exact fractions)
  V6  query row i == decode over the sequence truncated to P_i + 1 tokens       (mask boundary, off-by-one)
  V7  rewriting tokens after P_i leaves row i unchanged, rewriting token P_i changes it (causality)
  V8  hand case: scores (0, ln 2, ln 3) seen by three successive queries -> weights
      (1), (1/3, 2/3), (1/6, 2/6, 3/6)                                          (by hand)
CPU only.
"""
import math

import numpy as np
import pytest
import torch

import oracle
from helpers import bf16_bits, bits_to_f64


def setup(seed, lens, Hq=8, Hkv=2, d=64, NB=96, bs=16):
    rng = np.random.default_rng(seed)
    dims = oracle.Dims(1, Hkv, d, bs, NB)
    kv = oracle.new_slab(dims, 0x7FC0)                      # NaN sentinel: an unmasked stray read poisons the row
    perm = rng.permutation(NB)
    blocks, p = [], 0
    K, V = [], []
    for n in lens:
        nb = (n + bs - 1) // bs
        blocks.append(perm[p:p + nb].astype(np.int32)); p += nb
        k = bf16_bits(rng.standard_normal((1, Hkv, n, d)))
        v = bf16_bits(rng.standard_normal((1, Hkv, n, d)))
        oracle.scatter(kv, dims, blocks[-1], 0, k, v)
        K.append(k); V.append(v)
    return rng, dims, kv, blocks, K, V


def sdpa_rows(K, V, q_bits, n, q_len, Hq, scale):
    """torch SDPA in fp64 for one request: q rows are the last q_len of n tokens."""
    Hkv = K.shape[1]
    G = Hq // Hkv
    k = torch.from_numpy(bits_to_f64(K[0])).repeat_interleave(G, 0)[None]       # [1][Hq][n][d]
    v = torch.from_numpy(bits_to_f64(V[0])).repeat_interleave(G, 0)[None]
    q = torch.from_numpy(bits_to_f64(q_bits)).permute(1, 0, 2)[None]            # [1][Hq][q_len][d]
    if q_len == n:
        o = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=True, scale=scale)
    else:
        i = torch.arange(q_len)[:, None] + (n - q_len)
        mask = torch.arange(n)[None, :] <= i                                      # lower-right aligned
        o = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=mask, scale=scale)
    return o[0].permute(1, 0, 2).numpy()                                          # [q_len][Hq][d]


def test_v1_qlen1_is_decode():
    lens = [17, 64, 130, 255, 1]
    rng, dims, kv, blocks, K, V = setup(1, lens)
    q = bf16_bits(rng.standard_normal((len(lens), 8, 64)))
    a = oracle.attention(kv, dims, 0, 8, blocks, lens, q)
    b = oracle.attention_varq(kv, dims, 0, 8, blocks, lens, [1] * len(lens), q)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (4, 4, 128), (8, 1, 64)])
def test_v2_v3_sdpa_causal(Hq, Hkv, d):
    lens = [33, 16, 100, 7, 250]
    q_lens = [33, 16, 100, 7, 250]            # V2: fresh prefill
    chunked = [5, 1, 37, 7, 128]              # V3: the last q_len tokens on top of p = n - q_len stored ones
    rng, dims, kv, blocks, K, V = setup(2, lens, Hq, Hkv, d, NB=64)
    scale = 1.0 / math.sqrt(d)
    for ql in (q_lens, chunked):
        q = bf16_bits(rng.standard_normal((sum(ql), Hq, d)))
        got, wsum = oracle.attention_varq(kv, dims, 0, Hq, blocks, lens, ql, q, return_wsum=True)
        assert np.all(np.abs(wsum - 1.0) < 1e-12)
        off = 0
        for r, n in enumerate(lens):
            want = sdpa_rows(K[r], V[r], q[off:off + ql[r]], n, ql[r], Hq, scale)
            assert np.max(np.abs(got[off:off + ql[r]] - want)) < 1e-10
            off += ql[r]


def test_v4_first_token_returns_v0():
    lens = [40, 3]
    rng, dims, kv, blocks, K, V = setup(3, lens)
    q = bf16_bits(rng.standard_normal((sum(lens), 8, 64)))
    got = oracle.attention_varq(kv, dims, 0, 8, blocks, lens, lens, q)
    off = 0
    for r, n in enumerate(lens):
        for h in range(8):
            assert np.array_equal(got[off, h], bits_to_f64(V[r][0, h // 4, 0]))
        off += n


def test_v5_zero_query_running_mean():
    n, p, Hq, Hkv, d = 77, 20, 4, 2, 64
    dims = oracle.Dims(1, Hkv, d, 16, 8)
    kv = oracle.new_slab(dims, 0x7FC0)
    blocks = [np.array([5, 2, 7, 0, 3], dtype=np.int32)]
    k = bf16_bits(np.random.default_rng(0).standard_normal((1, Hkv, n, d)))
    v = np.zeros((1, Hkv, n, d))
    v[..., 0] = 1.0
    v[0, :, :, 1] = np.arange(n)[None, :]                     # exact in bf16 (n < 256)
    oracle.scatter(kv, dims, blocks[0], 0, k, bf16_bits(v))
    ql = n - p
    got = oracle.attention_varq(kv, dims, 0, Hq, blocks, [n], [ql], np.zeros((ql, Hq, d), np.uint16))
    for i in range(ql):
        P = p + i
        assert np.allclose(got[i, :, 0], 1.0, rtol=0, atol=1e-14)
        assert np.allclose(got[i, :, 1], P / 2.0, rtol=0, atol=1e-12)   # mean of 0..P
        assert np.all(got[i, :, 2:] == 0.0)


def test_v6_rows_equal_truncated_decode():
    lens, ql = [50, 130], [50, 19]
    rng, dims, kv, blocks, K, V = setup(6, lens)
    q = bf16_bits(rng.standard_normal((sum(ql), 8, 64)))
    got = oracle.attention_varq(kv, dims, 0, 8, blocks, lens, ql, q)
    off = 0
    for r, n in enumerate(lens):
        for i in range(ql[r]):
            P = n - ql[r] + i
            want = oracle.attention(kv, dims, 0, 8, [blocks[r]], [P + 1], q[off + i][None])
            assert np.array_equal(got[off + i], want[0])
        off += ql[r]


def test_v7_causality():
    n, ql = 48, 48
    rng, dims, kv, blocks, K, V = setup(7, [n])
    q = bf16_bits(rng.standard_normal((ql, 8, 64)))
    base = oracle.attention_varq(kv, dims, 0, 8, blocks, [n], [ql], q)
    cut = 29
    k2, v2 = K[0].copy(), V[0].copy()
    k2[:, :, cut:] = bf16_bits(rng.standard_normal(k2[:, :, cut:].shape))
    v2[:, :, cut:] = bf16_bits(rng.standard_normal(v2[:, :, cut:].shape))
    oracle.scatter(kv, dims, blocks[0], 0, k2, v2)
    new = oracle.attention_varq(kv, dims, 0, 8, blocks, [n], [ql], q)
    assert np.array_equal(new[:cut], base[:cut])                     # rows before the cut never saw it
    assert np.all(np.abs(new[cut:] - base[cut:]).max(axis=(1, 2)) > 1e-6)   # rows from the cut on did (own token included)


def test_v8_hand_case():
    """K rows chosen so that q.K = 0, ln 2, ln 3 with sm_scale = 1 (scores exact up to the bf16 of ln 2, ln 3:
    use the bf16 values themselves as the definition).  V = e_0, e_1, e_2.  Query i sees tokens 0..i."""
    d = 64
    dims = oracle.Dims(1, 1, d, 16, 2)
    kv = oracle.new_slab(dims, 0x7FC0)
    k = np.zeros((1, 1, 3, d)); v = np.zeros((1, 1, 3, d))
    ln2 = bits_to_f64(bf16_bits([math.log(2)]))[0]
    ln3 = bits_to_f64(bf16_bits([math.log(3)]))[0]
    k[0, 0, 1, 0], k[0, 0, 2, 0] = ln2, ln3
    for t in range(3):
        v[0, 0, t, t] = 1.0
    oracle.scatter(kv, dims, np.array([1], np.int32), 0, bf16_bits(k), bf16_bits(v))
    q = np.zeros((3, 1, d)); q[:, 0, 0] = 1.0
    got = oracle.attention_varq(kv, dims, 0, 1, [np.array([1], np.int32)], [3], [3], bf16_bits(q), scale=1.0)
    e2, e3 = math.exp(ln2), math.exp(ln3)
    want = np.zeros((3, d))
    want[0, 0] = 1.0
    want[1, :2] = np.array([1.0, e2]) / (1.0 + e2)
    want[2, :3] = np.array([1.0, e2, e3]) / (1.0 + e2 + e3)
    assert np.max(np.abs(got[:, 0] - want)) < 1e-15
    assert abs(got[1, 0, 1] - 2.0 / 3.0) < 3e-3 and abs(got[2, 0, 2] - 0.5) < 3e-3   # (1/3, 2/3), (1/6, 2/6, 3/6)


def test_bad_q_len_is_an_error():
    rng, dims, kv, blocks, K, V = setup(9, [10])
    with pytest.raises(ValueError):
        oracle.attention_varq(kv, dims, 0, 8, blocks, [10], [11], np.zeros((11, 8, 64), np.uint16))
    with pytest.raises(ValueError):
        oracle.attention_varq(kv, dims, 0, 8, blocks, [10], [0], np.zeros((0, 8, 64), np.uint16))
