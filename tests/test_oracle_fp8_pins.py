"""Pins of the oracle's FP8 (e4m3) KV functions (readings C1-C4) against
things other than themselves.  CPU only.

  F1  e4m3 decode table          == torch.float8_e4m3fn on all 256 codes                    (library)
  F2  RNE encoder                == torch's float32 -> float8_e4m3fn cast on every representable value,
                                    every midpoint between neighbours (ties to even), one fp32 ulp either
                                    side of each midpoint, a dense random sweep, the subnormal range;
                                    saturation to +-448 by definition above 448                 (library)
  F3  quantising scatter         == an independent numpy float32 + torch-float8 statement over the WHOLE
                                    slab (untouched bytes keep the sentinel); brute force: no other code
                                    is nearer; the amax element gets code +-448; zero rows get scale 1;
                                    |x - x^| <= 16 scale (half the top-binade spacing)
  F4  attention over an FP8 pool == oracle_attention on a bf16 pool when every row is exactly
                                    representable (power-of-two scale), and torch SDPA in fp64 on the
                                    dequantised values for random data                          (library)
"""
import math

import numpy as np
import pytest
import torch

import oracle
from helpers import bf16_bits, bits_to_f64


def torch_e4m3(y32: np.ndarray) -> np.ndarray:
    return torch.from_numpy(np.ascontiguousarray(y32, dtype=np.float32)).to(torch.float8_e4m3fn).view(torch.uint8).numpy()


def test_f1_decode_table():
    ref = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).double().numpy()
    got = oracle.e4m3_decode_table()
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.isnan(got).sum() == 2
    assert np.array_equal(got[~np.isnan(got)], ref[~np.isnan(ref)])
    assert got[0x7e] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6 and got[0x38] == 1.0


def test_f2_encoder_matches_torch():
    table = oracle.e4m3_decode_table()
    pos = np.sort(table[:0x7f])                                   # 0 .. 448, the 127 non-negative finite values
    mids = (pos[:-1] + pos[1:]) / 2                               # exactly representable in fp32
    pts = np.concatenate([pos, mids, np.nextafter(mids.astype(np.float32), np.float32(0)),
                          np.nextafter(mids.astype(np.float32), np.float32(1e9))]).astype(np.float32)
    rng = np.random.default_rng(0)
    sweep = np.concatenate([pts, rng.uniform(0, 448, 200000).astype(np.float32),
                            (rng.uniform(0, 1, 50000) * 2.0 ** -5).astype(np.float32),
                            np.exp(rng.uniform(math.log(1e-6), math.log(448), 100000)).astype(np.float32)])
    sweep = np.concatenate([sweep, -sweep])
    got, ref = oracle.e4m3_encode(sweep), torch_e4m3(sweep)
    bad = np.nonzero(got != ref)[0]
    assert bad.size == 0, (sweep[bad[:5]], got[bad[:5]], ref[bad[:5]])
    # ties to even, spelled out: 1.0625 is halfway between 1.0 (0x38, even) and 1.125 (0x39)
    assert list(oracle.e4m3_encode([1.0625, 1.1875, 2.0 ** -10, 3 * 2.0 ** -10])) == [0x38, 0x3A, 0x00, 0x02]
    # satfinite (torch's cast is non-saturating above 464; quantised rows never exceed 448 (1 + 2^-23))
    assert list(oracle.e4m3_encode([448.0, 448.0001, 464.0, 480.0, 1e9, -1e9, np.inf])) == [0x7E] * 5 + [0xFE, 0x7E]


def numpy_quantise(x_bits):
    """Independent statement of DESIGN.md C1-C4 for rows [..., d]: numpy float32 arithmetic + torch float8 cast."""
    x = bits_to_f64(x_bits).astype(np.float32)
    amax = np.abs(x).max(axis=-1, keepdims=True)
    zero = amax == 0
    safe = np.where(zero, np.float32(1), amax)
    scale = np.where(zero, np.float32(1), safe / np.float32(448)).astype(np.float32)
    inv = np.where(zero, np.float32(1), np.float32(448) / safe).astype(np.float32)
    y = (x * inv).astype(np.float32)
    return torch_e4m3(np.minimum(np.maximum(y, -448), 448)), scale[..., 0]


@pytest.mark.parametrize("d,Hkv", [(64, 2), (128, 1)])
def test_f3_quantising_scatter(d, Hkv):
    rng = np.random.default_rng(1)
    L, NB, n, start = 2, 12, 53, 7
    dims = oracle.Dims(L, Hkv, d, 16, NB)
    blocks = rng.permutation(NB)[: (start + n + 15) // 16].astype(np.int32)
    k = rng.standard_normal((L, Hkv, n, d)) * np.exp(rng.uniform(-6, 6, (L, Hkv, n, 1)))   # row scales 1e-3 .. 4e2
    v = rng.standard_normal((L, Hkv, n, d))
    k[0, 0, 3] = 0.0                                               # a zero row
    kb, vb = bf16_bits(k), bf16_bits(v)
    kv8 = oracle.new_slab_fp8(dims, 0xA5)
    oracle.scatter_fp8(kv8, dims, blocks, start, kb, vb)
    # independent whole-slab statement
    want = np.full(dims.fp8_bytes, 0xA5, dtype=np.uint8)
    T = dims.fp8_tile_bytes
    kc, ks = numpy_quantise(kb)
    vc, vs = numpy_quantise(vb)
    for l in range(L):
        for h in range(Hkv):
            for t in range(n):
                pos = start + t
                base = ((l * NB + int(blocks[pos // 16])) * Hkv + h) * T
                want[base + (pos % 16) * d: base + (pos % 16 + 1) * d] = kc[l, h, t]
                want[base + 16 * d + (pos % 16) * d: base + 16 * d + (pos % 16 + 1) * d] = vc[l, h, t]
                want[base + 32 * d + (pos % 16) * 8: base + 32 * d + (pos % 16) * 8 + 8] = \
                    np.array([ks[l, h, t], vs[l, h, t]], dtype=np.float32).view(np.uint8)
    assert np.array_equal(kv8, want)
    # properties, via the dequantising reader
    kd, vd = oracle.dequant_fp8(kv8, dims, 1, blocks, start + n)
    table = oracle.e4m3_decode_table()
    finite = table[~np.isnan(table)]
    x = bits_to_f64(kb)[1]                                          # layer 1: [Hkv][n][d]
    xh = kd[:, start:]
    sc = ks[1].astype(np.float64)[..., None]
    assert np.all(np.abs(x - xh) <= 16 * sc * (1 + 1e-6))
    am = np.abs(x).argmax(axis=-1)
    assert np.all(np.abs(np.take_along_axis(xh, am[..., None], -1)[..., 0]) == 448 * sc[..., 0])
    # brute force on a few rows: the stored code is a nearest grid point of fl32(x * inv)
    for h, t in [(0, 0), (Hkv - 1, n - 1), (0, 17)]:
        amax = np.float32(np.abs(x[h, t]).max())
        y = (x[h, t].astype(np.float32) * (np.float32(448) / amax)).astype(np.float64)
        stored = xh[h, t] / sc[h, t]
        best = np.abs(y[:, None] - finite[None, :]).min(axis=1)
        assert np.all(np.abs(y - stored) <= best + 1e-12)
    assert np.all(oracle.dequant_fp8(kv8, dims, 0, blocks, start + n)[0][0, start + 3] == 0.0)


def test_f4_exactly_representable_rows_reduce_to_the_bf16_oracle():
    rng = np.random.default_rng(2)
    Hq, Hkv, d, NB = 8, 2, 64, 16
    lens = [37, 100]
    dims = oracle.Dims(1, Hkv, d, 16, NB)
    kv8, kv16 = oracle.new_slab_fp8(dims, 0xFF), oracle.new_slab(dims, 0x7FC0)
    grid = oracle.e4m3_decode_table()[:0x7f]
    blocks, p = [], 0
    for n in lens:
        nb = (n + 15) // 16
        blocks.append(np.arange(p, p + nb, dtype=np.int32)); p += nb
        # every row: e4m3 grid values times 2^k, with one element equal to +-448 * 2^k  ->  scale = 2^k exactly
        def rows():
            x = rng.choice(grid, size=(1, Hkv, n, d)) * rng.choice([-1.0, 1.0], size=(1, Hkv, n, d))
            x[..., 0] = 448.0
            return x * 2.0 ** rng.integers(-12, -5, size=(1, Hkv, n, 1))
        k, v = bf16_bits(rows()), bf16_bits(rows())
        oracle.scatter_fp8(kv8, dims, blocks[-1], 0, k, v)
        oracle.scatter(kv16, dims, blocks[-1], 0, k, v)
    q = bf16_bits(rng.standard_normal((2, Hq, d)) * 4)
    a = oracle.attention_fp8(kv8, dims, 0, Hq, blocks, lens, q)
    b = oracle.attention(kv16, dims, 0, Hq, blocks, lens, q)
    assert np.max(np.abs(a - b)) < 1e-13


def test_f4_sdpa_on_dequantised_values():
    rng = np.random.default_rng(3)
    Hq, Hkv, d, NB = 8, 2, 128, 40
    lens = [1, 17, 255, 300]
    dims = oracle.Dims(1, Hkv, d, 16, NB)
    kv8 = oracle.new_slab_fp8(dims, 0xFF)                          # 0xFF = e4m3 NaN: a stray read poisons the row
    perm, blocks, p = rng.permutation(NB), [], 0
    for n in lens:
        nb = (n + 15) // 16
        blocks.append(perm[p:p + nb].astype(np.int32)); p += nb
        oracle.scatter_fp8(kv8, dims, blocks[-1], 0, bf16_bits(rng.standard_normal((1, Hkv, n, d))),
                           bf16_bits(rng.standard_normal((1, Hkv, n, d))))
    q = bf16_bits(rng.standard_normal((len(lens), Hq, d)))
    got, wsum = oracle.attention_fp8(kv8, dims, 0, Hq, blocks, lens, q, return_wsum=True)
    assert np.all(np.abs(wsum - 1) < 1e-12)
    for r, n in enumerate(lens):
        kd, vd = oracle.dequant_fp8(kv8, dims, 0, blocks[r], n)
        kk = torch.from_numpy(kd).repeat_interleave(Hq // Hkv, 0)[None]
        vv = torch.from_numpy(vd).repeat_interleave(Hq // Hkv, 0)[None]
        qq = torch.from_numpy(bits_to_f64(q[r]))[None, :, None, :]
        want = torch.nn.functional.scaled_dot_product_attention(qq, kk, vv)[0, :, 0].numpy()
        assert np.max(np.abs(got[r] - want)) < 1e-10
    # n = 1: the output is the dequantised V_0 exactly
    _, vd = oracle.dequant_fp8(kv8, dims, 0, blocks[0], 1)
    assert np.array_equal(got[0], np.repeat(vd[:, 0], Hq // Hkv, axis=0))


def test_f5_varq_over_fp8_pool():
    """oracle_attention_varq_fp8: q_len = 1 == attention_fp8 (bit for bit); exactly representable rows ==
    attention_varq on the bf16 pool; random data == torch SDPA (causal, lower-right aligned, fp64) on the
    dequantised values."""
    rng = np.random.default_rng(4)
    Hq, Hkv, d, NB = 8, 2, 64, 40
    lens, qls = [37, 100, 9, 260], [37, 13, 1, 130]
    dims = oracle.Dims(1, Hkv, d, 16, NB)
    kv8 = oracle.new_slab_fp8(dims, 0xFF)
    perm, blocks, p = rng.permutation(NB), [], 0
    for n in lens:
        nb = (n + 15) // 16
        blocks.append(perm[p:p + nb].astype(np.int32)); p += nb
        oracle.scatter_fp8(kv8, dims, blocks[-1], 0, bf16_bits(rng.standard_normal((1, Hkv, n, d))),
                           bf16_bits(rng.standard_normal((1, Hkv, n, d))))
    q1 = bf16_bits(rng.standard_normal((len(lens), Hq, d)))
    assert np.array_equal(oracle.attention_varq_fp8(kv8, dims, 0, Hq, blocks, lens, [1] * len(lens), q1),
                          oracle.attention_fp8(kv8, dims, 0, Hq, blocks, lens, q1))
    q = bf16_bits(rng.standard_normal((sum(qls), Hq, d)))
    got, wsum = oracle.attention_varq_fp8(kv8, dims, 0, Hq, blocks, lens, qls, q, return_wsum=True)
    assert np.all(np.abs(wsum - 1) < 1e-12)
    off = 0
    for r, (n, ql) in enumerate(zip(lens, qls)):
        kd, vd = oracle.dequant_fp8(kv8, dims, 0, blocks[r], n)
        kk = torch.from_numpy(kd).repeat_interleave(Hq // Hkv, 0)[None]
        vv = torch.from_numpy(vd).repeat_interleave(Hq // Hkv, 0)[None]
        qq = torch.from_numpy(bits_to_f64(q[off:off + ql])).permute(1, 0, 2)[None]
        mask = torch.arange(n)[None, :] <= (torch.arange(ql)[:, None] + (n - ql))
        want = torch.nn.functional.scaled_dot_product_attention(qq, kk, vv, attn_mask=mask)[0].permute(1, 0, 2).numpy()
        assert np.max(np.abs(got[off:off + ql] - want)) < 1e-10
        off += ql
    # exactly representable rows: the FP8 pool and the bf16 pool hold the same values
    kv8b, kv16 = oracle.new_slab_fp8(dims, 0xFF), oracle.new_slab(dims, 0x7FC0)
    grid = oracle.e4m3_decode_table()[:0x7f]
    for b, n in zip(blocks, lens):
        def rows():
            x = rng.choice(grid, size=(1, Hkv, n, d)) * rng.choice([-1.0, 1.0], size=(1, Hkv, n, d))
            x[..., 0] = 448.0
            return x * 2.0 ** rng.integers(-12, -5, size=(1, Hkv, n, 1))
        k, v = bf16_bits(rows()), bf16_bits(rows())
        oracle.scatter_fp8(kv8b, dims, b, 0, k, v)
        oracle.scatter(kv16, dims, b, 0, k, v)
    a = oracle.attention_varq_fp8(kv8b, dims, 0, Hq, blocks, lens, qls, q)
    c = oracle.attention_varq(kv16, dims, 0, Hq, blocks, lens, qls, q)
    assert np.max(np.abs(a - c)) < 1e-13
