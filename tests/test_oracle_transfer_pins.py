"""Pins of the oracle's NEXT-4 functions ("block fragmentation and
count", PAPER.md:360 KV-cache transmitter into the consumer's KV-cache blocks) against things other
than themselves.  CPU only.

  T1  transfer A -> B          == oracle_scatter of the ORIGINAL contiguous source through B's block
                                  list, over the WHOLE sentinel-filled slab of B (so: gather o scatter,
                                  no stray writes); A is untouched; gather(B) returns the source
  T2  transfer A -> B          == an independent numpy fancy-index statement on 6-d views of both slabs
                                  (a wrong stride, a swapped K|V or a swapped block list fails it)
  T3  ragged tail / geometry   : pools of different num_blocks and different block lists; slots past
                                  the request's end in B's last block keep the sentinel; n = 0 is a no-op;
                                  a layer slice touches only its layers
  T4  transfer_fp8 A -> B      == oracle_scatter_fp8 of the original source into B (codes AND scales,
                                  byte for byte, whole slab) and a numpy byte-view statement; A untouched
  G1  gather_fp8               : codes x scales == oracle_dequant_fp8 of every layer; equals a numpy index
                                  statement of the documented tile layout K8[16][d] | V8[16][d] | sc[16][2]
"""
import numpy as np
import pytest

import oracle

SENT = 0x7FC0


def rand_bits(rng, shape):
    return rng.integers(0, 1 << 16, size=shape, dtype=np.uint16)   # arbitrary bit patterns: a copy must not care


def blocks_for(rng, n_blocks_pool, count):
    return rng.permutation(n_blocks_pool)[:count].astype(np.int32)


@pytest.mark.parametrize("n", [1, 15, 16, 17, 64, 130, 255])
def test_t1_transfer_equals_scatter_of_source(n):
    rng = np.random.default_rng(n)
    L, H, d = 3, 2, 64
    A = oracle.Dims(L, H, d, 16, 40)
    B = oracle.Dims(L, H, d, 16, 23)                       # a different pool size
    nb = (n + 15) // 16
    ba, bb = blocks_for(rng, 40, nb), blocks_for(rng, 23, nb)
    k, v = rand_bits(rng, (L, H, n, d)), rand_bits(rng, (L, H, n, d))
    slab_a = oracle.new_slab(A, 0x1234)
    oracle.scatter(slab_a, A, ba, 0, k, v)
    keep_a = slab_a.copy()
    slab_b = oracle.new_slab(B, SENT)
    oracle.transfer(slab_a, A, ba, slab_b, B, bb, n)
    want = oracle.new_slab(B, SENT)
    oracle.scatter(want, B, bb, 0, k, v)
    assert np.array_equal(slab_b, want)
    assert np.array_equal(slab_a, keep_a)                  # the producer's pool is read-only
    gk, gv = oracle.gather(slab_b, B, bb, n)
    assert np.array_equal(gk, k) and np.array_equal(gv, v)


def test_t2_transfer_equals_numpy_index_statement():
    rng = np.random.default_rng(7)
    L, H, d, n = 2, 3, 128, 77
    A, B = oracle.Dims(L, H, d, 16, 19), oracle.Dims(L, H, d, 16, 31)
    nb = (n + 15) // 16
    ba, bb = blocks_for(rng, 19, nb), blocks_for(rng, 31, nb)
    slab_a = rand_bits(rng, A.kv_elems)                    # whole pool random: no scatter involved at all
    slab_b = oracle.new_slab(B, SENT)
    oracle.transfer(slab_a, A, ba, slab_b, B, bb, n)
    va, want = slab_a.reshape(A.shape()), oracle.new_slab(B, SENT).reshape(B.shape())
    t = np.arange(n)
    want[:, bb[t // 16], :, :, t % 16, :] = va[:, ba[t // 16], :, :, t % 16, :]
    assert np.array_equal(slab_b.reshape(B.shape()), want)


def test_t3_tail_slots_layers_and_empty():
    rng = np.random.default_rng(11)
    L, H, d, n = 4, 2, 64, 37                              # last block holds 5 tokens
    A, B = oracle.Dims(L, H, d, 16, 8), oracle.Dims(L, H, d, 16, 9)
    ba, bb = np.array([5, 0, 7], np.int32), np.array([2, 8, 3], np.int32)
    slab_a = rand_bits(rng, A.kv_elems)
    slab_b = oracle.new_slab(B, SENT)
    oracle.transfer(slab_a, A, ba, slab_b, B, bb, n, layer_begin=1, layer_count=2)
    vb, va = slab_b.reshape(B.shape()), slab_a.reshape(A.shape())
    assert np.all(vb[0] == SENT) and np.all(vb[3] == SENT)                     # layers outside the slice
    assert np.all(vb[1:3, 3, :, :, 5:, :] == SENT)                             # slots past the end
    assert np.array_equal(vb[1:3, 3, :, :, :5, :], va[1:3, 7, :, :, :5, :])
    assert np.array_equal(vb[1:3, 2], va[1:3, 5]) and np.array_equal(vb[1:3, 8], va[1:3, 0])
    untouched = np.setdiff1d(np.arange(9), bb)
    assert np.all(vb[:, untouched] == SENT)
    before = slab_b.copy()
    oracle.transfer(slab_a, A, ba, slab_b, B, bb, 0)
    assert np.array_equal(slab_b, before)


@pytest.mark.parametrize("d,n", [(64, 33), (128, 16), (128, 50)])
def test_t4_transfer_fp8(d, n):
    rng = np.random.default_rng(d + n)
    L, H = 2, 2
    A, B = oracle.Dims(L, H, d, 16, 12), oracle.Dims(L, H, d, 16, 7)
    nb = (n + 15) // 16
    ba, bb = blocks_for(rng, 12, nb), blocks_for(rng, 7, nb)
    # finite bf16 rows with a wide spread of magnitudes
    x = (rng.standard_normal((2, L, H, n, d)) * np.exp(rng.uniform(-4, 4, (2, L, H, n, 1)))).astype(np.float32)
    bits = (x.view(np.uint32) >> 16).astype(np.uint16)
    slab_a = oracle.new_slab_fp8(A, 0xEE)
    oracle.scatter_fp8(slab_a, A, ba, 0, bits[0], bits[1])
    keep_a = slab_a.copy()
    slab_b = oracle.new_slab_fp8(B, 0xFF)
    oracle.transfer_fp8(slab_a, A, ba, slab_b, B, bb, n)
    want = oracle.new_slab_fp8(B, 0xFF)
    oracle.scatter_fp8(want, B, bb, 0, bits[0], bits[1])
    assert np.array_equal(slab_b, want)
    assert np.array_equal(slab_a, keep_a)
    # numpy byte-view statement of the same move on a fully random source pool
    slab_r = rng.integers(0, 256, size=A.fp8_bytes, dtype=np.uint8)
    got = oracle.new_slab_fp8(B, 0xFF)
    oracle.transfer_fp8(slab_r, A, ba, got, B, bb, n)
    ta, tb = slab_r.reshape(L, 12, H, 32 * d + 128), oracle.new_slab_fp8(B, 0xFF).reshape(L, 7, H, 32 * d + 128)
    for t in range(n):
        s, a, b = t % 16, ba[t // 16], bb[t // 16]
        tb[:, b, :, s * d:(s + 1) * d] = ta[:, a, :, s * d:(s + 1) * d]
        tb[:, b, :, 16 * d + s * d:16 * d + (s + 1) * d] = ta[:, a, :, 16 * d + s * d:16 * d + (s + 1) * d]
        tb[:, b, :, 32 * d + 8 * s:32 * d + 8 * s + 8] = ta[:, a, :, 32 * d + 8 * s:32 * d + 8 * s + 8]
    assert np.array_equal(got.reshape(tb.shape), tb)


@pytest.mark.parametrize("d", [64, 128])
def test_g1_gather_fp8(d):
    rng = np.random.default_rng(d)
    L, H, n = 3, 2, 45
    D = oracle.Dims(L, H, d, 16, 10)
    blocks = blocks_for(rng, 10, 3)
    x = (rng.standard_normal((2, L, H, n, d)) * np.exp(rng.uniform(-3, 3, (2, L, H, n, 1)))).astype(np.float32)
    bits = (x.view(np.uint32) >> 16).astype(np.uint16)
    slab = oracle.new_slab_fp8(D, 0xFF)
    oracle.scatter_fp8(slab, D, blocks, 0, bits[0], bits[1])
    kc, ks, vc, vs = oracle.gather_fp8(slab, D, blocks, n)
    table = oracle.e4m3_decode_table()
    for l in range(L):
        kd, vd = oracle.dequant_fp8(slab, D, l, blocks, n)
        assert np.array_equal(table[kc[l]] * ks[l][..., None].astype(np.float64), kd)
        assert np.array_equal(table[vc[l]] * vs[l][..., None].astype(np.float64), vd)
    # numpy index statement of the tile layout
    tiles = slab.reshape(L, 10, H, 32 * d + 128)
    t = np.arange(n)
    codes_k = tiles[..., : 16 * d].reshape(L, 10, H, 16, d)[:, blocks[t // 16], :, t % 16, :]      # [n][L][H][d]
    codes_v = tiles[..., 16 * d: 32 * d].reshape(L, 10, H, 16, d)[:, blocks[t // 16], :, t % 16, :]
    sc = tiles[..., 32 * d:].copy().view(np.float32).reshape(L, 10, H, 16, 2)[:, blocks[t // 16], :, t % 16, :]
    assert np.array_equal(kc, codes_k.transpose(1, 2, 0, 3)) and np.array_equal(vc, codes_v.transpose(1, 2, 0, 3))
    assert np.array_equal(ks, sc[..., 0].transpose(1, 2, 0)) and np.array_equal(vs, sc[..., 1].transpose(1, 2, 0))
