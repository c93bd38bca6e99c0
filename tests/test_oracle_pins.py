"""Pins of the oracle against things other than itself.

Every check compares oracle/kv_oracle.c with a value fixed by the paper's formula
(Eq. 1) and plain mathematics: hand-computed fixtures, closed forms,
invariants, and library routines (torch SDPA in fp64, scipy softmax + numpy matmul on
independently gathered rows).  CPU only.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.special
import torch

import oracle
from helpers import bf16_bits, bits_to_f64, exact_bf16

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def make_pool(L=1, Hkv=2, d=64, bs=16, NB=64, fill=0):
    dims = oracle.Dims(L, Hkv, d, bs, NB)
    return dims, oracle.new_slab(dims, fill)


def perm_blocks(rng, NB, n_tokens, bs=16):
    """Disjoint random block lists for a list of context lengths."""
    perm = rng.permutation(NB)
    out, p = [], 0
    for n in n_tokens:
        nb = (n + bs - 1) // bs
        out.append(perm[p:p + nb].astype(np.int32))
        p += nb
    assert p <= NB
    return out


def fill_requests(dims, kv, blocks, K, V):
    """K[r], V[r]: float arrays [L][Hkv][n][d] -> scatter as bf16 bits.  Returns the bit tensors."""
    kb, vb = [], []
    for b, k, v in zip(blocks, K, V):
        kbits, vbits = bf16_bits(k), bf16_bits(v)
        oracle.scatter(kv, dims, b, 0, kbits, vbits)
        kb.append(kbits)
        vb.append(vbits)
    return kb, vb


# --------------------------------------------------------------------------------------------
# P7: hand-computed cases (tests/golden/hand_cases.json)
# --------------------------------------------------------------------------------------------

@pytest.mark.parametrize("d", [64, 128])
def test_p7_hand_cases(d):
    with open(os.path.join(GOLDEN, "hand_cases.json")) as f:
        cases = json.load(f)["cases"]
    for case in cases:
        n = len(case["K"])
        dims, kv = make_pool(d=d, Hkv=1, NB=8, fill=0x7FC0)  # NaN sentinel in unused slots
        pad = lambda rows: np.array([r + [0] * (d - len(r)) for r in rows], dtype=np.float64)
        K, V, q = pad(case["K"]), pad(case["V"]), pad([case["q"]])
        assert exact_bf16(K) and exact_bf16(V) and exact_bf16(q)
        blocks = np.array([5], dtype=np.int32)
        oracle.scatter(kv, dims, blocks, 0, bf16_bits(K)[None, None], bf16_bits(V)[None, None])
        out, wsum = oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(q)[None], scale=math.log(2.0),
                                     return_wsum=True)
        want = pad([case["out"]])[0]
        assert np.allclose(out[0, 0], want, rtol=0, atol=1e-13), case["name"]
        # the fixture's rational weights reproduce its own `out` (fixture self-consistency)
        w = [Fraction(s) for s in case["weights"]]
        assert sum(w) == 1
        byhand = sum(float(wi) * V[i] for i, wi in enumerate(w))
        assert np.allclose(byhand, want, atol=1e-13)
        assert abs(wsum[0, 0] - 1) < 1e-12


def test_p7_sixths_in_doubles():
    """scores (0, ln 2, ln 3) with scale 1 -> weights (1/6, 2/6, 3/6); K entries are the bf16
    roundings of ln 2 / ln 3, so expected weights use the rounded values (closed form)."""
    dims, kv = make_pool(d=64, Hkv=1, NB=4)
    kvals = bits_to_f64(bf16_bits([0.0, math.log(2.0), math.log(3.0)]))
    K = np.zeros((3, 64)); K[:, 0] = kvals
    V = np.zeros((3, 64)); V[0, 0] = V[1, 1] = V[2, 2] = 1.0
    q = np.zeros((1, 64)); q[0, 0] = 1.0
    blocks = np.array([2], dtype=np.int32)
    oracle.scatter(kv, dims, blocks, 0, bf16_bits(K)[None, None], bf16_bits(V)[None, None])
    out = oracle.attention(kv, dims, 0, 1, [blocks], [3], bf16_bits(q)[None], scale=1.0)
    e = np.exp(kvals)
    assert np.allclose(out[0, 0, :3], e / e.sum(), atol=1e-14)
    assert np.allclose(out[0, 0, :3], [1 / 6, 2 / 6, 3 / 6], atol=3e-3)  # bf16(ln 2), bf16(ln 3) rounding


# --------------------------------------------------------------------------------------------
# P1, P2, P5, P8: closed forms
# --------------------------------------------------------------------------------------------

def test_p1_single_token_returns_v_exactly():
    rng = np.random.default_rng(1)
    dims, kv = make_pool(Hkv=2, d=64, NB=8, fill=0x7FC0)
    K = rng.standard_normal((1, 2, 1, 64)); V = rng.standard_normal((1, 2, 1, 64))
    blocks = np.array([3], dtype=np.int32)
    oracle.scatter(kv, dims, blocks, 0, bf16_bits(K), bf16_bits(V))
    q = bf16_bits(rng.standard_normal((1, 8, 64)))
    out = oracle.attention(kv, dims, 0, 8, [blocks], [1], q)
    Vb = bits_to_f64(bf16_bits(V))
    for h in range(8):
        assert np.array_equal(out[0, h], Vb[0, h // 4, 0])


@pytest.mark.parametrize("n", [1, 15, 16, 17, 64, 130, 255, 700])
def test_p2_zero_query_gives_mean_of_v(n):
    dims, kv = make_pool(Hkv=2, d=64, NB=64, fill=0x7FC0)
    rng = np.random.default_rng(n)
    K = rng.standard_normal((1, 2, n, 64))
    V = np.zeros((1, 2, n, 64)); V[..., 0] = 1.0; V[..., 1] = (np.arange(n) % 256)[None, None, :]
    V[..., 2] = (np.arange(n) % 7 == 3)
    blocks = perm_blocks(rng, 64, [n])[0]
    oracle.scatter(kv, dims, blocks, 0, bf16_bits(K), bf16_bits(V))
    out = oracle.attention(kv, dims, 0, 8, [blocks], [n], np.zeros((1, 8, 64), np.uint16))
    for h in range(8):
        assert abs(out[0, h, 0] - 1.0) < 1e-12
        assert abs(out[0, h, 1] - np.mean(np.arange(n) % 256)) < 1e-9
        assert abs(out[0, h, 2] - np.mean(np.arange(n) % 7 == 3)) < 1e-12
        assert np.all(out[0, h, 3:] == 0)


def test_p5_weights_sum_to_one_and_v_ones():
    rng = np.random.default_rng(5)
    lens = [17, 64, 130, 255]
    dims, kv = make_pool(Hkv=2, d=64, NB=128, fill=0x7FC0)
    blocks = perm_blocks(rng, 128, lens)
    K = [rng.standard_normal((1, 2, n, 64)) * 3 for n in lens]
    V = [np.ones((1, 2, n, 64)) for n in lens]
    fill_requests(dims, kv, blocks, K, V)
    q = bf16_bits(rng.standard_normal((4, 8, 64)) * 3)
    out, wsum = oracle.attention(kv, dims, 0, 8, blocks, lens, q, return_wsum=True)
    assert np.max(np.abs(wsum - 1)) < 1e-12
    assert np.max(np.abs(out - 1)) < 1e-12


def test_p8_gqa_head_mapping():
    rng = np.random.default_rng(8)
    for Hq, Hkv in [(8, 2), (32, 8), (64, 8), (4, 4)]:
        G = Hq // Hkv
        dims, kv = make_pool(Hkv=Hkv, d=64, NB=16)
        n = 40
        K = rng.standard_normal((1, Hkv, n, 64))
        V = np.broadcast_to(np.arange(Hkv, dtype=np.float64)[None, :, None, None], (1, Hkv, n, 64)).copy()
        blocks = perm_blocks(rng, 16, [n])[0]
        oracle.scatter(kv, dims, blocks, 0, bf16_bits(K), bf16_bits(V))
        out = oracle.attention(kv, dims, 0, Hq, [blocks], [n], bf16_bits(rng.standard_normal((1, Hq, 64))))
        for h in range(Hq):
            assert np.allclose(out[0, h], h // G, atol=1e-12)


# --------------------------------------------------------------------------------------------
# P3: needle — addressing at every block boundary
# --------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [17, 130, 255, 1040])
def test_p3_needle_positions(n):
    d, bs = 64, 16
    rng = np.random.default_rng(n)
    positions = sorted({0, 15, 16, 31, 32, n - 1, (n - 1) // bs * bs, max(0, (n - 1) // bs * bs - 1), n // 2} & set(range(n)))
    qf = np.zeros(d); qf[0] = 8.0                      # |q|^2 = 64, scale = 1/8 -> score = K[t][0]
    for pos in positions:
        dims, kv = make_pool(Hkv=1, d=d, NB=80, fill=0x7FC0)
        K = np.zeros((1, 1, n, d)); K[0, 0, :, 1:] = rng.standard_normal((n, d - 1))  # orthogonal noise
        K[0, 0, pos, 0] = 64.0                       # needle score 64 vs 0 for every other token
        V = np.zeros((1, 1, n, d)); V[0, 0, :, 0] = np.arange(n) % 128; V[0, 0, :, 1] = np.arange(n) // 128
        blocks = perm_blocks(rng, 80, [n])[0]
        oracle.scatter(kv, dims, blocks, 0, bf16_bits(K), bf16_bits(V))
        out = oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(qf)[None, None])
        bound = (n - 1) * math.exp(-64.0) * 128
        assert abs(out[0, 0, 0] - pos % 128) <= bound + 1e-12
        assert abs(out[0, 0, 1] - pos // 128) <= bound + 1e-12


# --------------------------------------------------------------------------------------------
# P4: physical placement does not matter
# --------------------------------------------------------------------------------------------

def test_p4_block_permutation_invariance():
    lens = [17, 64, 130, 255]
    rng = np.random.default_rng(4)
    K = [rng.standard_normal((1, 2, n, 64)) for n in lens]
    V = [rng.standard_normal((1, 2, n, 64)) for n in lens]
    q = bf16_bits(rng.standard_normal((4, 8, 64)))
    outs = []
    for seed, fill in [(10, 0), (11, 0x7FC0), (12, 0xFF80)]:       # 0, NaN, -inf sentinels
        dims, kv = make_pool(Hkv=2, d=64, NB=128, fill=fill)
        blocks = perm_blocks(np.random.default_rng(seed), 128, lens)
        fill_requests(dims, kv, blocks, K, V)
        outs.append(oracle.attention(kv, dims, 0, 8, blocks, lens, q))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    assert np.all(np.isfinite(outs[0]))


# --------------------------------------------------------------------------------------------
# P9 + brute force: library routines on independently gathered rows
# --------------------------------------------------------------------------------------------

@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 8, 128), (4, 4, 128), (64, 8, 128)])
def test_p9_matches_torch_sdpa_and_scipy(Hq, Hkv, d):
    rng = np.random.default_rng(Hq * 1000 + d)
    lens = [1, 17, 64, 130, 255, 33]
    L = 2
    dims, kv = make_pool(L=L, Hkv=Hkv, d=d, NB=64, fill=0x7FC0)
    blocks = perm_blocks(rng, 64, lens)
    K = [rng.standard_normal((L, Hkv, n, d)) for n in lens]
    V = [rng.standard_normal((L, Hkv, n, d)) for n in lens]
    kb, vb = fill_requests(dims, kv, blocks, K, V)
    qb = bf16_bits(rng.standard_normal((len(lens), Hq, d)))
    G = Hq // Hkv
    for layer in range(L):
        out, wsum = oracle.attention(kv, dims, layer, Hq, blocks, lens, qb, return_wsum=True)
        assert np.max(np.abs(wsum - 1)) < 1e-12
        for r, n in enumerate(lens):
            Kr = torch.from_numpy(bits_to_f64(kb[r][layer]))          # [Hkv][n][d]
            Vr = torch.from_numpy(bits_to_f64(vb[r][layer]))
            qr = torch.from_numpy(bits_to_f64(qb[r]))                 # [Hq][d]
            Ke = Kr.repeat_interleave(G, dim=0)                       # query head h <- KV head h // G
            Ve = Vr.repeat_interleave(G, dim=0)
            ref = torch.nn.functional.scaled_dot_product_attention(qr[:, None, :], Ke, Ve)  # scale 1/sqrt(d)
            assert torch.allclose(torch.from_numpy(out[r]), ref[:, 0, :], rtol=0, atol=1e-10)
            # scipy softmax + numpy matmul
            for h in range(Hq):
                s = (Kr[h // G].numpy() @ qr[h].numpy()) / math.sqrt(d)
                want = scipy.special.softmax(s) @ Vr[h // G].numpy()
                assert np.allclose(out[r, h], want, rtol=0, atol=1e-10)


def test_explicit_scale_is_used():
    """A1: scale is an argument; doubling it equals doubling q (exact in bf16)."""
    rng = np.random.default_rng(3)
    dims, kv = make_pool(Hkv=1, d=64, NB=8)
    n = 50
    blocks = perm_blocks(rng, 8, [n])[0]
    oracle.scatter(kv, dims, blocks, 0, bf16_bits(rng.standard_normal((1, 1, n, 64))),
                   bf16_bits(rng.standard_normal((1, 1, n, 64))))
    qf = bits_to_f64(bf16_bits(rng.standard_normal((1, 1, 64))))
    a = oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(qf), scale=0.25)
    b = oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(2 * qf), scale=0.125)
    c = oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(qf), scale=None)
    assert np.allclose(a, b, atol=1e-13)
    assert not np.allclose(c, a, atol=1e-6)          # default scale 1/sqrt(64) = 1/8 differs from 1/4
    d = oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(qf), scale=1 / 8)
    assert np.array_equal(c, d)


# --------------------------------------------------------------------------------------------
# P6: chunk + combine == unsplit
# --------------------------------------------------------------------------------------------

def test_p6_split_and_combine_identity():
    rng = np.random.default_rng(6)
    n, d = 700, 128
    dims, kv = make_pool(Hkv=2, d=d, NB=64, fill=0x7FC0)
    blocks = perm_blocks(rng, 64, [n])[0]
    oracle.scatter(kv, dims, blocks, 0, bf16_bits(rng.standard_normal((1, 2, n, d)) * 2),
                   bf16_bits(rng.standard_normal((1, 2, n, d))))
    qb = bf16_bits(rng.standard_normal((1, 4, d)) * 2)
    full = oracle.attention(kv, dims, 0, 4, [blocks], [n], qb)
    scale = 1 / math.sqrt(d)
    for cuts in ([0, n], [0, 1, n], [0, 16, 17, 256, 699, n], [0, 512, n], list(range(0, n, 64)) + [n]):
        for h in range(4):
            parts = [oracle.chunk(kv, dims, 0, h // 2, blocks, a, b, qb[0, h], scale) for a, b in zip(cuts, cuts[1:])]
            got = oracle.combine([p[0] for p in parts], [p[1] for p in parts], np.stack([p[2] for p in parts]))
            assert np.allclose(got, full[0, h], rtol=0, atol=1e-12)


# --------------------------------------------------------------------------------------------
# P13: shift invariance, large scores
# --------------------------------------------------------------------------------------------

def test_p13_shift_invariance_and_no_overflow():
    rng = np.random.default_rng(13)
    n, d = 100, 64
    K = np.zeros((1, 1, n, d)); K[..., :32] = rng.standard_normal((1, 1, n, 32))
    V = rng.standard_normal((1, 1, n, d))
    qf = np.zeros((1, 1, d)); qf[..., :32] = rng.standard_normal((1, 1, 32))
    outs = []
    for shift in [0.0, 1.0, -4.0, 640.0]:       # adds 8*shift... to every score: q[40]=8, K[:,40]=shift
        dims, kv = make_pool(Hkv=1, d=d, NB=8)
        Ks = K.copy(); Ks[..., 40] = shift
        qs = qf.copy(); qs[..., 40] = 8.0
        blocks = np.arange(7, dtype=np.int32)
        oracle.scatter(kv, dims, blocks, 0, bf16_bits(Ks), bf16_bits(V))
        outs.append(oracle.attention(kv, dims, 0, 1, [blocks], [n], bf16_bits(qs)))
    for o in outs[1:]:
        assert np.all(np.isfinite(o))
        assert np.allclose(o, outs[0], rtol=0, atol=1e-9)
    # one dominating score of +/- 5000 before scaling: still finite, picks / ignores that token
    dims, kv = make_pool(Hkv=1, d=d, NB=8)
    Kb = np.zeros((1, 1, n, d)); Kb[0, 0, 7, 0] = 5000.0; Kb[0, 0, 9, 0] = -5000.0
    oracle.scatter(kv, dims, np.arange(7, dtype=np.int32), 0, bf16_bits(Kb), bf16_bits(V))
    qb = np.zeros((1, 1, d)); qb[0, 0, 0] = 8.0
    o = oracle.attention(kv, dims, 0, 1, [np.arange(7, dtype=np.int32)], [n], bf16_bits(qb))
    assert np.allclose(o[0, 0], bits_to_f64(bf16_bits(V))[0, 0, 7], atol=1e-12)


# --------------------------------------------------------------------------------------------
# P10, P12: scatter / gather
# --------------------------------------------------------------------------------------------

def numpy_scatter(kv6, blocks, start, k_src, v_src, layer_begin, bs):
    """Independent statement with numpy fancy indexing (a library routine, not loops)."""
    lc, Hkv, n, d = k_src.shape
    pos = start + np.arange(n)
    blk, slot = np.asarray(blocks)[pos // bs], pos % bs
    for ll in range(lc):
        kv6[layer_begin + ll, blk, :, 0, slot, :] = np.transpose(k_src[ll], (1, 0, 2))
        kv6[layer_begin + ll, blk, :, 1, slot, :] = np.transpose(v_src[ll], (1, 0, 2))


@pytest.mark.parametrize("sentinel", [0x0000, 0x7FC0, 0xABCD])
def test_p10_scatter_matches_numpy_and_roundtrips(sentinel):
    rng = np.random.default_rng(10)
    lens = [17, 64, 130, 255, 1, 16]
    L, Hkv, d, bs, NB = 3, 2, 64, 16, 128
    dims, kv = make_pool(L=L, Hkv=Hkv, d=d, NB=NB, fill=sentinel)
    ref = np.full(dims.shape(), sentinel, dtype=np.uint16)
    blocks = perm_blocks(rng, NB, lens)
    srcs = []
    for b, n in zip(blocks, lens):
        k = rng.integers(0, 65536, size=(L, Hkv, n, d), dtype=np.uint16)   # arbitrary bit patterns
        v = rng.integers(0, 65536, size=(L, Hkv, n, d), dtype=np.uint16)
        oracle.scatter(kv, dims, b, 0, k, v)
        numpy_scatter(ref, b, 0, k, v, 0, bs)
        srcs.append((k, v))
    assert np.array_equal(kv, ref.reshape(-1))                 # whole slab, incl. untouched sentinel bytes
    used = sum((n + bs - 1) // bs for n in lens)
    untouched = np.setdiff1d(np.arange(NB), np.concatenate(blocks))
    assert untouched.size == NB - used
    assert np.all(kv.reshape(dims.shape())[:, untouched] == sentinel)
    for b, n, (k, v) in zip(blocks, lens, srcs):
        gk, gv = oracle.gather(kv, dims, b, n)
        assert np.array_equal(gk, k) and np.array_equal(gv, v)


def test_p12_append_splits_are_equivalent():
    rng = np.random.default_rng(12)
    L, Hkv, d, NB, n = 2, 2, 64, 32, 77
    dims = oracle.Dims(L, Hkv, d, 16, NB)
    k = rng.integers(0, 65536, size=(L, Hkv, n, d), dtype=np.uint16)
    v = rng.integers(0, 65536, size=(L, Hkv, n, d), dtype=np.uint16)
    blocks = perm_blocks(rng, NB, [n])[0]
    base = oracle.new_slab(dims, 0x7FC0)
    oracle.scatter(base, dims, blocks, 0, k, v)
    for cuts in ([0, 5, n], [0, 16, 32, n], [0, 17, 18, 50, n], list(range(n + 1))):
        kv = oracle.new_slab(dims, 0x7FC0)
        for a, b in zip(cuts, cuts[1:]):
            oracle.scatter(kv, dims, blocks, a, np.ascontiguousarray(k[:, :, a:b]), np.ascontiguousarray(v[:, :, a:b]))
        assert np.array_equal(kv, base)
    # layer-sliced ingest == all layers at once
    kv = oracle.new_slab(dims, 0x7FC0)
    for l in range(L):
        oracle.scatter(kv, dims, blocks, 0, k[l:l + 1], v[l:l + 1], layer_begin=l)
    assert np.array_equal(kv, base)


def test_a11_empty_context_is_an_error():
    dims, kv = make_pool(Hkv=1, d=64, NB=4)
    with pytest.raises(ValueError):
        oracle.attention(kv, dims, 0, 1, [np.zeros(0, np.int32)], [0], np.zeros((1, 1, 64), np.uint16))
