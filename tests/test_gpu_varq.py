"""-m gpu parity of paged_varlen_attention (in-place prefill of
ultra-short requests merged with decoding) against oracle_attention_varq, element by element,
through the C-ABI.  Mixed batches of decode rows (q_len = 1), fresh prefill rows (q_len = len)
and chunked prefill rows (0 < q_len < len); every GQA group size the kernel packs differently
(G = 1: 8 query tokens per tile ... G = 8: one); contexts long enough to be split into chunks
(a later chunk is then invisible to the earlier query tokens of a tile: the -inf guards)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from gpu_harness import DEV, apply_options, compare_attention, dims_of, kv_src, make_pool, oracle_ingest, oracle_slab, pool_bits
from helpers import bf16_bits, bits_of, bits_to_f64

pytestmark = pytest.mark.gpu

MODES = [dict(), dict(min_chunk_blocks=1, items_per_slot=1024), dict(min_chunk_blocks=3, items_per_slot=1024),
         dict(min_chunk_blocks=2, items_per_slot=2, ctas_per_sm=1), dict(ring=2), dict(pdl=0), dict(pdl=0, min_chunk_blocks=1, items_per_slot=1024),
         dict(tma=1), dict(tma=1, min_chunk_blocks=1, items_per_slot=1024)]
SHAPES = [(8, 2, 64), (32, 32, 128), (64, 8, 128), (6, 2, 64), (5, 1, 128), (4, 2, 128)]   # G = 4, 1, 8, 3, 5, 2


def oracle_varq(slab, pool, layer, ids, q_lens, q, scale=None):
    lists, lens = zip(*[pool.block_table(i) for i in ids])
    return oracle.attention_varq(slab, dims_of(pool), layer, pool.cfg.num_q_heads, list(lists), list(lens), q_lens,
                                 bits_of(q), scale=scale)


def build(Hq, Hkv, d, lens, opts, L=1, seed=4242, alloc_seed=9):
    w = W.Workload("varq", L, Hq, Hkv, d, len(lens), None, seed, max_len=max(lens) + 16)
    pool = make_pool(w, sum((n + 15) // 16 for n in lens) + 8, max_requests=len(lens) + 4, alloc_seed=alloc_seed)
    apply_options(pool, opts)
    slab = oracle_slab(pool)
    ids = list(range(900, 900 + len(lens)))
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    for uid, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, uid, 0, n)
    return w, pool, slab, ids


@pytest.mark.parametrize("opts", MODES)
@pytest.mark.parametrize("Hq,Hkv,d", SHAPES)
def test_mixed_batch_matches_oracle(Hq, Hkv, d, opts):
    lens = [17, 64, 130, 255, 1, 16, 33, 700, 1100, 5, 48, 100]
    q_lens = [17, 1, 130, 7, 1, 16, 1, 1, 300, 5, 31, 100]          # fresh / decode / chunked prefill rows
    w, pool, slab, ids = build(Hq, Hkv, d, lens, opts)
    q = W.q_values(w.seed, 3, 0, sum(q_lens), Hq, d, DEV)
    out = pool.varlen_attention(0, ids, q_lens, q)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab), "attention modified the pool"
    want = oracle_varq(slab, pool, 0, ids, q_lens, q)
    compare_attention(out, want)


@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 32, 128), (64, 8, 128)])
def test_qlen1_equals_decode_call(Hq, Hkv, d):
    """With every q_len = 1 the call is the decode step: same bits as paged_decode_attention when the
    plans coincide (unsplit units), within tolerance of the oracle always."""
    lens = [17, 64, 130, 255, 1, 2000]
    w, pool, slab, ids = build(Hq, Hkv, d, lens, dict(min_chunk_blocks=4096))
    q = W.q_values(w.seed, 5, 0, len(lens), Hq, d, DEV)
    a = pool.attention(0, ids, q)
    b = pool.varlen_attention(0, ids, [1] * len(lens), q)
    torch.cuda.synchronize()
    assert torch.equal(a.view(torch.int16), b.view(torch.int16))
    compare_attention(b, oracle_varq(slab, pool, 0, ids, [1] * len(lens), q))


def test_structured_running_mean_and_first_token():
    """q = 0 -> row i is the mean of V over tokens 0..P_i (closed form, counts every visible token once
    across block, tile and chunk boundaries); first row of a fresh prefill returns V_0's bits."""
    Hq, Hkv, d, n, p0 = 8, 2, 64, 200, 37
    w = W.Workload("varq_s", 1, Hq, Hkv, d, 2, None, 1, max_len=n + 16)
    for opts in MODES:
        pool = make_pool(w, 40, alloc_seed=3)
        apply_options(pool, opts)
        v = np.zeros((1, Hkv, n, d)); v[..., 0] = 1.0
        v[0, :, :, 1] = (np.arange(n) % 256)[None, :]
        k = np.random.default_rng(0).standard_normal((1, Hkv, n, d))
        tb = lambda x: torch.from_numpy(bf16_bits(x).view(np.int16).copy()).view(torch.bfloat16).to(DEV)
        pool.ingest([1, 2], [tb(k), tb(k)], [tb(v), tb(v)])
        ql = [n - p0, n]
        out = pool.varlen_attention(0, [1, 2], ql, torch.zeros((sum(ql), Hq, d), dtype=torch.bfloat16, device=DEV))
        got = bits_to_f64(bits_of(out))
        for base, q_len, start in ((0, ql[0], p0), (ql[0], ql[1], 0)):
            P = start + np.arange(q_len)
            assert np.all(np.abs(got[base:base + q_len, :, 0] - 1.0) <= 2.0 ** -8)
            assert np.all(np.abs(got[base:base + q_len, :, 1] - (P / 2.0)[:, None]) <= (P / 2.0)[:, None] * 2.0 ** -8 + 1e-6)
            assert np.all(got[base:base + q_len, :, 2:] == 0.0)
        # V_0 exactly: second request, first row, a random q
        q = W.q_values(7, 0, 0, sum(ql), Hq, d, DEV)
        out = pool.varlen_attention(0, [1, 2], ql, q)
        assert np.array_equal(bits_of(out)[ql[0]], np.repeat(bf16_bits(v)[0, :, 0], Hq // Hkv, axis=0))
        pool.close()


def test_layers_and_plan_cache():
    """Layer-sliced in-place prefill as a model would run it: per layer, ingest that layer's K/V of the new
    tokens, then attend; decode rows appended the same way.  The plan is reused across layers."""
    Hq, Hkv, d, L = 32, 8, 128, 3
    lens0 = [300, 64, 0, 0, 1500]            # stored before the step (0: a fresh ultra-short request)
    add = [1, 1, 40, 100, 1]                 # tokens computed in this step (decode rows: 1)
    w = W.Workload("varq_l", L, Hq, Hkv, d, len(lens0), None, 77, max_len=2048)
    pool = make_pool(w, 200, alloc_seed=5)
    slab = oracle_slab(pool)
    ids = list(range(10, 10 + len(lens0)))
    live = [(u, n) for u, n in zip(ids, lens0) if n]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in live]
    pool.ingest([u for u, _ in live], [s[0] for s in srcs], [s[1] for s in srcs])
    for u, n in live:
        oracle_ingest(slab, pool, w, u, 0, n)
    n_launch = pool.launches
    for l in range(L):
        new = [kv_src(w, u, n, n + a, DEV, layer_begin=l, layer_count=1) for u, n, a in zip(ids, lens0, add)]
        pool.ingest(ids, [s[0] for s in new], [s[1] for s in new], layer_begin=l, layer_count=1)
        q = W.q_values(w.seed, 9, l, sum(add), Hq, d, DEV)
        out = pool.varlen_attention(l, ids, add, q)
        torch.cuda.synchronize()
        if l == 0:
            for u, n, a in zip(ids, lens0, add):
                oracle_ingest(slab, pool, w, u, n, n + a)
        want = oracle_varq(slab, pool, l, ids, add, q)
        compare_attention(out, want)
    assert np.array_equal(pool_bits(pool), slab)
    assert pool.launches - n_launch == 2 * L


def test_errors_change_nothing():
    w, pool, slab, ids = build(8, 2, 64, [20, 30], dict())
    q = torch.zeros((64, 8, 64), dtype=torch.bfloat16, device=DEV)
    for bad_ids, ql, status in [([900, 901], [21, 1], B.KV_ERR_INVALID), ([900, 901], [0, 1], B.KV_ERR_INVALID),
                                ([900, 900], [1, 1], B.KV_ERR_INVALID), ([900, 7], [1, 1], B.KV_ERR_UNKNOWN_REQUEST)]:
        with pytest.raises(B.KVError) as e:
            pool.varlen_attention(0, bad_ids, ql, q[: sum(ql)].contiguous())
        assert e.value.status == status
    out = pool.varlen_attention(0, ids, [20, 30], q[:50].contiguous())   # still works afterwards
    torch.cuda.synchronize()
    assert np.all(np.isfinite(bits_to_f64(bits_of(out))))
