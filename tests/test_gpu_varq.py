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


# ---------------------------------------------------------------------------------------------
# paged_varlen_step: the new tokens' K/V written into the pool as the step goes
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("opts", [dict(), dict(min_chunk_blocks=1, items_per_slot=1024), dict(pdl=0)])
@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 8, 128), (32, 32, 128)])
def test_varlen_step_equals_ingest_then_attention_and_oracle(Hq, Hkv, d, opts):
    """Two steps over three layers of a mixed batch: decode rows (one new token), fresh in-place prefills (requests that
    do not exist before the step) and a chunked prefill on top of a stored prefix.  The fused call == layer-sliced
    kv_ingest + paged_varlen_attention on a twin pool, bit for bit (pool and outputs), the pool == the
    oracle's scatter over the whole slab, the outputs == oracle_attention_varq."""
    L = 3
    prefix = [40, 0, 255, 16, 0, 700]                 # stored before the first step (0: the request does not exist yet)
    steps = [[1, 33, 1, 48, 130, 1], [1, 1, 1, 17, 1, 1]]
    w = W.Workload("varq_step", L, Hq, Hkv, d, len(prefix), None, 777, max_len=1024)
    nb = sum((p + sum(s[i] for s in steps) + 15) // 16 for i, p in enumerate(prefix)) + 8
    pools = [make_pool(w, nb, max_requests=16, alloc_seed=13) for _ in range(2)]
    for p in pools:
        apply_options(p, opts)
    ids = list(range(40, 40 + len(prefix)))
    have = [(u, n) for u, n in zip(ids, prefix) if n > 0]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in have]
    for p in pools:
        p.ingest([u for u, _ in have], [s[0] for s in srcs], [s[1] for s in srcs])
    slab = oracle_slab(pools[0])
    for u, n in have:
        oracle_ingest(slab, pools[0], w, u, 0, n)
    lens = list(prefix)
    for step, q_lens in enumerate(steps):
        new = [kv_src(w, u, n, n + ql, DEV) for u, n, ql in zip(ids, lens, q_lens)]       # [L][Hkv][ql][d] each
        for layer in range(L):                         # twin pool: kv_ingest(layer 0) makes the reservation, layers 1.. continue it
            q = W.q_values(w.seed, step, layer, sum(q_lens), Hq, d, DEV)
            kl = [k[layer].contiguous() for k, _ in new]
            vl = [v[layer].contiguous() for _, v in new]
            n0 = pools[0].launches
            out_a = pools[0].varlen_step(layer, ids, q_lens, q, kl, vl, reserve=(layer == 0))
            assert pools[0].launches - n0 == 2                                            # scatter + attention
            B.kv_ingest(pools[1].handle, ids, q_lens, kl, vl, layer, 1)
            out_b = pools[1].varlen_attention(layer, ids, q_lens, q)
            torch.cuda.synchronize()
            assert torch.equal(out_a.view(torch.int16), out_b.view(torch.int16))
            if layer == 0:
                for u, n, ql in zip(ids, lens, q_lens):
                    oracle_ingest(slab, pools[0], w, u, n, n + ql)
            compare_attention(out_a, oracle_varq(slab, pools[0], layer, ids, q_lens, q))
        lens = [n + ql for n, ql in zip(lens, q_lens)]
        assert np.array_equal(pool_bits(pools[0]), slab), "the step's rows are not where the oracle puts them"
        assert torch.equal(pools[0].slab[: pools[0].kv_bytes], pools[1].slab[: pools[1].kv_bytes])
    assert pools[0].counter("plans_uploaded") == len(steps)                               # one plan per step, three layers each


def test_varlen_step_errors_change_nothing():
    w = W.Workload("varq_step_err", 2, 8, 2, 64, 2, None, 5, max_len=512)
    pool = make_pool(w, 11, max_requests=4, alloc_seed=0)                                # 3 blocks used below, 8 free
    ids = [900, 901]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, [32, 16])]
    pool.ingest(ids, [s_[0] for s_ in srcs], [s_[1] for s_ in srcs])
    torch.cuda.synchronize()
    q = torch.zeros((400, 8, 64), dtype=torch.bfloat16, device=DEV)
    kn = [torch.zeros((2, 200, 64), dtype=torch.bfloat16, device=DEV) for _ in range(2)]
    stats, bits = pool.stats(), pool_bits(pool).copy()
    for a_ids, ql, layer, reserve, status in [
            ([900, 901], [200, 200], 0, True, B.KV_ERR_NO_BLOCKS),         # 2 x 13 new blocks, 8 free
            ([7, 900], [1, 1], 1, False, B.KV_ERR_UNKNOWN_REQUEST),
            ([900, 901], [1, 1], 1, True, B.KV_ERR_INVALID),                # reserve needs layer 0
            ([900, 901], [1, 1], 0, False, B.KV_ERR_INVALID),               # no one-token reservation to continue
            ([900, 901], [0, 1], 0, True, B.KV_ERR_INVALID),
            ([900, 900], [1, 1], 0, True, B.KV_ERR_INVALID)]:
        with pytest.raises(B.KVError) as e:
            pool.varlen_step(layer, a_ids, ql, q[: max(sum(ql), 1)].contiguous(), [k[:, : max(n, 1)].contiguous() for k, n in zip(kn, ql)],
                             [k[:, : max(n, 1)].contiguous() for k, n in zip(kn, ql)], reserve=reserve)
        assert e.value.status == status, (a_ids, ql, layer, reserve)
        assert pool.stats() == stats and pool.block_table(900)[1] == 32 and pool.block_table(901)[1] == 16
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), bits)
    out = pool.varlen_step(0, ids, [1, 3], q[:4].contiguous(), [kn[0][:, :1].contiguous(), kn[1][:, :3].contiguous()],
                           [kn[0][:, :1].contiguous(), kn[1][:, :3].contiguous()], reserve=True)   # still works afterwards
    torch.cuda.synchronize()
    assert pool.block_table(900)[1] == 33 and pool.block_table(901)[1] == 19 and np.all(np.isfinite(bits_to_f64(bits_of(out))))


def test_varlen_step_fp8_pool_equals_ingest_then_attention():
    """FP8 pool: the fused call quantises the new rows exactly as kv_ingest does (same bytes over the whole pool) and
    returns the bits of paged_varlen_attention."""
    import paper_2511_20982_b200 as kv
    L, Hq, Hkv, d = 2, 32, 8, 128
    prefix, q_lens = [300, 0, 17], [1, 90, 40]
    w = W.Workload("varq_step_fp8", L, Hq, Hkv, d, 3, None, 31, max_len=512)
    pools = []
    for _ in range(2):
        cfg = kv.PoolConfig(num_layers=L, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d, num_blocks=40, max_requests=8,
                            max_blocks_per_request=32, alloc_seed=21, kv_dtype=B.KV_DTYPE_FP8_E4M3)
        p = kv.KVPool(cfg, device=DEV)
        p.slab[: p.kv_bytes].fill_(0xFF)
        pools.append(p)
    ids = [5, 6, 7]
    have = [(u, n) for u, n in zip(ids, prefix) if n > 0]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in have]
    for p in pools:
        p.ingest([u for u, _ in have], [s[0] for s in srcs], [s[1] for s in srcs])
    new = [kv_src(w, u, n, n + ql, DEV) for u, n, ql in zip(ids, prefix, q_lens)]
    for layer in range(L):
        q = W.q_values(w.seed, 0, layer, sum(q_lens), Hq, d, DEV)
        kl = [k[layer].contiguous() for k, _ in new]
        vl = [v[layer].contiguous() for _, v in new]
        out_a = pools[0].varlen_step(layer, ids, q_lens, q, kl, vl, reserve=(layer == 0))
        B.kv_ingest(pools[1].handle, ids, q_lens, kl, vl, layer, 1)
        out_b = pools[1].varlen_attention(layer, ids, q_lens, q)
        torch.cuda.synchronize()
        assert torch.equal(out_a.view(torch.int16), out_b.view(torch.int16))
        assert np.all(np.isfinite(bits_to_f64(bits_of(out_a))))
    assert torch.equal(pools[0].slab[: pools[0].kv_bytes], pools[1].slab[: pools[1].kv_bytes])
