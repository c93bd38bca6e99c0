"""GPU parity of the fused decode step (paged_decode_step: a3 + a4 + a5 in one launch), the
host-buffer entry points and the per-kernel profiling counters, against the oracle."""
import numpy as np
import pytest
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from gpu_harness import (apply_options, DEV, compare_attention, dims_of, kv_src, make_pool, oracle_attention, oracle_ingest,
                         oracle_slab, pool_bits)
from helpers import bits_of

pytestmark = pytest.mark.gpu

MODES = [dict(), dict(fuse_combine=0), dict(min_chunk_blocks=1, items_per_slot=1024),
         dict(min_chunk_blocks=3, items_per_slot=1024, fuse_combine=0),
         dict(min_chunk_blocks=1, items_per_slot=2), dict(min_chunk_blocks=5, items_per_slot=1),
         dict(ring=2), dict(pdl=0), dict(pdl=0, min_chunk_blocks=1, items_per_slot=1024), dict(ring=2, min_chunk_blocks=3, items_per_slot=1024),
         dict(tma=1), dict(tma=1, min_chunk_blocks=1, items_per_slot=1024), dict(tma=1, min_chunk_blocks=3, items_per_slot=2, fuse_combine=0), dict(side_upload=0), dict(side_upload=0, min_chunk_blocks=1, items_per_slot=1024)]
SHAPES = [(8, 2, 64), (32, 32, 128), (64, 8, 128)]
# lengths BEFORE the first step: fill a block (15 -> 16), open a new one (16 -> 17), mid-block, one token,
# empty (0 -> 1), exact multiples, and contexts long enough to be split into several chunks
LENS = [15, 16, 17, 1, 0, 31, 32, 255, 256, 1039, 1040, 2047, 700]


def new_rows(w, ids, lens, L, device):
    """K/V rows of the token each request appends this step (its logical position = current length)."""
    k = W.kv_values_at(w.seed, W.KIND_K, ids, lens, w.num_kv_heads, w.head_dim, 0, L, device)
    v = W.kv_values_at(w.seed, W.KIND_V, ids, lens, w.num_kv_heads, w.head_dim, 0, L, device)
    return k, v


def oracle_append(slab, pool, ids, lens, kc, vc):
    """Scatter row i of kc / vc ([L][B][Hkv][d], cpu bf16) at position lens[i] of request ids[i]."""
    for i, (uid, n) in enumerate(zip(ids, lens)):
        blocks, _ = pool.block_table(uid)
        oracle.scatter(slab, dims_of(pool), blocks, n, bits_of(kc[:, i].unsqueeze(2)), bits_of(vc[:, i].unsqueeze(2)))


@pytest.mark.parametrize("opts", MODES)
@pytest.mark.parametrize("Hq,Hkv,d", SHAPES)
def test_fused_step_matches_oracle_and_leaves_pool_bit_exact(Hq, Hkv, d, opts):
    L = 2
    w = W.Workload("step", L, Hq, Hkv, d, len(LENS), None, 4242, max_len=2048 + 64)
    ids = list(range(300, 300 + len(LENS)))
    lens = list(LENS)
    pool = make_pool(w, sum((n + 15) // 16 + 1 for n in lens) + 8, alloc_seed=11)
    apply_options(pool, opts)
    slab = oracle_slab(pool)
    have = [(u, n) for u, n in zip(ids, lens) if n > 0]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in have]
    pool.ingest([u for u, _ in have], [s[0] for s in srcs], [s[1] for s in srcs])
    for u, n in have:
        oracle_ingest(slab, pool, w, u, 0, n)
    for step in range(3):
        pool.reserve(ids, [1] * len(ids))                                       # a1 for this step
        kd, vd = new_rows(w, ids, lens, L, DEV)
        kc, vc = new_rows(w, ids, lens, L, "cpu")
        oracle_append(slab, pool, ids, lens, kc, vc)
        lens = [n + 1 for n in lens]
        before = pool.launches
        for layer in range(L):
            q = W.q_values(w.seed, step, layer, len(ids), Hq, d, DEV)
            out = pool.decode_step(layer, ids, q, kd[layer], vd[layer])
            compare_attention(out, oracle_attention(slab, pool, layer, ids, q))
        per_layer = 1 if opts.get("fuse_combine", 1) else 2
        assert pool.launches - before == per_layer * L                          # one launch per layer when fused
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)                                # appended rows only, bit-exact
    # the device block_table mirror saw every block the fused steps opened: the unfused path agrees
    q = W.q_values(w.seed, 9, 1, len(ids), Hq, d, DEV)
    compare_attention(pool.attention(1, ids, q), oracle_attention(slab, pool, 1, ids, q))
    # and the gather kernel (which also reads the mirror's source of truth) round-trips
    k, v = pool.gather(ids[1])
    want_k, want_v = oracle.gather(slab, dims_of(pool), pool.block_table(ids[1])[0], lens[1])
    assert np.array_equal(bits_of(k), want_k) and np.array_equal(bits_of(v), want_v)


def test_fused_step_is_bitwise_the_unfused_path():
    """Same seeded inputs through kv_ingest(n=1) + paged_decode_attention and through paged_decode_step:
    identical pools; outputs agree to bf16 rounding (the fused unit visits its last tile first, so the
    fp32 accumulation order differs)."""
    w = W.CONFIGS["cfg2_7b_mha"].scaled(batch=10)
    lens0 = [int(x) for x in w.draw_lengths()]
    lens0[:3] = [511, 512, 2047]
    ids = list(range(10))
    outs, pools = [], []
    for fused in (False, True):
        lens = list(lens0)
        pool = make_pool(w, sum((n + 20) // 16 + 1 for n in lens), alloc_seed=w.seed)
        srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, lens)]
        pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
        got = []
        for step in range(3):
            kd, vd = new_rows(w, ids, lens, 1, DEV)
            q = W.q_values(w.seed, step, 0, len(ids), w.num_q_heads, w.head_dim, DEV)
            if fused:
                pool.reserve(ids, [1] * len(ids))
                got.append(pool.decode_step(0, ids, q, kd[0], vd[0]))
            else:
                pool.ingest(ids, [kd[:, i].unsqueeze(2).contiguous() for i in range(len(ids))],
                            [vd[:, i].unsqueeze(2).contiguous() for i in range(len(ids))])
                got.append(pool.attention(0, ids, q))
            lens = [n + 1 for n in lens]
        torch.cuda.synchronize()
        outs.append([bits_of(o) for o in got])
        pools.append(pool_bits(pool))
    assert np.array_equal(pools[0], pools[1])
    from helpers import bits_to_f64
    for a, b in zip(*outs):
        assert np.max(np.abs(bits_to_f64(a) - bits_to_f64(b))) <= 2e-3


def test_fused_step_needs_a_one_token_reservation():
    w = W.Workload("err", 1, 8, 2, 64, 2, None, 1, max_len=256)
    pool = make_pool(w, 64)
    ids = [1, 2]
    srcs = [kv_src(w, u, 0, 20, DEV) for u in ids]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    q = W.q_values(1, 0, 0, 2, 8, 64, DEV)
    kn, vn = new_rows(w, ids, [20, 20], 1, DEV)
    before = pool_bits(pool).copy()
    with pytest.raises(kv.KVError) as e:                                         # last reservation was 20 tokens
        pool.decode_step(0, ids, q, kn[0], vn[0])
    assert e.value.status == B.KV_ERR_INVALID
    pool.reserve(ids, [1, 2])
    with pytest.raises(kv.KVError) as e:                                         # one request reserved two tokens
        pool.decode_step(0, ids, q, kn[0], vn[0])
    assert e.value.status == B.KV_ERR_INVALID
    with pytest.raises(kv.KVError) as e:
        B.paged_decode_step(pool.handle, 0, ids, q.data_ptr(), 0, vn.data_ptr(), q.data_ptr())
    assert e.value.status == B.KV_ERR_INVALID
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), before)
    pool.reserve(ids, [1, 1])
    pool.decode_step(0, ids, q, kn[0], vn[0])                                    # now fine


def test_host_buffer_entry_points():
    """kv_ingest_host / paged_decode_attention_host / paged_decode_step_host: pinned host tensors in,
    pinned host output back; same bits as the device-pointer calls."""
    w = W.Workload("host", 2, 32, 8, 128, 3, None, 77, max_len=1024)
    lens, ids = [100, 333, 48], [5, 6, 7]
    pool = make_pool(w, 128, alloc_seed=5)
    slab = oracle_slab(pool)
    L, Hkv, d = 2, 8, 128
    # requests 0 and 1 adjacent in one pinned buffer (exercises the merged copy), request 2 on its own
    tok = L * Hkv * d
    big_k = torch.empty((lens[0] + lens[1]) * tok, dtype=torch.bfloat16).pin_memory()
    big_v = torch.empty_like(big_k).pin_memory()
    hk, hv = [], []
    off = 0
    for u, n in zip(ids[:2], lens[:2]):
        k, v = kv_src(w, u, 0, n, "cpu")
        big_k[off:off + n * tok] = k.reshape(-1); big_v[off:off + n * tok] = v.reshape(-1)
        hk.append(big_k.data_ptr() + off * 2); hv.append(big_v.data_ptr() + off * 2)
        off += n * tok
    k2, v2 = (t.pin_memory() for t in kv_src(w, ids[2], 0, lens[2], "cpu"))
    hk.append(k2.data_ptr()); hv.append(v2.data_ptr())
    need = sum(2 * ((n * tok * 2 + 255) // 256 * 256) for n in lens)
    staging = torch.empty(need, dtype=torch.uint8, device=DEV)
    s = torch.cuda.current_stream().cuda_stream
    with pytest.raises(kv.KVError) as e:
        B.kv_ingest_host(pool.handle, ids, lens, hk, hv, 0, L, staging.data_ptr(), need - 256, s)
    assert e.value.status == B.KV_ERR_INVALID and pool.stats()["live_requests"] == 0
    B.kv_ingest_host(pool.handle, ids, lens, hk, hv, 0, L, staging.data_ptr(), need, s)
    for u, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, u, 0, n)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)

    q = W.q_values(77, 0, 1, 3, 32, 128, "cpu").pin_memory()
    out = torch.empty_like(q).pin_memory()
    st2 = torch.empty(1 << 20, dtype=torch.uint8, device=DEV)
    B.paged_decode_attention_host(pool.handle, 1, ids, q.data_ptr(), out.data_ptr(), 0.0, st2.data_ptr(), st2.numel(), s)
    torch.cuda.synchronize()
    want = oracle_attention(slab, pool, 1, ids, q)
    compare_attention(out, want)
    assert np.array_equal(bits_of(out), bits_of(pool.attention(1, ids, q.to(DEV))))

    pool.reserve(ids, [1, 1, 1])
    kc, vc = new_rows(w, ids, lens, L, "cpu")
    oracle_append(slab, pool, ids, lens, kc, vc)
    kp, vp = kc.pin_memory(), vc.pin_memory()
    for layer in range(L):
        ql = W.q_values(77, 1, layer, 3, 32, 128, "cpu").pin_memory()
        B.paged_decode_step_host(pool.handle, layer, ids, ql.data_ptr(), kp[layer].data_ptr(), vp[layer].data_ptr(),
                                 out.data_ptr(), 0.0, st2.data_ptr(), st2.numel(), s)
        torch.cuda.synchronize()
        compare_attention(out, oracle_attention(slab, pool, layer, ids, ql))
    assert np.array_equal(pool_bits(pool), slab)
    with pytest.raises(kv.KVError) as e:
        B.paged_decode_attention_host(pool.handle, 0, ids, q.data_ptr(), out.data_ptr(), 0.0, st2.data_ptr(), 1024, s)
    assert e.value.status == B.KV_ERR_INVALID


def test_host_ingest_staged_in_groups():
    """kv_ingest_host with host_zero_copy = 0: the copy engine fills the staging buffer group of requests by group of
    requests on the pool's own stream while the previous group is scattered; two calls back to back reuse the
    staging buffer (the second call's copies wait for the first call's scatters).  Whole slab == oracle."""
    L, Hkv, d = 2, 8, 128
    w = W.Workload("stage", L, 32, Hkv, d, 10, None, 91, max_len=8192)
    lens_a, ids_a = [4000, 3000, 4100, 17, 3900, 4200], [1, 2, 3, 4, 5, 6]      # ~150 MB of K + V: three groups
    lens_b, ids_b = [3500, 4500, 1, 2600], [11, 12, 13, 14]
    pool = make_pool(w, sum((n + 15) // 16 for n in lens_a + lens_b) + 8, alloc_seed=3, max_requests=16, max_len=8192)
    pool.set_option("host_zero_copy", 0)
    slab = oracle_slab(pool)
    tok = L * Hkv * d * 2
    need = max(sum(2 * ((n * tok + 255) // 256 * 256) for n in ls) for ls in (lens_a, lens_b))
    staging = torch.empty(need, dtype=torch.uint8, device=DEV)
    s = torch.cuda.current_stream().cuda_stream
    keep = []
    for ids, lens in ((ids_a, lens_a), (ids_b, lens_b)):
        src = [tuple(t.pin_memory() for t in kv_src(w, u, 0, n, "cpu")) for u, n in zip(ids, lens)]
        keep.append(src)
        B.kv_ingest_host(pool.handle, ids, lens, [k.data_ptr() for k, _ in src], [v.data_ptr() for _, v in src], 0, L,
                         staging.data_ptr(), need, s)
    for ids, lens in ((ids_a, lens_a), (ids_b, lens_b)):
        for u, n in zip(ids, lens):
            oracle_ingest(slab, pool, w, u, 0, n)
    torch.cuda.synchronize()
    assert pool.counter("host_ingest_staged") == 2 and pool.counter("host_ingest_zero_copy") == 0
    assert np.array_equal(pool_bits(pool), slab)


def test_profile_counts_every_launch():
    w = W.Workload("prof", 1, 8, 2, 64, 4, None, 3, max_len=4096)
    pool = make_pool(w, 600)
    pool.set_option("profile", 1)
    pool.set_option("fuse_combine", 0)
    pool.set_option("min_chunk_blocks", 2)
    ids, lens = [1, 2, 3, 4], [40, 2000, 900, 16]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    q = W.q_values(3, 0, 0, 4, 8, 64, DEV)
    for _ in range(5):
        pool.attention(0, ids, q)
    pool.gather(2)
    prof = pool.profile()
    assert prof["ingest"][0] == 1 and prof["attn"][0] == 5 and prof["combine"][0] == 5 and prof["gather"][0] == 1
    assert all(ms > 0 for n, ms in prof.values() if n) and prof["varq"] == (0, 0.0)
    assert sum(n for n, _ in prof.values()) == pool.launches
    pool.profile_reset()
    assert pool.profile()["attn"] == (0, 0.0)
    pool.set_option("profile", 0)
    pool.attention(0, ids, q)
    assert pool.profile()["attn"][0] == 0
