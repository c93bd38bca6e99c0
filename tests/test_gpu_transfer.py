"""-m gpu tests of round 2's additions, through the C-ABI, against the oracle:

  * NEXT-4 kv_transfer (paged -> paged between two pools on one device, bf16 and FP8): the consumer's WHOLE slab
    == oracle.transfer into a sentinel-filled slab through the two block lists; the producer's slab untouched;
    layer-sliced transfer; attention on the consumer == oracle; error paths atomic.
  * paged_decode_step_layers (one host call, PDL-chained launches) == per-layer paged_decode_step, bit for bit,
    and == the oracle; its KV_STEP_RESERVE form; rollback on error.
  * attention calls of one pool issued on different streams are ordered by the library (shared workspace).
  * kv_ingest's atomicity promise: a failing call leaves allocator, tables and pool bytes as they were.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from gpu_harness import (apply_options, DEV, NAN_BITS, compare_attention, dims_of, kv_src, make_pool, oracle_attention, oracle_ingest,
                         oracle_slab, pool_bits)
from helpers import bits_of

pytestmark = pytest.mark.gpu


def fp8_pool(w, num_blocks, alloc_seed, max_requests=32, sentinel=0xFF):
    cfg = kv.PoolConfig(num_layers=w.num_layers, num_q_heads=w.num_q_heads, num_kv_heads=w.num_kv_heads,
                        head_dim=w.head_dim, num_blocks=num_blocks, max_requests=max_requests,
                        max_blocks_per_request=(w.max_len + 15) // 16, alloc_seed=alloc_seed, kv_dtype=B.KV_DTYPE_FP8_E4M3)
    pool = kv.KVPool(cfg, device=DEV)
    pool.slab[: pool.kv_bytes].fill_(sentinel)
    return pool


def raw(pool) -> np.ndarray:
    return pool.slab[: pool.kv_bytes].cpu().numpy()


LENS = [1, 15, 16, 17, 64, 130, 255, 1029, 700]


@pytest.mark.parametrize("Hq,Hkv,d,L", [(8, 2, 64, 3), (32, 8, 128, 2)])
def test_transfer_bf16_whole_slab(Hq, Hkv, d, L):
    w = W.Workload("xfer", L, Hq, Hkv, d, len(LENS), None, 777, max_len=2048)
    nb = sum((n + 15) // 16 for n in LENS)
    A = make_pool(w, nb + 40, alloc_seed=3, max_requests=32)          # the producer: its own size and permutation
    Bp = make_pool(w, nb + 9, alloc_seed=91, max_requests=32)         # the consumer
    src_ids = list(range(100, 100 + len(LENS)))
    dst_ids = list(range(900, 900 + len(LENS)))
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(src_ids, LENS)]
    A.ingest(src_ids, [s[0] for s in srcs], [s[1] for s in srcs])
    torch.cuda.synchronize()
    a_before = pool_bits(A).copy()
    Bp.reserve([5], [40])                                             # the consumer already holds something
    Bp.transfer_from(A, dst_ids, src_ids)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(A), a_before), "kv_transfer modified the producer's pool"
    want = oracle_slab(Bp)
    for s_id, d_id, n in zip(src_ids, dst_ids, LENS):
        sb, sn = A.block_table(s_id)
        db, dn = Bp.block_table(d_id)
        assert sn == dn == n and len(db) == (n + 15) // 16
        oracle.transfer(a_before, dims_of(A), sb, want, dims_of(Bp), db, n)
    assert np.array_equal(pool_bits(Bp), want), "consumer slab != oracle.transfer (whole slab)"
    # ... which is the scatter of the original sources through the consumer's block lists
    direct = oracle_slab(Bp)
    for u, d_id, n in zip(src_ids, dst_ids, LENS):
        k, v = kv_src(w, u, 0, n, "cpu")
        oracle.scatter(direct, dims_of(Bp), Bp.block_table(d_id)[0], 0, bits_of(k), bits_of(v))
    assert np.array_equal(want, direct)
    # the consumer attends over what it received
    q = W.q_values(w.seed, 0, L - 1, len(dst_ids), Hq, d, DEV)
    compare_attention(Bp.attention(L - 1, dst_ids, q), oracle_attention(want, Bp, L - 1, dst_ids, q))
    assert Bp.profile()["transfer"][0] == 0                            # profiling is off by default
    # gather on the consumer returns the producer's source tensors
    k, v = Bp.gather(dst_ids[7])
    assert torch.equal(k, srcs[7][0]) and torch.equal(v, srcs[7][1])


def test_transfer_layer_sliced_and_errors():
    L, Hq, Hkv, d = 4, 8, 2, 64
    w = W.Workload("xfer2", L, Hq, Hkv, d, 3, None, 778, max_len=512)
    A = make_pool(w, 24, alloc_seed=5, max_requests=8)
    Bp = make_pool(w, 12, alloc_seed=6, max_requests=4)
    lens = [33, 100, 16]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip([1, 2, 3], lens)]
    A.ingest([1, 2, 3], [s[0] for s in srcs], [s[1] for s in srcs])
    torch.cuda.synchronize()
    a_bits = pool_bits(A).copy()

    def state(p, ids):
        return (p.stats(), [(list(p.block_table(i)[0]), p.block_table(i)[1]) for i in ids], pool_bits(p).copy())

    before = state(Bp, [])
    for dst, src, lb, lc, status in [([7, 8], [1, 9], 0, L, B.KV_ERR_UNKNOWN_REQUEST),     # producer id not live
                                     ([7, 7], [1, 2], 0, L, B.KV_ERR_INVALID),            # duplicate consumer id
                                     ([7, 8], [1, 1], 0, L, B.KV_ERR_INVALID),            # duplicate producer id
                                     ([7, 8, 9], [1, 2, 3], 0, L, B.KV_ERR_NO_BLOCKS),    # 3 + 7 + 1 = 11 of 12: fits; see below
                                     ([7], [1], 1, 1, B.KV_ERR_UNKNOWN_REQUEST),          # continuation of nothing
                                     ([7], [1], 0, L + 1, B.KV_ERR_INVALID)]:
        if status == B.KV_ERR_NO_BLOCKS:
            Bp.reserve([50], [32])                                     # 2 blocks taken: now 11 do not fit in 10
        with pytest.raises(B.KVError) as e:
            Bp.transfer_from(A, dst, src, lb, lc)
        assert e.value.status == status, (dst, src, lb, lc)
        if status == B.KV_ERR_NO_BLOCKS:
            Bp.free([50])
        now = state(Bp, [])
        assert now[0]["blocks_free"] == before[0]["blocks_free"] and now[0]["live_requests"] == 0
        assert np.array_equal(now[2], before[2])
    with pytest.raises(B.KVError) as e:
        B.kv_transfer(A.handle, A.handle, [7], [1], 0, L)             # src == dst
    assert e.value.status == B.KV_ERR_INVALID
    # layer by layer, as a producer that streams its KV would
    want = oracle_slab(Bp)
    Bp.transfer_from(A, [7, 8], [2, 1], 0, 1)
    for l in range(1, L):
        Bp.transfer_from(A, [7, 8], [2, 1], l, 1)
    torch.cuda.synchronize()
    for d_id, s_id, n in [(7, 2, 100), (8, 1, 33)]:
        oracle.transfer(a_bits, dims_of(A), A.block_table(s_id)[0], want, dims_of(Bp), Bp.block_table(d_id)[0], n)
    assert np.array_equal(pool_bits(Bp), want)
    with pytest.raises(B.KVError) as e:                                # a live consumer id cannot be re-created
        Bp.transfer_from(A, [7], [3])
    assert e.value.status == B.KV_ERR_INVALID


@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 8, 128)])
def test_transfer_fp8_codes_and_scales_verbatim(Hq, Hkv, d):
    L = 2
    w = W.Workload("xfer8", L, Hq, Hkv, d, len(LENS), None, 779, max_len=2048)
    nb = sum((n + 15) // 16 for n in LENS)
    A, Bp = fp8_pool(w, nb + 17, 21, sentinel=0xEE), fp8_pool(w, nb + 3, 22)
    src_ids = list(range(10, 10 + len(LENS)))
    dst_ids = list(range(60, 60 + len(LENS)))
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(src_ids, LENS)]
    A.ingest(src_ids, [s[0] for s in srcs], [s[1] for s in srcs])
    torch.cuda.synchronize()
    a_before = raw(A).copy()
    Bp.transfer_from(A, dst_ids, src_ids)
    torch.cuda.synchronize()
    assert np.array_equal(raw(A), a_before)
    want = oracle.new_slab_fp8(dims_of(Bp), 0xFF)
    direct = oracle.new_slab_fp8(dims_of(Bp), 0xFF)
    for (k, v), s_id, d_id, n in zip(srcs, src_ids, dst_ids, LENS):
        oracle.transfer_fp8(a_before, dims_of(A), A.block_table(s_id)[0], want, dims_of(Bp), Bp.block_table(d_id)[0], n)
        oracle.scatter_fp8(direct, dims_of(Bp), Bp.block_table(d_id)[0], 0, bits_of(k), bits_of(v))
    assert np.array_equal(raw(Bp), want), "FP8 consumer slab != oracle.transfer_fp8 (whole slab)"
    assert np.array_equal(want, direct)                                # == quantising scatter of the original source
    q = W.q_values(w.seed, 0, 1, len(dst_ids), Hq, d, DEV)
    lists = [Bp.block_table(u)[0] for u in dst_ids]
    compare_attention(Bp.attention(1, dst_ids, q), oracle.attention_fp8(want, dims_of(Bp), 1, Hq, lists, LENS, bits_of(q)))
    with pytest.raises(B.KVError) as e:                                # bf16 -> FP8: geometry mismatch
        bf = make_pool(w, 8, max_requests=4)
        B.kv_transfer(bf.handle, A.handle, [1], [src_ids[0]], 0, L)
    assert e.value.status == B.KV_ERR_INVALID


# ---------------------------------------------------------------------------------------------
# paged_decode_step_layers
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("fp8", [False, True])
@pytest.mark.parametrize("opts", [dict(), dict(pdl=0), dict(min_chunk_blocks=1, items_per_slot=1024), dict(fuse_combine=0), dict(tc=0),
                                  dict(tc=0, min_chunk_blocks=1, items_per_slot=1024)])
def test_step_layers_equals_per_layer_calls_and_oracle(opts, fp8):
    L, Hq, Hkv, d = 4, 32, 8, 128
    lens0 = [15, 16, 17, 1, 0, 31, 255, 1039, 2047, 700]
    ids = list(range(300, 300 + len(lens0)))
    w = W.Workload("layers", L, Hq, Hkv, d, len(ids), None, 4243, max_len=2048 + 64)
    nb = sum((n + 15) // 16 + 1 for n in lens0) + 8
    pools = [fp8_pool(w, nb, 11) if fp8 else make_pool(w, nb, alloc_seed=11, max_requests=32) for _ in range(2)]
    for p in pools:
        apply_options(p, opts)
        p.set_option("profile", 1)
    have = [(u, n) for u, n in zip(ids, lens0) if n > 0]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in have]
    for p in pools:
        p.ingest([u for u, _ in have], [s[0] for s in srcs], [s[1] for s in srcs])
    slab = oracle.new_slab_fp8(dims_of(pools[0]), 0xFF) if fp8 else oracle_slab(pools[0])
    scatter = oracle.scatter_fp8 if fp8 else oracle.scatter
    for (u, n), (k, v) in zip(have, srcs):
        scatter(slab, dims_of(pools[0]), pools[0].block_table(u)[0], 0, bits_of(k), bits_of(v))
    lens = list(lens0)
    s = torch.cuda.current_stream().cuda_stream
    for step in range(3):
        kd = W.kv_values_at(w.seed, W.KIND_K, ids, lens, Hkv, d, 0, L, DEV)            # [L][B][Hkv][d]
        vd = W.kv_values_at(w.seed, W.KIND_V, ids, lens, Hkv, d, 0, L, DEV)
        q = torch.stack([W.q_values(w.seed, step, l, len(ids), Hq, d, DEV) for l in range(L)])
        out_a, out_b = torch.empty_like(q), torch.empty_like(q)
        n0 = pools[0].launches
        B.paged_decode_step_layers(pools[0].handle, 0, L, ids, q.data_ptr(), kd.data_ptr(), vd.data_ptr(), out_a.data_ptr(),
                                   q[0].numel() * 2, kd[0].numel() * 2, 0.0, B.KV_STEP_RESERVE, s)
        per_layer = 1 if opts.get("fuse_combine", 1) else 2
        assert pools[0].launches - n0 == per_layer * L
        pools[1].reserve(ids, [1] * len(ids))
        for l in range(L):
            pools[1].decode_step(l, ids, q[l], kd[l], vd[l], out=out_b[l])
        torch.cuda.synchronize()
        assert torch.equal(out_a.view(torch.int16), out_b.view(torch.int16)), "layers call != per-layer calls"
        assert torch.equal(pools[0].slab[: pools[0].kv_bytes], pools[1].slab[: pools[1].kv_bytes])
        for i, (u, n) in enumerate(zip(ids, lens)):
            scatter(slab, dims_of(pools[0]), pools[0].block_table(u)[0], n, bits_of(kd[:, i].unsqueeze(2)), bits_of(vd[:, i].unsqueeze(2)))
        lens = [n + 1 for n in lens]
        lists = [pools[0].block_table(u)[0] for u in ids]
        for l in range(L):
            want = (oracle.attention_fp8 if fp8 else oracle.attention)(slab, dims_of(pools[0]), l, Hq, lists, lens, bits_of(q[l]))
            compare_attention(out_a[l], want)
    assert np.array_equal(raw(pools[0]) if fp8 else pool_bits(pools[0]), slab)
    assert pools[0].profile()["attn"][0] == 3 * L                       # a group of L launches counts as L
    if opts.get("pdl", 1) and opts.get("fuse_combine", 1):              # layers 1..L-1 of every step chain behind layer 0
        assert pools[0].counter("attn_chained_launches") == 3 * (L - 1) and pools[0].counter("plans_uploaded") == 3
    else:
        assert pools[0].counter("attn_chained_launches") == 0
    # attention only (no append) over several layers in one call == per-layer paged_decode_attention
    out_c, out_d = torch.empty_like(q), torch.empty_like(q)
    B.paged_decode_step_layers(pools[0].handle, 1, L - 1, ids, q[1].data_ptr(), 0, 0, out_c[1].data_ptr(), q[0].numel() * 2, 0, 0.0, 0, s)
    for l in range(1, L):
        pools[1].attention(l, ids, q[l], out=out_d[l])
    torch.cuda.synchronize()
    assert torch.equal(out_c[1:].view(torch.int16), out_d[1:].view(torch.int16))


def test_step_layers_errors_roll_back():
    L, Hq, Hkv, d = 2, 8, 2, 64
    w = W.Workload("layers_err", L, Hq, Hkv, d, 2, None, 1, max_len=64)
    pool = make_pool(w, 4, alloc_seed=0, max_requests=4)
    k, v = kv_src(w, 1, 0, 32, DEV)
    k2, v2 = kv_src(w, 2, 0, 16, DEV)
    pool.ingest([1, 2], [k, k2], [v, v2])                               # 3 of 4 blocks; both requests sit on a block boundary
    torch.cuda.synchronize()
    q = torch.zeros((L, 2, Hq, d), dtype=torch.bfloat16, device=DEV)
    kn = torch.zeros((L, 2, Hkv, d), dtype=torch.bfloat16, device=DEV)
    out = torch.empty_like(q)
    stats, bits = pool.stats(), pool_bits(pool).copy()
    args = lambda ids, lb, lc, flags, kptr=None: (pool.handle, lb, lc, ids, q.data_ptr(), kn.data_ptr() if kptr is None else kptr,
                                                  kn.data_ptr() if kptr is None else kptr, out.data_ptr(), q[0].numel() * 2,
                                                  kn[0].numel() * 2, 0.0, flags, 0)
    for a, status in [(args([1, 2], 0, L, B.KV_STEP_RESERVE), B.KV_ERR_NO_BLOCKS),        # both need a new block, 1 free
                      (args([1, 9], 0, L, 0), B.KV_ERR_UNKNOWN_REQUEST),
                      (args([1], 1, 1, B.KV_STEP_RESERVE), B.KV_ERR_INVALID),            # reserve needs layer_begin 0
                      (args([1], 0, L, B.KV_STEP_RESERVE, kptr=0), B.KV_ERR_INVALID),    # reserve needs k_new
                      (args([1], 0, L, 0), B.KV_ERR_INVALID),                            # append without a 1-token reservation
                      (args([1], 0, L + 1, 0), B.KV_ERR_INVALID),
                      (args([1], 0, L, 2), B.KV_ERR_INVALID)]:                           # unknown flag
        with pytest.raises(B.KVError) as e:
            B.paged_decode_step_layers(*a)
        assert e.value.status == status
        assert pool.stats() == stats and pool.block_table(1)[1] == 32 and pool.block_table(2)[1] == 16
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), bits)
    B.paged_decode_step_layers(*args([1], 0, L, B.KV_STEP_RESERVE))                      # one request fits
    torch.cuda.synchronize()
    assert pool.block_table(1)[1] == 33 and pool.stats()["blocks_free"] == 0


# ---------------------------------------------------------------------------------------------
# attention launches of one pool on two streams
# ---------------------------------------------------------------------------------------------

def test_attention_on_two_streams_is_ordered_by_the_library():
    L, Hq, Hkv, d = 2, 32, 8, 128
    lens = [2047, 1500, 900, 1800, 64, 1200, 2000, 333] * 4             # split into many chunks: the workspace is busy
    ids = list(range(len(lens)))
    w = W.Workload("streams", L, Hq, Hkv, d, len(ids), None, 55, max_len=2048 + 64)
    pool = make_pool(w, sum((n + 15) // 16 for n in lens) + 8, alloc_seed=4, max_requests=64)
    pool.set_option("min_chunk_blocks", 4)
    slab = oracle_slab(pool)
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    for u, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, u, 0, n)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    half = len(ids) // 2
    qs, outs = [], []
    for rep in range(6):                                                 # alternate streams and batches, never synchronising
        st, batch = (s1, ids[:half]) if rep % 2 == 0 else (s2, ids[half:])
        q = W.q_values(w.seed, rep, rep % L, len(batch), Hq, d, DEV)
        torch.cuda.current_stream().synchronize()
        outs.append((batch, rep % L, q, pool.attention(rep % L, batch, q, stream=st)))
    torch.cuda.synchronize()
    assert pool.counter("attn_stream_switches") == 5                     # every call after the first changed stream
    for batch, layer, q, out in outs:
        compare_attention(out, oracle_attention(slab, pool, layer, batch, q))


# ---------------------------------------------------------------------------------------------
# kv_ingest is atomic
# ---------------------------------------------------------------------------------------------

def test_failed_ingest_changes_nothing():
    L, Hq, Hkv, d = 2, 8, 2, 64
    w = W.Workload("atomic", L, Hq, Hkv, d, 2, None, 3, max_len=256)
    pool = make_pool(w, 6, alloc_seed=9, max_requests=3)
    k, v = kv_src(w, 1, 0, 40, DEV)
    pool.ingest([1], [k], [v])                                           # 3 of 6 blocks
    torch.cuda.synchronize()
    stats, table, bits = pool.stats(), pool.block_table(1), pool_bits(pool).copy()
    kb, vb = kv_src(w, 2, 0, 70, DEV)                                    # 5 blocks: does not fit
    stage = torch.empty(1 << 20, dtype=torch.uint8, device=DEV)
    kh, vh = kb.cpu().pin_memory(), vb.cpu().pin_memory()
    for call in [lambda: pool.ingest([2], [kb], [vb]),
                 lambda: B.kv_ingest_host(pool.handle, [2], [70], [kh.data_ptr()], [vh.data_ptr()], 0, L, stage.data_ptr(), stage.numel(), 0),
                 lambda: pool.ingest([1, 2], [k[:, :, :8].contiguous(), kb[:, :, :60].contiguous()],
                                     [v[:, :, :8].contiguous(), vb[:, :, :60].contiguous()])]:   # 0 + 4 blocks > 3 free
        with pytest.raises(B.KVError) as e:
            call()
        assert e.value.status == B.KV_ERR_NO_BLOCKS
        torch.cuda.synchronize()
        assert pool.stats() == stats
        assert np.array_equal(pool.block_table(1)[0], table[0]) and pool.block_table(1)[1] == table[1]
        with pytest.raises(B.KVError):
            pool.block_table(2)
        assert np.array_equal(pool_bits(pool), bits)
    # the host-buffer form refuses before touching the stream, then works once there is room: pinned sources are read in
    # place by the scatter kernel (zero-copy), pageable ones go through the staging buffer — same bytes either way
    pool.free([1])
    B.kv_ingest_host(pool.handle, [2], [70], [kh.data_ptr()], [vh.data_ptr()], 0, L, stage.data_ptr(), stage.numel(), 0)
    torch.cuda.synchronize()
    assert pool.counter("host_ingest_zero_copy") == 1 and pool.counter("host_ingest_staged") == 0
    gk, gv = pool.gather(2)
    assert torch.equal(gk, kb) and torch.equal(gv, vb)
    pool.free([2])
    kp, vp = kb.cpu(), vb.cpu()                                          # pageable host memory
    B.kv_ingest_host(pool.handle, [3], [70], [kp.data_ptr()], [vp.data_ptr()], 0, L, stage.data_ptr(), stage.numel(), 0)
    torch.cuda.synchronize()
    assert pool.counter("host_ingest_staged") == 1
    gk, gv = pool.gather(3)
    assert torch.equal(gk, kb) and torch.equal(gv, vb)
