"""-m gpu: KV-head sharding of a TP-sharded D-instance ("TP" multiplies capacity and bandwidth,
PAPER.md:206/:212) — correct by construction and checked on ONE GPU: TP shard pools, each
holding num_kv_heads / TP heads of every block, ingest their slice from the SAME full-width producer tensors
(pool options src_kv_heads / src_head_begin), take identical allocator decisions (same seed), attend with their own
query heads, and the concatenated outputs are the unsharded result — no collective inside the path."""
import numpy as np
import pytest
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from gpu_harness import DEV, NAN_BITS, compare_attention, dims_of, kv_src, pool_bits
from helpers import bits_of

pytestmark = pytest.mark.gpu

L, HQ, HKV, D, TP = 2, 32, 8, 128, 4
LENS = [17, 64, 130, 700, 1, 2100]
NB = sum((n + 15) // 16 for n in LENS) + 16


def make(hq, hkv, kv_dtype=B.KV_DTYPE_BF16, fill=NAN_BITS):
    cfg = kv.PoolConfig(num_layers=L, num_q_heads=hq, num_kv_heads=hkv, head_dim=D, num_blocks=NB, max_requests=16,
                        max_blocks_per_request=256, alloc_seed=77, kv_dtype=kv_dtype)
    pool = kv.KVPool(cfg, device=DEV)
    if kv_dtype == B.KV_DTYPE_BF16:
        pool.slab[: pool.kv_bytes].view(torch.int16).fill_(int(np.uint16(fill).astype(np.int16)))
    else:
        pool.slab[: pool.kv_bytes].fill_(0xFF)
    return pool


def sources():
    w = W.Workload("tp", L, HQ, HKV, D, len(LENS), None, 31, max_len=4096)
    ids = list(range(40, 40 + len(LENS)))
    return w, ids, [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, LENS)]


@pytest.mark.parametrize("opts", [dict(min_chunk_blocks=4096), dict(), dict(min_chunk_blocks=2, items_per_slot=1024)])
def test_sharded_pools_reproduce_the_unsharded_result(opts):
    w, ids, srcs = sources()
    full = make(HQ, HKV)
    for k_, v_ in opts.items():
        full.set_option(k_, v_)
    full.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    q = [W.q_values(w.seed, 0, l, len(ids), HQ, D, DEV) for l in range(L)]
    out_full = [full.attention(l, ids, q[l]) for l in range(L)]
    torch.cuda.synchronize()
    hq, hkv = HQ // TP, HKV // TP
    for r in range(TP):
        shard = make(hq, hkv)
        for k_, v_ in opts.items():
            shard.set_option(k_, v_)
        shard.set_option("src_kv_heads", HKV)
        shard.set_option("src_head_begin", r * hkv)
        B.kv_ingest(shard.handle, ids, LENS, [s[0] for s in srcs], [s[1] for s in srcs], 0, L,
                    torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        # replicated allocator decisions: the same block lists on every shard
        for u in ids:
            assert np.array_equal(shard.block_table(u)[0], full.block_table(u)[0])
        # the shard's pool is the oracle scatter of its head slice, bit for bit, sentinel elsewhere
        slab = oracle.new_slab(dims_of(shard), NAN_BITS)
        for u, n, (k, v) in zip(ids, LENS, srcs):
            ks = bits_of(k[:, r * hkv:(r + 1) * hkv].contiguous())
            vs = bits_of(v[:, r * hkv:(r + 1) * hkv].contiguous())
            oracle.scatter(slab, dims_of(shard), shard.block_table(u)[0], 0, ks, vs)
        assert np.array_equal(pool_bits(shard), slab)
        for l in range(L):
            ql = q[l][:, r * hq:(r + 1) * hq].contiguous()
            out = shard.attention(l, ids, ql)
            torch.cuda.synchronize()
            lists = [shard.block_table(u)[0] for u in ids]
            want = oracle.attention(slab, dims_of(shard), l, hq, lists, LENS, bits_of(ql))
            compare_attention(out, want)
            if opts.get("min_chunk_blocks") == 4096:            # unsplit units: the very same arithmetic per head
                assert torch.equal(out.view(torch.int16), out_full[l][:, r * hq:(r + 1) * hq].contiguous().view(torch.int16))
        shard.close()


def test_gather_from_shards_rebuilds_the_full_width_tensor():
    w, ids, srcs = sources()
    hkv = HKV // TP
    u, n = ids[3], LENS[3]
    k_dst = torch.zeros((L, HKV, n, D), dtype=torch.bfloat16, device=DEV)
    v_dst = torch.zeros_like(k_dst)
    for r in range(TP):
        shard = make(HQ // TP, hkv)
        shard.set_option("src_kv_heads", HKV)
        shard.set_option("src_head_begin", r * hkv)
        B.kv_ingest(shard.handle, [u], [n], [srcs[3][0]], [srcs[3][1]], 0, L, torch.cuda.current_stream().cuda_stream)
        B.kv_gather(shard.handle, u, k_dst.data_ptr(), v_dst.data_ptr(), torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        shard.close()
    assert torch.equal(k_dst.view(torch.int16), srcs[3][0].view(torch.int16))
    assert torch.equal(v_dst.view(torch.int16), srcs[3][1].view(torch.int16))


def test_sharded_fp8_pool_and_host_buffers():
    w, ids, srcs = sources()
    hq, hkv, r = HQ // TP, HKV // TP, 2
    shard = make(hq, hkv, kv_dtype=B.KV_DTYPE_FP8_E4M3)
    shard.set_option("src_kv_heads", HKV)
    shard.set_option("src_head_begin", r * hkv)
    # arrivals in pinned host memory, full width, through kv_ingest_host
    kh = [torch.empty(s[0].shape, dtype=s[0].dtype, pin_memory=True).copy_(s[0]) for s in srcs]
    vh = [torch.empty(s[1].shape, dtype=s[1].dtype, pin_memory=True).copy_(s[1]) for s in srcs]
    need = sum(2 * ((k.numel() * 2 + 255) // 256 * 256) for k in kh)
    stage = torch.empty(need, dtype=torch.uint8, device=DEV)
    B.kv_ingest_host(shard.handle, ids, LENS, [k.data_ptr() for k in kh], [v.data_ptr() for v in vh], 0, L,
                     stage.data_ptr(), stage.numel(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    slab = oracle.new_slab_fp8(dims_of(shard), 0xFF)
    for u, n, (k, v) in zip(ids, LENS, srcs):
        oracle.scatter_fp8(slab, dims_of(shard), shard.block_table(u)[0], 0,
                           bits_of(k[:, r * hkv:(r + 1) * hkv].contiguous()), bits_of(v[:, r * hkv:(r + 1) * hkv].contiguous()))
    assert np.array_equal(shard.slab[: shard.kv_bytes].cpu().numpy(), slab)
    ql = W.q_values(w.seed, 1, 0, len(ids), HQ, D, DEV)[:, r * hq:(r + 1) * hq].contiguous()
    out = shard.attention(0, ids, ql)
    torch.cuda.synchronize()
    want = oracle.attention_fp8(slab, dims_of(shard), 0, hq, [shard.block_table(u)[0] for u in ids], LENS, bits_of(ql))
    compare_attention(out, want)


def test_option_validation():
    shard = make(HQ // TP, HKV // TP)
    for key, val in [("src_kv_heads", 1), ("src_head_begin", 1)]:       # narrower than the pool / outside the source
        with pytest.raises(B.KVError):
            shard.set_option(key, val)
    shard.set_option("src_kv_heads", HKV)
    with pytest.raises(B.KVError):
        shard.set_option("src_head_begin", HKV - 1)
    shard.set_option("src_head_begin", HKV - HKV // TP)
    shard.set_option("src_kv_heads", 0)                                 # back to unsharded
