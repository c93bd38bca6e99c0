"""-m gpu: paged_decode_attention_static — the entry point that allocates nothing (split-KV workspace in a file-scope
`static __device__` array of the library, include/kv_pool.h) — against the existing path, paged_decode_attention, on
the same pool and inputs, on two calls in a row whose plans differ (so the second call meets the arrival counters and
partials the first one left behind), and against the oracle.  Collected last on purpose (the suite runs with -x)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from gpu_harness import DEV, apply_options, compare_attention, kv_src, make_pool, oracle_attention, oracle_ingest, oracle_slab
from helpers import bits_of, bits_to_f64

pytestmark = pytest.mark.gpu

SPLIT = dict(min_chunk_blocks=1, items_per_slot=1024)   # every request split into many chunks: partials and merges everywhere


def n_partials(pool, ids):
    items, _ = pool.plan(ids)
    return int(sum(1 for it in items if it[4] >= 0))


def close_to_existing(got, ref, same_plan=True):
    """The tolerance the attention parity tests use (BASELINE.json north_star: max abs <= 1e-2, mean abs <= 1e-3) —
    and, where the two calls ran the same plan (same split, same kernel, partials merged in chunk order), the same bits."""
    a, b = bits_to_f64(bits_of(got)), bits_to_f64(bits_of(ref))
    assert np.all(np.isfinite(a))
    err = np.abs(a - b)
    assert err.max() <= 1e-2 and err.mean() <= 1e-3, (float(err.max()), float(err.mean()))
    if same_plan:
        assert np.array_equal(bits_of(got), bits_of(ref)), (float(err.max()), float(err.mean()))


def fill(pool, w, ids, lens, slab=None):
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    if slab is not None:
        for uid, n in zip(ids, lens):
            oracle_ingest(slab, pool, w, uid, 0, n)


@pytest.mark.parametrize("opts", [SPLIT, dict(SPLIT, fuse_combine=0), dict()])
@pytest.mark.parametrize("Hq,Hkv,d", [(32, 8, 128), (8, 8, 64)])
def test_bf16_two_calls_match_existing_path_and_oracle(Hq, Hkv, d, opts):
    lens = [1, 15, 16, 17, 200, 333, 1024, 2047, 900, 31]
    w = W.Workload("no_alloc", 2, Hq, Hkv, d, len(lens), None, 20251105, max_len=2048)
    pool = make_pool(w, sum((n + 15) // 16 for n in lens) + 16, alloc_seed=5)
    apply_options(pool, opts)
    ids = list(range(70, 70 + len(lens)))
    slab = oracle_slab(pool)
    fill(pool, w, ids, lens, slab)
    assert B.kv_static_scratch_bytes() == B.KV_STATIC_MAX_PARTIALS * (4 + 8 * 2 * 4 + 8 * 128 * 4)
    # call 1: the whole batch, layer 1; call 2, right behind it: another layer, a permuted sub-batch (another plan)
    calls = [(1, ids), (0, [ids[6], ids[0], ids[7], ids[4], ids[3]])]
    outs = []
    launches0 = pool.launches
    for layer, sub in calls:
        q = W.q_values(w.seed, 0, layer, len(sub), Hq, d, DEV)
        out = torch.full_like(q, float("nan"))
        pool.decode_attention_static(layer, sub, q, out=out)
        outs.append((layer, sub, q, out))
    assert pool.launches > launches0            # the library's own kernels ran
    torch.cuda.synchronize()
    if opts.get("min_chunk_blocks") == 1:
        assert n_partials(pool, ids) > 0        # the static workspace was really in use
    for layer, sub, q, out in outs:
        ref = pool.attention(layer, sub, q)
        torch.cuda.synchronize()
        close_to_existing(out, ref)
        compare_attention(out, oracle_attention(slab, pool, layer, sub, q))
    # and once more after the existing path has run in between (its plan cache was dropped and rebuilt)
    layer, sub, q, out = outs[0]
    again = pool.decode_attention_static(layer, sub, q)
    torch.cuda.synchronize()
    assert np.array_equal(bits_of(again), bits_of(out))


@pytest.mark.parametrize("opts", [dict(tc=1, **SPLIT), dict(tc=0, **SPLIT), dict()])
def test_fp8_two_calls_match_existing_path(opts):
    Hq, Hkv, d = 32, 8, 128
    lens = [129, 16, 700, 1500, 4000, 257, 3]
    w = W.Workload("no_alloc_fp8", 2, Hq, Hkv, d, len(lens), None, 77, max_len=4096)
    cfg = kv.PoolConfig(num_layers=2, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d,
                        num_blocks=sum((n + 15) // 16 for n in lens) + 8, max_requests=16, max_blocks_per_request=256,
                        alloc_seed=3, kv_dtype=B.KV_DTYPE_FP8_E4M3)
    pool = kv.KVPool(cfg, device=DEV)
    pool.slab[: pool.kv_bytes].fill_(0xFF)
    apply_options(pool, opts)
    ids = list(range(300, 300 + len(lens)))
    fill(pool, w, ids, lens)
    for layer, sub in [(0, ids), (1, ids[2:6])]:
        q = W.q_values(w.seed, 1, layer, len(sub), Hq, d, DEV)
        out = pool.decode_attention_static(layer, sub, q)
        ref = pool.attention(layer, sub, q)
        torch.cuda.synchronize()
        close_to_existing(out, ref)


def test_second_call_allocates_no_device_memory_and_limit_is_enforced():
    Hq = Hkv = 8
    d = 64
    lens = [2048] * 48
    w = W.Workload("no_alloc_limit", 1, Hq, Hkv, d, len(lens), None, 9, max_len=2048)
    pool = make_pool(w, 48 * 128 + 8, max_requests=64, alloc_seed=0)
    ids = list(range(len(lens)))
    fill(pool, w, ids, lens)                    # (the ingest kernel also writes the device block_table the kernels read)
    q = W.q_values(w.seed, 2, 0, len(ids), Hq, d, DEV)
    out = torch.empty_like(q)
    pool.decode_attention_static(0, ids, q, out=out)          # first call: symbol look-up, lazy kernel loading
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    pool.decode_attention_static(0, ids, q, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the call took device memory"
    ref = pool.attention(0, ids, q)
    torch.cuda.synchronize()
    close_to_existing(out, ref)
    # a plan beyond the static array's KV_STATIC_MAX_PARTIALS partial slots is refused, and nothing changes
    pool.set_option("min_chunk_blocks", 1)
    pool.set_option("items_per_slot", 64)
    assert n_partials(pool, ids) > B.KV_STATIC_MAX_PARTIALS
    before = out.clone()
    launches = pool.launches
    with pytest.raises(kv.KVError) as e:
        pool.decode_attention_static(0, ids, q, out=out)
    assert e.value.status == B.KV_ERR_SCRATCH_LIMIT and "static scratch" in kv.kv_strerror(e.value.status)
    torch.cuda.synchronize()
    assert pool.launches == launches and torch.equal(out.view(torch.int16), before.view(torch.int16))
    ref = pool.attention(0, ids, q)            # the existing path has no such limit (a finer split: other roundings)
    torch.cuda.synchronize()
    close_to_existing(ref, before, same_plan=False)
