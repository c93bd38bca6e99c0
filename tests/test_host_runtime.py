"""Host logic through the C-ABI, CPU only (no compute calls): the library loads and exports
every symbol include/kv_pool.h declares; allocator / block_table invariants
against a set-based model; split-KV plan properties."""
import os
import re

import numpy as np
import pytest

import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def host_pool(**kw):
    cfg = dict(num_layers=2, num_q_heads=8, num_kv_heads=2, head_dim=64, num_blocks=128, max_requests=16,
               max_blocks_per_request=32, alloc_seed=0)
    cfg.update(kw)
    return kv.KVPool(kv.PoolConfig(**cfg))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "kv_pool.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(kv_[a-z_]+|paged_[a-z_]+)\s*\(", header))
    assert {"kv_pool_create", "kv_ingest", "paged_decode_attention", "kv_free"} <= declared
    for name in declared:
        assert hasattr(B.lib, name), f"libkvpool.so does not export {name}"
    assert declared == set(B.EXPORTS)
    assert re.fullmatch(r"\d+\.\d+\.\d+", kv.kv_version())
    assert kv.kv_strerror(0) == "ok" and "exhausted" in kv.kv_strerror(B.KV_ERR_NO_BLOCKS)


def test_config_validation():
    ok = dict(num_layers=1, num_q_heads=8, num_kv_heads=2, head_dim=64, num_blocks=8, max_requests=4,
              max_blocks_per_request=4)
    assert kv.kv_pool_kv_bytes(kv.PoolConfig(**ok)) == 1 * 8 * 2 * 2 * 16 * 64 * 2
    assert kv.kv_pool_required_bytes(kv.PoolConfig(**ok)) > kv.kv_pool_kv_bytes(kv.PoolConfig(**ok))
    for bad in [dict(head_dim=96), dict(block_size=32), dict(num_q_heads=7), dict(num_q_heads=32, num_kv_heads=2),
                dict(num_blocks=0), dict(max_requests=0), dict(num_layers=0)]:
        with pytest.raises(kv.KVError) as e:
            kv.kv_pool_required_bytes(kv.PoolConfig(**{**ok, **bad}))
        assert e.value.status == B.KV_ERR_INVALID


def test_host_only_pool_refuses_kernel_calls():
    p = host_pool()
    p.reserve([1], [20])
    with pytest.raises(kv.KVError) as e:
        kv.kv_ingest(p.handle, [2], [4], [256], [512], 0, 2)
    assert e.value.status == B.KV_ERR_NO_DEVICE
    with pytest.raises(kv.KVError) as e:
        kv.paged_decode_attention(p.handle, 0, [1], 256, 512)
    assert e.value.status == B.KV_ERR_NO_DEVICE
    with pytest.raises(kv.KVError) as e:                   # the no-allocation form: same checks before any GPU work
        kv.paged_decode_attention_static(p.handle, 0, [1], 256, 512)
    assert e.value.status == B.KV_ERR_NO_DEVICE
    with pytest.raises(kv.KVError) as e:
        kv.paged_decode_attention_static(p.handle, 0, [1], 0, 512)
    assert e.value.status == B.KV_ERR_INVALID
    assert p.launches == 0
    # its static scratch: KV_STATIC_MAX_PARTIALS slots of (arrival counter, (m, l) x 8 heads, O x 8 heads x 128) fp32
    assert kv.kv_static_scratch_bytes() == B.KV_STATIC_MAX_PARTIALS * (4 + 8 * 2 * 4 + 8 * 128 * 4) == 17055744
    assert "static scratch" in kv.kv_strerror(B.KV_ERR_SCRATCH_LIMIT)


def test_sequential_and_seeded_free_lists():
    p = host_pool(alloc_seed=0)
    p.reserve([7], [40])
    blocks, n = p.block_table(7)
    assert list(blocks) == [0, 1, 2] and n == 40
    a = host_pool(alloc_seed=123, max_blocks_per_request=64)
    b = host_pool(alloc_seed=123, max_blocks_per_request=64)
    c = host_pool(alloc_seed=124, max_blocks_per_request=64)
    for q in (a, b, c):
        q.reserve([1, 2], [16 * 60, 16 * 60])
    la = np.concatenate([a.block_table(1)[0], a.block_table(2)[0]])
    lb = np.concatenate([b.block_table(1)[0], b.block_table(2)[0]])
    lc = np.concatenate([c.block_table(1)[0], c.block_table(2)[0]])
    assert np.array_equal(la, lb) and not np.array_equal(la, lc)
    assert len(set(la.tolist())) == 120 and not np.array_equal(la, np.arange(120))   # a permutation, fragmented


def test_errors_are_atomic():
    p = host_pool(num_blocks=10, max_requests=3, max_blocks_per_request=8)
    p.reserve([1, 2], [16 * 4, 16 * 3])                   # 7 of 10 blocks
    before = (p.stats(), p.block_table(1), p.block_table(2))

    def unchanged():
        now = (p.stats(), p.block_table(1), p.block_table(2))
        assert now[0] == before[0]
        assert all(np.array_equal(x[0], y[0]) and x[1] == y[1] for x, y in zip(now[1:], before[1:]))

    for ids, n, status in [([1, 3], [16, 16 * 3], B.KV_ERR_NO_BLOCKS),       # needs 4, only 3 free
                           ([3, 3], [1, 1], B.KV_ERR_INVALID),               # duplicate id
                           ([1], [16 * 5], B.KV_ERR_TOO_LONG),               # 9 blocks > 8
                           ([3, 4], [1, 1], B.KV_ERR_TOO_MANY_REQUESTS),     # 4 live > 3
                           ([3], [-1], B.KV_ERR_INVALID)]:
        with pytest.raises(kv.KVError) as e:
            p.reserve(ids, n)
        assert e.value.status == status
        unchanged()
    for ids, status in [([1, 9], B.KV_ERR_UNKNOWN_REQUEST), ([1, 1], B.KV_ERR_INVALID)]:
        with pytest.raises(kv.KVError) as e:
            p.free(ids)
        assert e.value.status == status
        unchanged()
    with pytest.raises(kv.KVError) as e:
        p.block_table(9)
    assert e.value.status == B.KV_ERR_UNKNOWN_REQUEST
    p.reserve([3], [0])                                   # empty request is allowed (A12)
    assert p.block_table(3)[1] == 0 and p.block_table(3)[0].size == 0
    with pytest.raises(kv.KVError):                       # ... but cannot be attended (A11)
        p.plan([3])


@pytest.mark.parametrize("seed", [0, 5])
def test_p11_allocator_model_check(seed):
    rng = np.random.default_rng(100 + seed)
    NB, MAXR, MAXB, bs = 96, 12, 24, 16
    p = host_pool(num_blocks=NB, max_requests=MAXR, max_blocks_per_request=MAXB, alloc_seed=seed)
    model = {}                        # id -> (len, [blocks])
    free = set(range(NB))
    hw = 0
    for step in range(3000):
        op = rng.random()
        if op < 0.55:                  # grow / create a few requests
            k = int(rng.integers(1, 4))
            ids = rng.choice(40, size=k, replace=False).tolist()
            n = rng.integers(0, 70, size=k).tolist()
            need = sum((model.get(i, (0, []))[0] + t + bs - 1) // bs - len(model.get(i, (0, []))[1]) for i, t in zip(ids, n))
            new = sum(1 for i in ids if i not in model)
            too_long = any(model.get(i, (0, []))[0] + t > MAXB * bs for i, t in zip(ids, n))
            try:
                p.reserve(ids, n)
                ok = True
            except kv.KVError as e:
                ok = False
                assert e.status in (B.KV_ERR_NO_BLOCKS, B.KV_ERR_TOO_LONG, B.KV_ERR_TOO_MANY_REQUESTS)
            assert ok == (not too_long and new + len(model) <= MAXR and need <= len(free))
            if ok:
                for i, t in zip(ids, n):
                    ln, bl = model.get(i, (0, []))
                    got, glen = p.block_table(i)
                    assert glen == ln + t and len(got) == (ln + t + bs - 1) // bs
                    assert list(got[:len(bl)]) == bl                      # existing blocks keep their place
                    fresh = list(got[len(bl):])
                    assert set(fresh) <= free and len(set(fresh)) == len(fresh)
                    free -= set(fresh)
                    model[i] = (ln + t, list(got))
        elif model:                    # free some
            k = int(rng.integers(1, min(3, len(model)) + 1))
            ids = rng.choice(sorted(model), size=k, replace=False).tolist()
            p.free(ids)
            for i in ids:
                free |= set(model.pop(i)[1])
        hw = max(hw, NB - len(free))
        st = p.stats()
        assert st["blocks_free"] == len(free) and st["live_requests"] == len(model)
        assert st["blocks_total"] == NB and st["blocks_high_water"] == hw
        live = [b for _, bl in model.values() for b in bl]
        assert len(live) == len(set(live)) == NB - len(free)              # pairwise disjoint, conserved
    assert hw > NB // 2


def check_plan(p, ids, lens, Hkv, bs=16):
    items, chunk = p.plan(ids)
    assert chunk >= 1
    cover = {}
    for b, h, b0, nb, pidx in items.tolist():
        assert nb >= 1 and nb <= chunk
        cover.setdefault((b, h), []).append((b0, nb, pidx))
    assert set(cover) == {(b, h) for b in range(len(ids)) for h in range(Hkv)}
    partials = []
    for (b, h), runs in cover.items():
        runs.sort()
        total = (lens[b] + bs - 1) // bs
        pos = 0
        for b0, nb, pidx in runs:                       # every block exactly once, in order
            assert b0 == pos
            pos += nb
        assert pos == total
        if len(runs) == 1:
            assert runs[0][2] == -1
        else:
            ps = [r[2] for r in runs]
            assert ps == list(range(ps[0], ps[0] + len(ps)))   # contiguous partial slots in chunk order
            partials += ps
            sizes = [r[1] for r in runs]
            # guided chunking: a chunk is sized to the work still unassigned, so within a request the
            # sizes never grow, except that the last one may absorb a remainder of up to a quarter chunk
            assert all(a >= b for a, b in zip(sizes[:-2], sizes[1:-1]))
            assert len(sizes) < 2 or sizes[-1] <= sizes[-2] + sizes[-2] // 4 + 1
    assert sorted(partials) == list(range(len(partials)))
    nbs = items[:, 3]
    assert np.all(nbs[:-1] >= nbs[1:])                  # longest first
    return items, chunk


def test_plan_covers_every_block_once():
    rng = np.random.default_rng(3)
    Hkv = 2
    p = host_pool(num_blocks=4096, max_requests=64, max_blocks_per_request=1024, num_kv_heads=Hkv)
    lens = [17, 64, 130, 255, 1, 16, 5000, 16000, 33, 2048]
    ids = list(range(100, 100 + len(lens)))
    p.reserve(ids, lens)
    for min_chunk, ips in [(16, 8), (1, 8), (4, 1), (64, 64), (1000, 1)]:
        p.set_option("min_chunk_blocks", min_chunk)
        p.set_option("items_per_slot", ips)
        items, chunk = check_plan(p, ids, lens, Hkv)
        assert chunk >= min_chunk
    # a permuted batch order only relabels batch_idx
    perm = rng.permutation(len(lens))
    check_plan(p, [ids[i] for i in perm], [lens[i] for i in perm], Hkv)
    with pytest.raises(kv.KVError) as e:
        p.plan([100, 100])
    assert e.value.status == B.KV_ERR_INVALID
    with pytest.raises(kv.KVError) as e:
        p.plan([100, 999])
    assert e.value.status == B.KV_ERR_UNKNOWN_REQUEST


def test_plan_respects_partials_workspace():
    Hkv = 8
    p = host_pool(num_q_heads=32, num_kv_heads=Hkv, head_dim=128, num_blocks=300000, max_requests=600,
                  max_blocks_per_request=2048)
    lens = [32768] * 128
    ids = list(range(128))
    p.reserve(ids, lens)
    p.set_option("min_chunk_blocks", 1)
    p.set_option("items_per_slot", 1024)                # asks for ~1.2M items: must be clamped
    items, chunk = check_plan(p, ids, lens, Hkv)
    assert (items[:, 4] >= 0).sum() <= 32768


def test_kv_head_shards_take_identical_allocator_decisions():
    """the shards of a TP-sharded D-instance hold different KV heads of the SAME blocks, so their
    allocators must decide identically — same seed, same op sequence => same block lists, whatever the head count;
    and the sharding options validate their range."""
    rng = np.random.default_rng(11)
    full = host_pool(num_q_heads=32, num_kv_heads=8, head_dim=128, num_blocks=512, alloc_seed=5, max_requests=32)
    shards = [host_pool(num_q_heads=8, num_kv_heads=2, head_dim=128, num_blocks=512, alloc_seed=5, max_requests=32)
              for _ in range(4)]
    for r, s in enumerate(shards):
        s.set_option("src_kv_heads", 8)
        s.set_option("src_head_begin", 2 * r)
    live = []
    for step in range(60):
        if live and rng.random() < 0.3:
            victim = live.pop(int(rng.integers(len(live))))
            for p in [full] + shards:
                p.free([victim])
        else:
            uid, n = 1000 + step, int(rng.integers(1, 200))
            for p in [full] + shards:
                p.reserve([uid], [n])
            live.append(uid)
        for uid in live:
            want = full.block_table(uid)
            for s in shards:
                got = s.block_table(uid)
                assert np.array_equal(got[0], want[0]) and got[1] == want[1]
    with pytest.raises(kv.KVError):
        shards[0].set_option("src_head_begin", 7)            # heads [7, 9) do not exist in an 8-head source
    with pytest.raises(kv.KVError):
        full.set_option("src_kv_heads", 4)                   # narrower than the pool itself


def test_round2_entry_points_check_their_arguments_on_the_host():
    """kv_transfer / paged_decode_step_layers / kv_gather_bytes / config caps: refusals that need no GPU."""
    a, b = host_pool(), host_pool(num_blocks=64)
    a.reserve([1], [40])
    for dst, src, ids, status in [(a, a, ([2], [1]), B.KV_ERR_INVALID),                      # a pool cannot feed itself
                                  (b, host_pool(head_dim=128), ([2], [1]), B.KV_ERR_INVALID),  # geometry mismatch
                                  (b, host_pool(kv_dtype=B.KV_DTYPE_FP8_E4M3), ([2], [1]), B.KV_ERR_INVALID),
                                  (b, a, ([2], [1]), B.KV_ERR_NO_DEVICE)]:                   # host-only pools launch nothing
        with pytest.raises(kv.KVError) as e:
            B.kv_transfer(dst.handle, src.handle, ids[0], ids[1], 0, 2)
        assert e.value.status == status
    assert b.stats()["live_requests"] == 0 and a.block_table(1)[1] == 40
    with pytest.raises(kv.KVError) as e:
        B.paged_decode_step_layers(a.handle, 0, 2, [1], 256, 512, 768, 1024, 4096, 1024, 0.0, B.KV_STEP_RESERVE, 0)
    assert e.value.status == B.KV_ERR_NO_DEVICE and a.block_table(1)[1] == 40                 # nothing was reserved
    cfg = kv.PoolConfig(num_layers=2, num_q_heads=8, num_kv_heads=2, head_dim=64, num_blocks=8, max_requests=4,
                        max_blocks_per_request=4)
    assert B.kv_gather_bytes(cfg, 10) == 2 * 2 * 10 * 64 * 2
    cfg8 = kv.PoolConfig(**{**cfg.__dict__, "kv_dtype": B.KV_DTYPE_FP8_E4M3})
    assert B.kv_gather_bytes(cfg8, 10) == 2 * 2 * 10 * 64 + 4 * 2 * 2 * 10                    # codes (16-byte multiple) + scales
    assert B.kv_gather_bytes(cfg8, 3) == (2 * 2 * 3 * 64 + 15) // 16 * 16 + 4 * 2 * 2 * 3
    # a request may not exceed 131072 blocks: lengths stay inside int32 and the plan's 16:16 packing holds
    big = kv.PoolConfig(**{**cfg.__dict__, "max_requests": 1, "max_blocks_per_request": 131073})
    with pytest.raises(kv.KVError) as e:
        kv.kv_pool_required_bytes(big)
    assert e.value.status == B.KV_ERR_INVALID
    assert kv.kv_pool_required_bytes(kv.PoolConfig(**{**cfg.__dict__, "max_requests": 1, "max_blocks_per_request": 131072})) > 0
    # removed tuning values are refused, new ones accepted
    for key, val, ok in [("ring", 0, False), ("fp8_ring", 0, False), ("ring", 2, True), ("pdl", 0, True), ("pdl", 2, False)]:
        if ok:
            a.set_option(key, val)
        else:
            with pytest.raises(kv.KVError):
                a.set_option(key, val)


def test_library_is_the_one_built_from_this_tree():
    """binding refuses a libkvpool.so whose source hash differs from the sources in the tree (a stale binary
    would make every GPU test meaningless); the check is by content, so it survives a copy to another box."""
    from paper_2511_20982_b200 import build
    assert not build.stale()
    assert open(build.STAMP).read().strip() == build.source_hash()
    deps = list(build.DEPS)
    try:
        build.DEPS.append(os.path.join("..", "binding.py"))              # any change to what is hashed flips it
        assert build.stale()
    finally:
        build.DEPS[:] = deps
