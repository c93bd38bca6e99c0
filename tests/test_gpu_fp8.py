"""-m gpu parity of the FP8 (e4m3) KV pool through the C-ABI:
  * kv_ingest into an FP8 pool == oracle.scatter_fp8, BYTE-exact over the whole KV region (codes, scales,
    sentinel everywhere else), for one-shot, split and token-by-token ingests (per-token scales make a
    row's bytes independent of how it arrived);
  * paged_decode_attention over the FP8 pool == oracle.attention_fp8 (Eq. 1 on the dequantised values)
    within the bf16-output tolerance, for every split mode and GQA group size, including rows whose
    magnitudes span e^-6 .. e^6 (the V scale rides in the softmax reference, not in the f16 weights)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from gpu_harness import DEV, apply_options, compare_attention, dims_of, kv_src
from helpers import bf16_bits, bits_of, bits_to_f64

pytestmark = pytest.mark.gpu

# tc=0: the mma.sync kernel (attn_kernel<Fp8Tiles>), which head_dim-64 pools run whatever the option says
MODES = [dict(), dict(tc=0), dict(tc=0, min_chunk_blocks=1, items_per_slot=1024), dict(tc=0, min_chunk_blocks=3, items_per_slot=1024),
         dict(tc=0, min_chunk_blocks=2, items_per_slot=2, fuse_combine=0), dict(tc=0, min_chunk_blocks=5, items_per_slot=1, ctas_per_sm=1),
         dict(tc=0, pdl=0), dict(tc=0, pdl=0, min_chunk_blocks=2, items_per_slot=1024),
         dict(tc=0, tma=1), dict(tc=0, tma=1, min_chunk_blocks=1, items_per_slot=1024), dict(tc=0, tma=1, min_chunk_blocks=3, items_per_slot=2, fuse_combine=0),
         # tc=1: attn_tc_kernel (tcgen05 / TMEM / TMA, 128-token tiles): single tile, many tiles per unit, one block per chunk
         dict(tc=1), dict(tc=1, min_chunk_blocks=1, items_per_slot=1024), dict(tc=1, min_chunk_blocks=9, items_per_slot=1024),
         dict(tc=1, min_chunk_blocks=3, items_per_slot=2, fuse_combine=0), dict(tc=1, pdl=0, min_chunk_blocks=17, items_per_slot=1)]
SENT = 0xFF   # e4m3 NaN code / NaN scale bytes: an unmasked read poisons the output


def make_fp8_pool(L, Hq, Hkv, d, num_blocks, max_requests=16, max_len=4096, alloc_seed=11):
    cfg = kv.PoolConfig(num_layers=L, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d, num_blocks=num_blocks,
                        max_requests=max_requests, max_blocks_per_request=(max_len + 15) // 16, alloc_seed=alloc_seed,
                        kv_dtype=B.KV_DTYPE_FP8_E4M3)
    pool = kv.KVPool(cfg, device=DEV)
    assert pool.kv_bytes == L * num_blocks * Hkv * (32 * d + 128)
    pool.slab[: pool.kv_bytes].fill_(SENT)
    return pool


def pool_bytes(pool) -> np.ndarray:
    return pool.slab[: pool.kv_bytes].cpu().numpy()


def tb(bits):
    return torch.from_numpy(bits.view(np.int16).copy()).view(torch.bfloat16).to(DEV)


def wide_rows(rng, L, Hkv, n, d):
    """N(0,1) rows with per-row magnitudes e^U(-6, 6), a zero row and a row with one huge element."""
    x = rng.standard_normal((L, Hkv, n, d)) * np.exp(rng.uniform(-6, 6, (L, Hkv, n, 1)))
    if n > 3:
        x[:, :, 2] = 0.0
        x[:, :, 3, 5] = 3.0e4
    return bf16_bits(x)


@pytest.mark.parametrize("d,Hkv,L", [(128, 8, 2), (64, 2, 3), (128, 32, 1)])
def test_ingest_is_byte_exact(d, Hkv, L):
    rng = np.random.default_rng(d + Hkv)
    lens = [17, 64, 130, 255, 1, 16, 33]
    ids = list(range(100, 100 + len(lens)))
    NB = sum((n + 15) // 16 for n in lens) + 5
    K = [wide_rows(rng, L, Hkv, n, d) for n in lens]
    V = [wide_rows(rng, L, Hkv, n, d) for n in lens]
    for mode in ("once", "split", "tokens"):
        pool = make_fp8_pool(L, Hkv, Hkv, d, NB)
        slab = oracle.new_slab_fp8(dims_of(pool), SENT)
        if mode == "once":
            pool.ingest(ids, [tb(k) for k in K], [tb(v) for v in V])
        else:
            for i, n in enumerate(lens):
                cuts = [0, n] if n < 3 else ([0, n // 3, n // 3 + 1, n] if mode == "split" else list(range(n + 1)))
                for a, b in zip(cuts[:-1], cuts[1:]):
                    pool.ingest([ids[i]], [tb(K[i][:, :, a:b].copy())], [tb(V[i][:, :, a:b].copy())])
        torch.cuda.synchronize()
        for i, n in enumerate(lens):
            oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(ids[i])[0], 0, K[i], V[i])
        got = pool_bytes(pool)
        assert np.array_equal(got, slab), f"{mode}: FP8 ingest is not byte-exact ({int((got != slab).sum())} bytes differ)"
        pool.close()


@pytest.mark.parametrize("opts", MODES)
@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 32, 128), (64, 8, 128), (32, 8, 128)])
def test_attention_matches_oracle(Hq, Hkv, d, opts):
    rng = np.random.default_rng(7)
    lens = [17, 64, 130, 255, 1, 16, 33, 700, 1900, 5]
    ids = list(range(300, 300 + len(lens)))
    pool = make_fp8_pool(1, Hq, Hkv, d, sum((n + 15) // 16 for n in lens) + 8)
    apply_options(pool, opts)
    w = W.Workload("fp8", 1, Hq, Hkv, d, len(lens), None, 99, max_len=4096)
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    for uid, n, (k, v) in zip(ids, lens, srcs):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(uid)[0], 0, bits_of(k), bits_of(v))
    q = W.q_values(w.seed, 1, 0, len(lens), Hq, d, DEV)
    out = pool.attention(0, ids, q)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bytes(pool), slab)
    lists = [pool.block_table(u)[0] for u in ids]
    want = oracle.attention_fp8(slab, dims_of(pool), 0, Hq, lists, lens, bits_of(q))
    compare_attention(out, want)
    # the quantisation itself: close to the bf16 oracle on the unquantised values (sanity, loose)
    s16 = oracle.new_slab(dims_of(pool), 0)
    for uid, n, (k, v) in zip(ids, lens, srcs):
        oracle.scatter(s16, dims_of(pool), pool.block_table(uid)[0], 0, bits_of(k), bits_of(v))
    exact = oracle.attention(s16, dims_of(pool), 0, Hq, lists, lens, bits_of(q))
    assert np.abs(want - exact).max() < 0.15 and np.abs(want - exact).mean() < 0.01


def test_default_picks_the_kernel_per_batch():
    """Option tc = 2 (default): attn_tc_kernel unless most of the batch's requests are one or two tiles long."""
    Hq, Hkv, d = 32, 8, 128
    lens = [40, 100, 200, 3000, 5000, 700, 33, 256]
    ids = list(range(len(lens)))
    pool = make_fp8_pool(1, Hq, Hkv, d, sum((n + 15) // 16 for n in lens) + 4, max_len=8192)
    w = W.Workload("fp8a", 1, Hq, Hkv, d, len(lens), None, 321, max_len=8192)
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    for uid, n, (k, v) in zip(ids, lens, srcs):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(uid)[0], 0, bits_of(k), bits_of(v))
    q = W.q_values(w.seed, 1, 0, len(lens), Hq, d, DEV)
    for sel, want_tc in (([0, 1, 2, 3, 6, 7], False), ([3, 4, 5, 0], True), (list(range(8)), False), ([3, 4, 5, 0, 1, 2], True)):
        before = pool.counter("attn_tc_launches")
        out = pool.attention(0, [ids[i] for i in sel], q[sel].contiguous())
        torch.cuda.synchronize()
        assert (pool.counter("attn_tc_launches") - before == 1) == want_tc, sel
        lists = [pool.block_table(ids[i])[0] for i in sel]
        compare_attention(out, oracle.attention_fp8(slab, dims_of(pool), 0, Hq, lists, [lens[i] for i in sel], bits_of(q[sel].contiguous())))


@pytest.mark.parametrize("opts", [dict(tc=0), dict(tc=1), dict(tc=1, min_chunk_blocks=9, items_per_slot=1024)])
@pytest.mark.parametrize("G", [2, 3, 5, 6, 7])
def test_attention_every_group_size(G, opts):
    """GQA groups that do not fill the 8 MMA columns (mma.sync kernel) / the 8 head rows of Q8 and P (tcgen05 kernel)."""
    Hkv, d = 2, 128
    Hq = G * Hkv
    lens = [1, 16, 17, 129, 1000, 2049]
    ids = list(range(40, 40 + len(lens)))
    pool = make_fp8_pool(1, Hq, Hkv, d, sum((n + 15) // 16 for n in lens) + 4)
    apply_options(pool, opts)
    w = W.Workload("fp8g", 1, Hq, Hkv, d, len(lens), None, 100 + G, max_len=4096)
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    for uid, n, (k, v) in zip(ids, lens, srcs):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(uid)[0], 0, bits_of(k), bits_of(v))
    q = W.q_values(w.seed, 1, 0, len(lens), Hq, d, DEV)
    out = pool.attention(0, ids, q)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bytes(pool), slab)
    lists = [pool.block_table(u)[0] for u in ids]
    compare_attention(out, oracle.attention_fp8(slab, dims_of(pool), 0, Hq, lists, lens, bits_of(q)))


@pytest.mark.parametrize("opts", [dict(tc=0), dict(tc=0, min_chunk_blocks=2, items_per_slot=1024), dict(tc=0, tma=1), dict(tc=1),
                                  dict(tc=1, min_chunk_blocks=2, items_per_slot=1024)])
def test_attention_wide_dynamic_range(opts):
    """Row magnitudes from e^-6 to e^6 in K and V, scaled-up queries, a zero row and an outlier element."""
    rng = np.random.default_rng(8)
    Hq, Hkv, d = 16, 4, 128
    lens = [40, 333, 1000]
    ids = [1, 2, 3]
    pool = make_fp8_pool(1, Hq, Hkv, d, 100)
    apply_options(pool, opts)
    K = [bf16_bits(rng.standard_normal((1, Hkv, n, d)) * 0.3) for n in lens]      # keep the scores moderate
    V = [wide_rows(rng, 1, Hkv, n, d) for n in lens]
    pool.ingest(ids, [tb(k) for k in K], [tb(v) for v in V])
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    for uid, k, v in zip(ids, K, V):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(uid)[0], 0, k, v)
    for qscale in (1.0, 2.0 ** 40, 2.0 ** -40):
        qb = bf16_bits(rng.standard_normal((3, Hq, d)) * qscale)
        sm = 0.0883883 / qscale                                   # exact power-of-two compensation in the scale
        out = pool.attention(0, ids, tb(qb), sm_scale=sm)
        torch.cuda.synchronize()
        lists = [pool.block_table(u)[0] for u in ids]
        want = oracle.attention_fp8(slab, dims_of(pool), 0, Hq, lists, lens, qb, scale=float(np.float32(sm)))
        got = bits_to_f64(bits_of(out))
        assert np.all(np.isfinite(got))
        err = np.abs(got - want)
        tol = 2.0 ** -7 * np.abs(want) + 1e-3 * np.sqrt((want ** 2).mean(axis=-1, keepdims=True)) + 1e-30
        assert np.all(err <= tol), float((err / tol).max())


def test_decode_loop_appends_with_ingest():
    Hq, Hkv, d, L = 32, 8, 128, 2
    lens = [15, 16, 31, 500, 1]
    ids = list(range(5))
    w = W.Workload("fp8d", L, Hq, Hkv, d, len(lens), None, 5, max_len=1024)
    pool = make_fp8_pool(L, Hq, Hkv, d, 64)
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    for u, n, (k, v) in zip(ids, lens, srcs):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(u)[0], 0, bits_of(k), bits_of(v))
    for step in range(3):
        new = [kv_src(w, u, n + step, n + step + 1, DEV) for u, n in zip(ids, lens)]
        pool.ingest(ids, [s[0] for s in new], [s[1] for s in new])
        for u, n, (k, v) in zip(ids, lens, new):
            oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(u)[0], n + step, bits_of(k), bits_of(v))
        for l in range(L):
            q = W.q_values(w.seed, step, l, len(ids), Hq, d, DEV)
            out = pool.attention(l, ids, q)
            torch.cuda.synchronize()
            lists = [pool.block_table(u)[0] for u in ids]
            want = oracle.attention_fp8(slab, dims_of(pool), l, Hq, lists, [n + step + 1 for n in lens], bits_of(q))
            compare_attention(out, want)
    assert np.array_equal(pool_bytes(pool), slab)


@pytest.mark.parametrize("Hkv,d", [(2, 64), (8, 128)])
def test_gather_fp8_returns_stored_codes_and_scales(Hkv, d):
    """kv_gather on an FP8 pool: the stored codes and row scales, contiguous, byte for byte == oracle.gather_fp8
    (the inverse of ingest's relocation, not of its quantisation); the pool is not modified."""
    L, lens = 2, [1, 16, 45, 300]
    pool = make_fp8_pool(L, Hkv * 4, Hkv, d, 40)
    w = W.Workload("fp8g", L, Hkv * 4, Hkv, d, len(lens), None, 5, max_len=512)
    ids = [11, 12, 13, 14]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in zip(ids, lens)]
    pool.ingest(ids, [x[0] for x in srcs], [x[1] for x in srcs])
    torch.cuda.synchronize()
    before = pool_bytes(pool).copy()
    for u, n in zip(ids, lens):
        assert B.kv_gather_bytes(pool.cfg, n) == (L * Hkv * n * d + 15) // 16 * 16 + 4 * L * Hkv * n
        kc, ks, vc, vs = pool.gather(u)
        torch.cuda.synchronize()
        wkc, wks, wvc, wvs = oracle.gather_fp8(before, dims_of(pool), pool.block_table(u)[0], n)
        assert np.array_equal(kc.cpu().numpy(), wkc) and np.array_equal(vc.cpu().numpy(), wvc)
        assert np.array_equal(ks.cpu().numpy().view(np.uint32), wks.view(np.uint32))
        assert np.array_equal(vs.cpu().numpy().view(np.uint32), wvs.view(np.uint32))
    assert np.array_equal(pool_bytes(pool), before)


@pytest.mark.parametrize("opts", [dict(), dict(tc=0), dict(tc=0, min_chunk_blocks=1, items_per_slot=1024), dict(tc=0, min_chunk_blocks=3, items_per_slot=2),
                                  dict(tc=0, tma=1), dict(tc=0, tma=1, min_chunk_blocks=1, items_per_slot=1024),
                                  dict(tc=1), dict(tc=1, min_chunk_blocks=1, items_per_slot=1024), dict(tc=1, min_chunk_blocks=9, items_per_slot=2)])
@pytest.mark.parametrize("Hq,Hkv,d", [(32, 8, 128), (8, 2, 64), (32, 32, 128)])
def test_fused_decode_step_quantises_like_ingest(Hq, Hkv, d, opts):
    """paged_decode_step on an FP8 pool: the appended row's codes and scales are the bytes kv_ingest would have
    written (whole pool == oracle.scatter_fp8), and the output is attention over len + 1 tokens."""
    L = 2
    lens = [15, 16, 31, 500, 1, 0, 1029, 47]          # fill a block, open a new one, empty request, split contexts
    ids = list(range(len(lens)))
    w = W.Workload("fp8s", L, Hq, Hkv, d, len(lens), None, 6, max_len=2048)
    pool = make_fp8_pool(L, Hq, Hkv, d, 160)
    apply_options(pool, opts)
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    live = [(u, n) for u, n in zip(ids, lens) if n]
    srcs = [kv_src(w, u, 0, n, DEV) for u, n in live]
    pool.ingest([u for u, _ in live], [s[0] for s in srcs], [s[1] for s in srcs])
    for (u, n), (k, v) in zip(live, srcs):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(u)[0], 0, bits_of(k), bits_of(v))
    for step in range(3):
        pool.reserve(ids, [1] * len(ids))
        n_launch = pool.launches
        for l in range(L):
            new = [kv_src(w, u, n + step, n + step + 1, DEV, layer_begin=l, layer_count=1) for u, n in zip(ids, lens)]
            k_new = torch.stack([s[0][0, :, 0] for s in new]).contiguous()          # [B][Hkv][d]
            v_new = torch.stack([s[1][0, :, 0] for s in new]).contiguous()
            q = W.q_values(w.seed, step, l, len(ids), Hq, d, DEV)
            out = pool.decode_step(l, ids, q, k_new, v_new)
            torch.cuda.synchronize()
            for u, n, (k, v) in zip(ids, lens, new):
                oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(u)[0], n + step, bits_of(k), bits_of(v), layer_begin=l)
            lists = [pool.block_table(u)[0] for u in ids]
            want = oracle.attention_fp8(slab, dims_of(pool), l, Hq, lists, [n + step + 1 for n in lens], bits_of(q))
            compare_attention(out, want)
        assert pool.launches - n_launch == L                          # one launch per layer
        assert np.array_equal(pool_bytes(pool), slab), f"step {step}: fused FP8 append is not byte-exact"


@pytest.mark.parametrize("opts", [dict(), dict(min_chunk_blocks=1, items_per_slot=1024), dict(min_chunk_blocks=3, items_per_slot=2),
                                  dict(tma=1), dict(tma=1, min_chunk_blocks=2, items_per_slot=1024)])
@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 32, 128), (64, 8, 128), (6, 2, 64)])
def test_varlen_attention_on_fp8_pool(Hq, Hkv, d, opts):
    """In-place prefill rows + decode rows over an FP8 pool == oracle.attention_varq_fp8."""
    lens = [17, 64, 130, 255, 1, 16, 33, 700, 1100, 5, 48, 100]
    q_lens = [17, 1, 130, 7, 1, 16, 1, 1, 300, 5, 31, 100]
    ids = list(range(700, 700 + len(lens)))
    pool = make_fp8_pool(1, Hq, Hkv, d, sum((n + 15) // 16 for n in lens) + 8)
    apply_options(pool, opts)
    w = W.Workload("fp8v", 1, Hq, Hkv, d, len(lens), None, 98, max_len=4096)
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    slab = oracle.new_slab_fp8(dims_of(pool), SENT)
    for uid, n, (k, v) in zip(ids, lens, srcs):
        oracle.scatter_fp8(slab, dims_of(pool), pool.block_table(uid)[0], 0, bits_of(k), bits_of(v))
    q = W.q_values(w.seed, 2, 0, sum(q_lens), Hq, d, DEV)
    out = pool.varlen_attention(0, ids, q_lens, q)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bytes(pool), slab)
    lists = [pool.block_table(u)[0] for u in ids]
    want = oracle.attention_varq_fp8(slab, dims_of(pool), 0, Hq, lists, lens, q_lens, bits_of(q))
    compare_attention(out, want)
