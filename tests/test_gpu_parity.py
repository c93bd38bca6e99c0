"""GPU parity: the CUDA path (through the C-ABI) against the oracle, element by element, on the
same seeded inputs.  Ingest / gather: bit-exact, whole slab.  Attention: max abs <= 1e-2 and
mean abs <= 1e-3 (BASELINE.json north_star) plus max err / rms <= 3e-2 per request (A9), and the
structured pins P1-P13 of SURVEY §8(c) re-run on the GPU where they are much stricter."""
import json
import math
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import workloads as W
from gpu_harness import (apply_options, DEV, NAN_BITS, compare_attention, dims_of, kv_src, make_pool, oracle_attention,
                         oracle_ingest, oracle_slab, pool_bits)
from helpers import bf16_bits, bits_of, bits_to_f64

pytestmark = pytest.mark.gpu

SPLIT_MODES = [dict(), dict(min_chunk_blocks=1, items_per_slot=1024), dict(min_chunk_blocks=3, items_per_slot=1024),
               dict(min_chunk_blocks=2, items_per_slot=1024, fuse_combine=0),
               dict(min_chunk_blocks=1, items_per_slot=2), dict(min_chunk_blocks=5, items_per_slot=1),
               dict(min_chunk_blocks=1, items_per_slot=1024, ctas_per_sm=1),
               dict(ring=2), dict(pdl=0), dict(pdl=0, min_chunk_blocks=1, items_per_slot=1024), dict(ring=2, min_chunk_blocks=3, items_per_slot=1024),
               dict(tma=1), dict(tma=1, min_chunk_blocks=1, items_per_slot=1024), dict(tma=1, min_chunk_blocks=3, items_per_slot=2, pdl=0), dict(side_upload=0), dict(side_upload=0, min_chunk_blocks=1, items_per_slot=1024)]


def from_bits(bits: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(bits.view(np.int16).copy()).view(torch.bfloat16).to(DEV)


def run_structured(Hq, Hkv, d, lens, K, V, q, scale=None, num_blocks=None, options=None, alloc_seed=7, L=1):
    """K[r], V[r]: float [L][Hkv][n][d]; q float [B][Hq][d].  Returns (gpu bf16 out, oracle f64 out) of layer L-1."""
    w = W.Workload("structured", L, Hq, Hkv, d, len(lens), None, 0, max_len=max(lens) + 16)
    nb = num_blocks or sum((n + 15) // 16 for n in lens) + 8
    pool = make_pool(w, nb, alloc_seed=alloc_seed)
    apply_options(pool, options)
    slab = oracle_slab(pool)
    ids = list(range(500, 500 + len(lens)))
    kb = [bf16_bits(k) for k in K]
    vb = [bf16_bits(v) for v in V]
    pool.ingest(ids, [from_bits(k) for k in kb], [from_bits(v) for v in vb])
    for i, uid in enumerate(ids):
        oracle.scatter(slab, dims_of(pool), pool.block_table(uid)[0], 0, kb[i], vb[i])
    qb = bf16_bits(q)
    out = pool.attention(L - 1, ids, from_bits(qb), sm_scale=0.0 if scale is None else scale)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)
    want = oracle.attention(slab, dims_of(pool), L - 1, Hq, [pool.block_table(u)[0] for u in ids], lens, qb, scale=scale)
    return out, want


# ---------------------------------------------------------------------------------------------
# config 1 (BASELINE.json configs[0]) — in full
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("opts", SPLIT_MODES)
def test_cfg1_tiny_full(opts):
    w = W.CONFIGS["cfg1_tiny"]
    lens = [int(x) for x in w.draw_lengths()]
    assert lens == [17, 64, 130, 255]
    ids = [10, 11, 12, 13]
    pool = make_pool(w, 128, alloc_seed=w.seed)
    apply_options(pool, opts)
    slab = oracle_slab(pool)
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    for uid, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, uid, 0, n)
    torch.cuda.synchronize()
    assert pool.stats()["blocks_free"] == 128 - 31
    assert np.array_equal(pool_bits(pool), slab), "ingest is not bit-exact over the whole slab"
    for uid, (k, v) in zip(ids, srcs):                     # P10: ingest o gather = identity
        gk, gv = pool.gather(uid)
        assert torch.equal(gk.view(torch.int16), k.view(torch.int16)) and torch.equal(gv.view(torch.int16), v.view(torch.int16))
    assert np.array_equal(pool_bits(pool), slab), "gather modified the pool"
    q = W.q_values(w.seed, 0, 0, 4, w.num_q_heads, w.head_dim, DEV)
    out = pool.attention(0, ids, q)
    want = oracle_attention(slab, pool, 0, ids, q)
    compare_attention(out, want)
    # a subset / permuted batch uses the same pool
    out2 = pool.attention(0, [13, 10], q[:2].contiguous())
    want2 = oracle_attention(slab, pool, 0, [13, 10], q[:2])
    compare_attention(out2, want2)

    # one-by-one ingest gives the same slab (and P4: another placement gives the same output)
    pool_b = make_pool(w, 128, alloc_seed=w.seed + 1)
    apply_options(pool_b, opts)
    for uid, (k, v) in zip(ids, srcs):
        pool_b.ingest([uid], [k], [v])
    slab_b = oracle_slab(pool_b)
    for uid, n in zip(ids, lens):
        oracle_ingest(slab_b, pool_b, w, uid, 0, n)
    out_b = pool_b.attention(0, ids, q)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool_b), slab_b)
    assert not np.array_equal(pool.block_table(13)[0], pool_b.block_table(13)[0])
    assert torch.equal(out_b.view(torch.int16), out.view(torch.int16)), "output depends on physical placement"


def test_p12_append_paths_are_bit_identical():
    """n tokens at once == split ingests (incl. mid-block) == single-token appends == layer-sliced."""
    w = W.CONFIGS["cfg1_tiny"].scaled(num_layers=3)
    n = 77
    k, v = kv_src(w, 1, 0, n, DEV)
    ref = None
    for cuts in ([0, n], [0, 5, n], [0, 16, 32, n], [0, 17, 18, 50, n], list(range(n + 1))):
        pool = make_pool(w, 32, alloc_seed=3)
        for a, b in zip(cuts, cuts[1:]):
            pool.ingest([1], [k[:, :, a:b].contiguous()], [v[:, :, a:b].contiguous()])
        torch.cuda.synchronize()
        bits = pool_bits(pool).copy()
        if ref is None:
            ref = bits
            slab = oracle_slab(pool)
            oracle_ingest(slab, pool, w, 1, 0, n)
            assert np.array_equal(ref, slab)
        assert np.array_equal(bits, ref), cuts
    pool = make_pool(w, 32, alloc_seed=3)
    for l in range(3):                                      # producer streams KV layer by layer
        pool.ingest([1], [k[l:l + 1].contiguous()], [v[l:l + 1].contiguous()], layer_begin=l, layer_count=1)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), ref)
    with pytest.raises(kv.KVError):                         # continuation must match the reservation
        pool.ingest([1], [k[1:2, :, :5].contiguous()], [v[1:2, :, :5].contiguous()], layer_begin=1, layer_count=1)


def test_ingest_errors_change_nothing():
    w = W.CONFIGS["cfg1_tiny"]
    pool = make_pool(w, 8, max_requests=4, alloc_seed=5)
    k, v = kv_src(w, 1, 0, 100, DEV)
    pool.ingest([1], [k], [v])                              # 7 of 8 blocks
    torch.cuda.synchronize()
    before = pool_bits(pool).copy()
    k2, v2 = kv_src(w, 2, 0, 40, DEV)
    with pytest.raises(kv.KVError) as e:
        pool.ingest([2], [k2], [v2])                        # needs 3, 1 free
    assert e.value.status == kv.binding.KV_ERR_NO_BLOCKS
    with pytest.raises(kv.KVError):
        pool.ingest([2, 2], [k2, k2], [v2, v2])
    with pytest.raises(kv.KVError):                         # misaligned source pointer
        kv.kv_ingest(pool.handle, [3], [4], [k2.data_ptr() + 2], [v2.data_ptr()], 0, 1)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), before) and pool.stats()["live_requests"] == 1
    q = W.q_values(1, 0, 0, 1, w.num_q_heads, w.head_dim, DEV)
    with pytest.raises(kv.KVError):
        pool.attention(0, [2], q)                           # unknown request
    pool.reserve([4], [0])
    with pytest.raises(kv.KVError):
        pool.attention(0, [4], q)                           # empty context (A11)
    pool.free([1])                                          # free then reuse
    pool.ingest([2], [k2], [v2])
    out = pool.attention(0, [2], q)
    slab = before.copy()
    oracle_ingest(slab, pool, w, 2, 0, 40)
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)            # stale bytes of request 1 remain, never read
    compare_attention(out, oracle_attention(slab, pool, 0, [2], q))


# ---------------------------------------------------------------------------------------------
# structured pins on the GPU
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("d", [64, 128])
def test_p7_hand_cases_on_gpu(d):
    with open(os.path.join(os.path.dirname(__file__), "golden", "hand_cases.json")) as f:
        cases = json.load(f)["cases"]
    for case in cases:
        pad = lambda rows: np.array([r + [0] * (d - len(r)) for r in rows], dtype=np.float64)
        K, V, q = pad(case["K"]), pad(case["V"]), pad([case["q"]])
        out, want = run_structured(1, 1, d, [len(case["K"])], [K[None, None]], [V[None, None]], q[None],
                                   scale=math.log(2.0))
        got = bits_to_f64(bits_of(out))[0, 0]
        assert np.allclose(want[0, 0], pad([case["out"]])[0], atol=1e-13)
        assert np.allclose(got, pad([case["out"]])[0], rtol=0, atol=2 ** -6), case["name"]  # 1/3, 1/7 in bf16


@pytest.mark.parametrize("Hq,Hkv,d", [(8, 2, 64), (32, 32, 128), (64, 8, 128)])
def test_p1_single_token_returns_v_bits(Hq, Hkv, d):
    rng = np.random.default_rng(1)
    lens = [1, 1, 1]
    K = [rng.standard_normal((1, Hkv, 1, d)) for _ in lens]
    V = [rng.standard_normal((1, Hkv, 1, d)) for _ in lens]
    out, want = run_structured(Hq, Hkv, d, lens, K, V, rng.standard_normal((3, Hq, d)))
    G = Hq // Hkv
    got = bits_of(out)
    for r in range(3):
        for h in range(Hq):
            assert np.array_equal(got[r, h], bf16_bits(V[r])[0, h // G, 0]), "n = 1 must return V_0 bit-exactly"


@pytest.mark.parametrize("opts", SPLIT_MODES)
@pytest.mark.parametrize("d", [64, 128])
def test_p2_p5_p8_closed_forms(d, opts):
    rng = np.random.default_rng(2)
    Hq, Hkv = 8, 2
    lens = [1, 15, 16, 17, 64, 130, 255, 700]
    K = [rng.standard_normal((1, Hkv, n, d)) for n in lens]
    V = []
    for n in lens:
        v = np.zeros((1, Hkv, n, d))
        v[..., 0] = 1.0                                          # P5: weights sum to 1
        v[..., 1] = (np.arange(n) % 256)[None, None, :]          # P2: every token counted once
        v[..., 2] = (np.arange(n) % 7 == 3)
        v[..., 3] = np.arange(Hkv)[None, :, None]                # P8: GQA map
        V.append(v)
    out, want = run_structured(Hq, Hkv, d, lens, K, V, np.zeros((len(lens), Hq, d)), options=opts)
    got = bits_to_f64(bits_of(out))
    for r, n in enumerate(lens):
        for h in range(Hq):
            assert abs(got[r, h, 0] - 1.0) <= 2 ** -8
            m1 = np.mean(np.arange(n) % 256)
            assert abs(got[r, h, 1] - m1) <= max(m1, 1) * 2 ** -7, (n, got[r, h, 1], m1)
            assert abs(got[r, h, 2] - np.mean(np.arange(n) % 7 == 3)) <= 2 ** -8
            assert abs(got[r, h, 3] - h // (Hq // Hkv)) <= 2 ** -8
            assert np.all(got[r, h, 4:] == 0)
    # values reach 127.5, where a bf16 ulp is 0.5: the absolute bar does not apply, a relative one does
    assert np.all(np.abs(got - want) <= 2 ** -7 * np.maximum(np.abs(want), 1.0))
    # P8 with random q as well
    out, want = run_structured(Hq, Hkv, d, lens, K, V, rng.standard_normal((len(lens), Hq, d)), options=opts)
    got = bits_to_f64(bits_of(out))
    for h in range(Hq):
        assert np.all(np.abs(got[:, h, 3] - h // (Hq // Hkv)) <= 2 ** -7)
        assert np.all(np.abs(got[:, h, 0] - 1.0) <= 2 ** -7)


@pytest.mark.parametrize("opts", SPLIT_MODES[:2] + [dict(tma=1), dict(tma=1, min_chunk_blocks=1, items_per_slot=1024)])
def test_p3_needle_every_boundary(opts):
    d, n = 128, 1040
    rng = np.random.default_rng(3)
    positions = [0, 1, 15, 16, 17, 31, 32, 47, 48, 255, 256, 511, 512, 513, 1023, 1024, 1039]
    qf = np.zeros(d); qf[0] = 16.0                              # scale 1/sqrt(128) -> score = sqrt(2) * K[t][0]
    K, V, lens = [], [], []
    for pos in positions:                                       # one request per needle position
        k = np.zeros((1, 1, n, d)); k[0, 0, :, 1:] = rng.standard_normal((n, d - 1))
        k[0, 0, pos, 0] = 32.0                                  # needle score ~45 above the rest
        v = np.zeros((1, 1, n, d)); v[0, 0, :, 0] = np.arange(n) % 128; v[0, 0, :, 1] = np.arange(n) // 128
        K.append(k); V.append(v); lens.append(n)
    q = np.broadcast_to(qf, (len(positions), 1, d)).copy()
    out, want = run_structured(1, 1, d, lens, K, V, q, options=opts)
    got = bits_to_f64(bits_of(out))
    # the other 1039 tokens weigh e^-45 each: the exact answer is V_needle + O(1e-15), which bf16
    # keeps as a tiny non-zero where V_needle is 0 — hence a 1e-9 band instead of equality
    for r, pos in enumerate(positions):
        assert abs(got[r, 0, 0] - pos % 128) <= 1e-9 and abs(got[r, 0, 1] - pos // 128) <= 1e-9, (pos, got[r, 0, :2])
        assert np.all(np.abs(got[r, 0] - want[r, 0]) <= 2 ** -7 * np.abs(want[r, 0]) + 1e-30)


def test_p13_large_scores_do_not_overflow():
    rng = np.random.default_rng(13)
    d, n = 64, 300
    K = np.zeros((1, 1, n, d)); K[..., :32] = rng.standard_normal((1, 1, n, 32)); K[..., 40] = 640.0
    V = rng.standard_normal((1, 1, n, d))
    q = np.zeros((1, 1, d)); q[..., :32] = rng.standard_normal((1, 1, 32)); q[..., 40] = 8.0   # +640 on every score
    out, want = run_structured(1, 1, d, [n], [K], [V], q)
    compare_attention(out, want)
    K0 = K.copy(); K0[..., 40] = 0.0
    out0, want0 = run_structured(1, 1, d, [n], [K0], [V], q)
    assert np.allclose(want, want0, atol=1e-9)
    Kb = np.zeros((1, 1, n, d)); Kb[0, 0, 7, 0] = 5000.0; Kb[0, 0, 9, 0] = -5000.0
    qb = np.zeros((1, 1, d)); qb[0, 0, 0] = 8.0
    out, want = run_structured(1, 1, d, [n], [Kb], [V], qb)
    assert np.array_equal(bits_of(out)[0, 0], bf16_bits(V)[0, 0, 7])


# ---------------------------------------------------------------------------------------------
# scaled-down copies of configs 2-5: several tiles, ragged tails, the configs' procedures
# ---------------------------------------------------------------------------------------------

def ingest_all(pool, w, ids, lens, slab):
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    for uid, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, uid, 0, n)


def append_one(pool, w, ids, lens, slab):
    srcs = [kv_src(w, uid, n, n + 1, DEV) for uid, n in zip(ids, lens)]
    pool.ingest(ids, [s[0] for s in srcs], [s[1] for s in srcs])
    for uid, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, uid, n, n + 1)


@pytest.mark.parametrize("opts", SPLIT_MODES[:2] + [dict(tma=1)])
def test_cfg2_scaled_decode_steps(opts):
    """7B-MHA shape (G = 1): ingest, then decode steps = append one token per request + attend."""
    w = W.CONFIGS["cfg2_7b_mha"].scaled(batch=12)
    lens = [int(x) for x in w.draw_lengths()]
    lens[:4] = [511, 527, 1024, 2047]                          # block-boundary crossings within the steps
    ids = list(range(12))
    pool = make_pool(w, sum((n + 24) // 16 + 1 for n in lens), alloc_seed=w.seed)
    apply_options(pool, opts)
    slab = oracle_slab(pool)
    ingest_all(pool, w, ids, lens, slab)
    for step in range(4):
        append_one(pool, w, ids, lens, slab)
        lens = [n + 1 for n in lens]
        q = W.q_values(w.seed, step, 0, len(ids), w.num_q_heads, w.head_dim, DEV)
        out = pool.attention(0, ids, q)
        compare_attention(out, oracle_attention(slab, pool, 0, ids, q))
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)


def test_cfg3_scaled_steady_state():
    """8B-GQA shape, several layers: per step free the oldest, ingest new, append, attend every layer."""
    w = W.CONFIGS["cfg3_8b_gqa"].scaled(num_layers=3, batch=24, ingest_per_step=3)
    lens_all = [int(x) for x in w.draw_lengths(40)]
    lens_all = [min(n, 3000) for n in lens_all]
    pool = make_pool(w, 6000, max_requests=64, alloc_seed=w.seed)
    slab = oracle_slab(pool)
    live = list(range(24))
    lens = {i: lens_all[i] for i in live}
    ingest_all(pool, w, live, [lens[i] for i in live], slab)
    nxt = 24
    for step in range(3):
        pool.free(live[:3])
        live = live[3:]
        new = list(range(nxt, nxt + 3)); nxt += 3
        for i in new:
            lens[i] = lens_all[i]
        ingest_all(pool, w, new, [lens[i] for i in new], slab)
        live += new
        append_one(pool, w, live, [lens[i] for i in live], slab)
        for i in live:
            lens[i] += 1
        launches = pool.launches
        for layer in range(3):
            q = W.q_values(w.seed, step, layer, len(live), w.num_q_heads, w.head_dim, DEV)
            out = pool.attention(layer, live, q)
            compare_attention(out, oracle_attention(slab, pool, layer, live, q))
        assert pool.launches - launches <= 6                    # main (+ combine) per layer
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)


def test_cfg4_scaled_fragmented_long_context():
    """70B shape (G = 8): interleaved slice-wise ingest on a permuted pool, long contexts, many chunks."""
    w = W.CONFIGS["cfg4_70b_long"].scaled(batch=6)
    lens = [4096, 5000, 8191, 6017, 4100, 7000]
    ids = list(range(6))
    pool = make_pool(w, sum((n + 15) // 16 for n in lens) + 64, alloc_seed=w.seed, max_len=8192 + 64)
    slab = oracle_slab(pool)
    done = [0] * 6
    while any(d < n for d, n in zip(done, lens)):               # round-robin 64-token slices => fragmentation
        batch = [(i, d, min(d + 64, n)) for i, (d, n) in enumerate(zip(done, lens)) if d < n]
        srcs = [kv_src(w, ids[i], a, b, DEV) for i, a, b in batch]
        pool.ingest([ids[i] for i, _, _ in batch], [s[0] for s in srcs], [s[1] for s in srcs])
        for i, a, b in batch:
            done[i] = b
    for uid, n in zip(ids, lens):
        oracle_ingest(slab, pool, w, uid, 0, n)
    bt = pool.block_table(0)[0]
    assert np.mean(np.abs(np.diff(bt)) == 1) < 0.05             # consecutive logical blocks are not adjacent
    torch.cuda.synchronize()
    assert np.array_equal(pool_bits(pool), slab)
    for opts in SPLIT_MODES[:2] + [dict(min_chunk_blocks=64, items_per_slot=1), dict(tma=1)]:
        apply_options(pool, opts)
        q = W.q_values(w.seed, 0, 0, len(ids), w.num_q_heads, w.head_dim, DEV)
        out = pool.attention(0, ids, q)
        compare_attention(out, oracle_attention(slab, pool, 0, ids, q))


def test_cfg5_scaled_bimodal_burst_on_second_stream():
    """Stress shape: bimodal lengths in one launch; a burst is ingested on stream B while stream A attends."""
    w = W.CONFIGS["cfg5_stress"].scaled(num_layers=2, batch=48, ingest_per_step=8,
                                        length_law=W.lengths_bimodal(0.2, (64, 256), (2048, 4096)))
    lens = [int(x) for x in w.draw_lengths()]
    assert min(lens) <= 256 and max(lens) >= 2048
    ids = list(range(48))
    pool = make_pool(w, 8000, max_requests=128, alloc_seed=w.seed, max_len=4096 + 64)
    slab = oracle_slab(pool)
    ingest_all(pool, w, ids, lens, slab)
    torch.cuda.synchronize()
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    burst_lens = [int(x) for x in w.draw_lengths(8, salt=1)]
    burst = list(range(100, 108))
    srcs = [kv_src(w, uid, 0, n, DEV) for uid, n in zip(burst, burst_lens)]
    qs = [W.q_values(w.seed, 0, layer, 48, w.num_q_heads, w.head_dim, DEV) for layer in range(2)]
    torch.cuda.synchronize()
    outs = []
    with torch.cuda.stream(sb):
        pool.ingest(burst, [s[0] for s in srcs], [s[1] for s in srcs], stream=sb)
    with torch.cuda.stream(sa):
        for layer in range(2):
            outs.append(pool.attention(layer, ids, qs[layer], stream=sa))
    torch.cuda.synchronize()
    for layer in range(2):
        compare_attention(outs[layer], oracle_attention(slab, pool, layer, ids, qs[layer]))
    for uid, n in zip(burst, burst_lens):
        oracle_ingest(slab, pool, w, uid, 0, n)
    assert np.array_equal(pool_bits(pool), slab)
    allr = ids + burst
    q = W.q_values(w.seed, 1, 1, len(allr), w.num_q_heads, w.head_dim, DEV)
    compare_attention(pool.attention(1, allr, q), oracle_attention(slab, pool, 1, allr, q))
