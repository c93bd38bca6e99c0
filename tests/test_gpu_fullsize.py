"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: the same
DecodeLoop (engine.py) that the bench drives — fused append + attention per layer on stream A, arrivals
ingested on stream B — runs a few steps of configs 2-5, and sampled outputs are checked against the oracle:

  * attention: sampled rows (short and long contexts interleaved) of the LAST step, first / last / one
    seeded-random layer, against oracle.attention on a private slab rebuilt from the logical values
    (workloads.kv_values) — so the row is right only if the initial ingest, every arrival's ingest, every
    step's append and the attention all were;
  * ingest: sampled live requests (a long-resident one, a newly arrived one, the longest) are gathered from
    the pool and compared BIT for bit with their regenerated values, all layers;
  * properties that hold at any size: finite outputs everywhere (the pool is NaN-filled underneath), pool
    occupancy equal to the schedule's block count.
Configs 2 and 4 are checked in FULL on the sampled layers (every batch row; "configs 1, 2, 4 are
checked in full"), and config 2 additionally runs its 64 decode steps from the initial state with every row of
steps {0, 15, 16, 63} compared.  For those the oracle's inputs are the shared seeded
generator's values evaluated on the GPU and copied to the host (the generator is torch integer arithmetic, the
same bits on either device — test_generator_gives_the_same_bits_on_cpu_and_cuda; on the CPU it would take
minutes per layer); the oracle itself runs on the host cores.
Config 5's pool is 60 % of device memory (~115 GB on a B200); tests that do not fit the device are skipped
with the reason stated."""
import numpy as np
import pytest
import torch

import oracle
from paper_2511_20982_b200 import binding as B
from paper_2511_20982_b200 import workloads as W
from paper_2511_20982_b200.engine import DecodeLoop
from gpu_harness import DEV, NAN_BITS
from helpers import bits_of, bits_to_f64

pytestmark = pytest.mark.gpu

STEPS = 3


def test_generator_gives_the_same_bits_on_cpu_and_cuda():
    """workloads.kv_values / kv_values_at / q_values: integer hashing + a table lookup, bit-identical on both devices."""
    for seed, kind, uid, H, d, l0, lc, t0, t1 in [(2098203, W.KIND_K, 7, 8, 128, 3, 2, 100, 1200), (5, W.KIND_V, 1 << 24, 2, 64, 0, 1, 0, 17),
                                                   (2098204, W.KIND_V, 90, 8, 128, 0, 1, 30000, 32768)]:
        a = W.kv_values(seed, kind, uid, H, d, l0, lc, t0, t1, "cpu")
        b = W.kv_values(seed, kind, uid, H, d, l0, lc, t0, t1, DEV)
        assert torch.equal(a.view(torch.int16), b.cpu().view(torch.int16))
    a = W.kv_values_at(9, W.KIND_K, [3, 4, 1 << 24], [0, 99, 5000], 8, 128, 1, 3, "cpu")
    b = W.kv_values_at(9, W.KIND_K, [3, 4, 1 << 24], [0, 99, 5000], 8, 128, 1, 3, DEV)
    assert torch.equal(a.view(torch.int16), b.cpu().view(torch.int16))
    assert torch.equal(W.q_values(3, 5, 2, 16, 32, 128, "cpu").view(torch.int16), W.q_values(3, 5, 2, 16, 32, 128, DEV).cpu().view(torch.int16))


def oracle_rows(loop, step, layer, rows, fp8=False, gen_device="cpu"):
    """Oracle output of batch rows `rows` of `step` at `layer`, from regenerated logical values only."""
    w, sp = loop.w, loop.sched.steps[step]
    reqs = [(loop.sched.content_uid[int(sp.batch[r])], int(sp.lens_after[r])) for r in rows]
    nblk = [(n + 15) // 16 for _, n in reqs]
    dims = oracle.Dims(1, w.num_kv_heads, w.head_dim, 16, sum(nblk))
    slab = oracle.new_slab_fp8(dims, 0xFF) if fp8 else oracle.new_slab(dims, NAN_BITS)
    lists, off = [], 0
    for (cu, n), b in zip(reqs, nblk):
        lists.append(np.arange(off, off + b, dtype=np.int32)); off += b
        k = bits_of(W.kv_values(w.seed, W.KIND_K, cu, w.num_kv_heads, w.head_dim, layer, 1, 0, n, gen_device))
        v = bits_of(W.kv_values(w.seed, W.KIND_V, cu, w.num_kv_heads, w.head_dim, layer, 1, 0, n, gen_device))
        (oracle.scatter_fp8 if fp8 else oracle.scatter)(slab, dims, lists[-1], 0, k, v)
    q = bits_of(loop.q[step][layer][rows])
    fn = oracle.attention_fp8 if fp8 else oracle.attention
    return fn(slab, dims, 0, w.num_q_heads, lists, [n for _, n in reqs], q)


def sample_rows(lens, n_short, n_long, rng):
    order = np.argsort(lens, kind="stable")
    pick = list(order[:n_short]) + list(order[::-1][:n_long]) + list(rng.choice(len(lens), size=4, replace=False))
    return np.asarray(sorted(set(int(x) for x in pick)))


def check_rows(loop, name, step, layer, rows, fp8, gen_device):
    want = oracle_rows(loop, step, layer, rows, fp8, gen_device)
    got = bits_to_f64(bits_of(loop.out[step][layer][torch.as_tensor(rows, device=loop.out[step].device)]))
    err = np.abs(got - want)
    assert np.all(np.isfinite(got))
    assert err.max() <= 1e-2 and err.mean() <= 1e-3, (name, step, layer, float(err.max()), float(err.mean()))
    rms = np.sqrt((want ** 2).mean(axis=(1, 2)))
    rel = (np.maximum(err - np.abs(want) * 2.0 ** -8, 0).max(axis=(1, 2)) / rms).max()
    assert rel <= 3e-2, (name, step, layer, float(rel))
    return float(err.max())


def run_config(name, n_short, n_long, kv_dtype=B.KV_DTYPE_BF16, fused=True, all_rows=False, options=None, inline_ingest=False):
    w = W.CONFIGS[name]
    free, total = torch.cuda.mem_get_info()
    try:
        loop = DecodeLoop(w, STEPS, device=DEV, sentinel=int(np.uint16(NAN_BITS).astype(np.int16)), profile=False,
                          kv_dtype=kv_dtype, fused=fused, options=options, inline_ingest=inline_ingest)
    except (torch.cuda.OutOfMemoryError, AssertionError) as e:
        pytest.skip(f"{name} does not fit this device ({free / 1e9:.0f} GB free of {total / 1e9:.0f}): {e}")
    fp8 = kv_dtype == B.KV_DTYPE_FP8_E4M3
    try:
        for _ in range(STEPS):
            loop.step()
        loop.join()
        torch.cuda.synchronize()
        s = STEPS - 1
        sp = loop.sched.steps[s]
        rng = np.random.default_rng(w.seed)
        rows = np.arange(len(sp.batch)) if all_rows else sample_rows(sp.lens_after, n_short, n_long, rng)
        layers = sorted({0, w.num_layers - 1, int(rng.integers(0, w.num_layers))})
        worst = 0.0
        for layer in layers:
            for c0 in range(0, len(rows), 16):            # 16 rows at a time bounds the oracle's private slab
                worst = max(worst, check_rows(loop, name, s, layer, rows[c0:c0 + 16], fp8, DEV if all_rows else "cpu"))
        # every output of the last step is finite (the pool is NaN underneath: no unmasked stale read anywhere)
        assert bool(torch.isfinite(loop.out[s].float()).all())
        # occupancy equals the schedule's live blocks (+ the arrivals that join at the next step)
        live = {int(i): int(n) for i, n in zip(sp.batch, sp.lens_after)}
        blocks = sum((n + 15) // 16 for n in live.values())
        blocks += sum((int(loop.sched.bank_lens[e]) + 15) // 16 for e in sp.arrive_bank)
        st = loop.pool.stats()
        assert st["blocks_total"] - st["blocks_free"] == blocks and st["live_requests"] == len(live) + len(sp.arrive)
        # ingest bit-exactness on sampled requests (bf16 pools: gather is the inverse of ingest)
        if not fp8:
            cand = [int(sp.batch[0]), int(sp.batch[-1]), int(sp.batch[int(np.argmax(sp.lens_after))])]
            for uid in dict.fromkeys(cand):
                n = live[uid]
                if n * w.num_layers * w.num_kv_heads * w.head_dim * 2 * 2 > (6 << 30):
                    continue
                k, v = loop.pool.gather(uid)
                torch.cuda.synchronize()
                cu = loop.sched.content_uid[uid]
                for l in sorted({0, w.num_layers - 1}):
                    wk = W.kv_values(w.seed, W.KIND_K, cu, w.num_kv_heads, w.head_dim, l, 1, 0, n, "cpu")
                    wv = W.kv_values(w.seed, W.KIND_V, cu, w.num_kv_heads, w.head_dim, l, 1, 0, n, "cpu")
                    assert torch.equal(k[l].cpu().view(torch.int16), wk[0].view(torch.int16)), (name, uid, l, "K")
                    assert torch.equal(v[l].cpu().view(torch.int16), wv[0].view(torch.int16)), (name, uid, l, "V")
        return worst
    finally:
        loop.close()
        del loop
        torch.cuda.empty_cache()


def test_cfg2_7b_mha_full():
    run_config("cfg2_7b_mha", n_short=8, n_long=8, all_rows=True)


def test_cfg2_7b_mha_64_decode_steps_from_the_initial_state():
    """BASELINE.json configs[1]: 64 x (append one token per request, attend); every request crosses block
    boundaries on the way.  Every row of steps {0, 15, 16, 63} against the oracle."""
    w = W.CONFIGS["cfg2_7b_mha"]
    loop = DecodeLoop(w, w.decode_steps, device=DEV, sentinel=int(np.uint16(NAN_BITS).astype(np.int16)), profile=False)
    try:
        assert np.array_equal(loop.sched.steps[0].lens_after, loop.sched.n0 + 1)
        for _ in range(w.decode_steps):
            loop.step()
        loop.join()
        torch.cuda.synchronize()
        assert np.array_equal(loop.sched.steps[63].lens_after, loop.sched.n0 + 64)
        crossed = (loop.sched.n0 + 64 + 15) // 16 - (loop.sched.n0 + 15) // 16
        assert crossed.min() >= 4                            # every request opened at least 4 new blocks
        rows = np.arange(w.batch)
        for s in (0, 15, 16, 63):
            for c0 in range(0, len(rows), 16):
                check_rows(loop, w.name, s, 0, rows[c0:c0 + 16], False, DEV)
            assert bool(torch.isfinite(loop.out[s].float()).all())
        st = loop.pool.stats()
        assert st["blocks_total"] - st["blocks_free"] == int(((loop.sched.n0 + 64 + 15) // 16).sum())
    finally:
        loop.close()
        del loop
        torch.cuda.empty_cache()


def test_cfg3_8b_gqa_full():
    run_config("cfg3_8b_gqa", n_short=12, n_long=6)


def test_cfg4_70b_long_full():
    run_config("cfg4_70b_long", n_short=3, n_long=2, all_rows=True)


def test_cfg5_stress_full():
    run_config("cfg5_stress", n_short=24, n_long=3)


def test_cfg3_8b_gqa_full_fp8_pool():
    """FP8 pool, default kernel = attn_tc_kernel (tcgen05 / TMEM / TMA): 32 PDL-chained launches per step, fused append,
    the arrivals' ingest in line on the decode stream (what bench.py times on FP8 pools)."""
    run_config("cfg3_8b_gqa", n_short=12, n_long=6, kv_dtype=B.KV_DTYPE_FP8_E4M3, inline_ingest=True)


def test_cfg3_8b_gqa_full_fp8_pool_mma_sync():
    """The same through attn_kernel<Fp8Tiles<128>> (option tc=0)."""
    run_config("cfg3_8b_gqa", n_short=12, n_long=6, kv_dtype=B.KV_DTYPE_FP8_E4M3, options=dict(tc=0))


def test_cfg2_7b_mha_full_fp8_pool():
    """G = 1, 32 kv heads, every unit owns its request's last block (fused append in every unit); tcgen05 kernel."""
    run_config("cfg2_7b_mha", n_short=8, n_long=8, kv_dtype=B.KV_DTYPE_FP8_E4M3)


def test_cfg2_7b_mha_full_unfused():
    run_config("cfg2_7b_mha", n_short=8, n_long=8, fused=False)
