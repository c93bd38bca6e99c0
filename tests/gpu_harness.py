"""Shared plumbing of the -m gpu parity tests: drive the CUDA path through the C-ABI binding
and build the oracle's view of the same seeded inputs on the CPU.

Values come from paper_2511_20982_b200.workloads (regenerated independently on each side);
the only thing the oracle side takes from the library is the host block_table (integer data
from kv_block_table — results do not depend on it)."""
import numpy as np
import torch

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import workloads as W
from helpers import bits_of, bits_to_f64

DEV = "cuda:0"
NAN_BITS = 0x7FC0  # bf16 quiet NaN: an unmasked read of a stale slot poisons the output


def sentinel_fill(pool, bits=NAN_BITS):
    pool.slab[: pool.kv_bytes].view(torch.int16).fill_(int(np.uint16(bits).astype(np.int16)))


def make_pool(w: W.Workload, num_blocks, max_requests=None, alloc_seed=1, sentinel=NAN_BITS, max_len=None):
    max_len = max_len or w.max_len
    cfg = kv.PoolConfig(num_layers=w.num_layers, num_q_heads=w.num_q_heads, num_kv_heads=w.num_kv_heads,
                        head_dim=w.head_dim, num_blocks=num_blocks, max_requests=max_requests or max(2 * w.batch, 8),
                        max_blocks_per_request=(max_len + 15) // 16, alloc_seed=alloc_seed)
    pool = kv.KVPool(cfg, device=DEV)
    if sentinel is not None:
        sentinel_fill(pool, sentinel)
    return pool


def apply_options(pool, opts):
    """set_option for every (key, value); a pool that cannot run the TMA / tcgen05 variants (head_dim 64) skips that mode."""
    import pytest
    for k_, v_ in (opts or {}).items():
        try:
            pool.set_option(k_, v_)
        except kv.KVError as e:
            if k_ in ("tma", "tc") and e.status == kv.binding.KV_ERR_UNSUPPORTED:
                pytest.skip(f"{k_}=1 needs head_dim 128")
            raise


def dims_of(pool) -> oracle.Dims:
    c = pool.cfg
    return oracle.Dims(c.num_layers, c.num_kv_heads, c.head_dim, c.block_size, c.num_blocks)


def kv_src(w: W.Workload, uid: int, t0: int, t1: int, device, layer_begin=0, layer_count=None):
    lc = w.num_layers - layer_begin if layer_count is None else layer_count
    k = W.kv_values(w.seed, W.KIND_K, uid, w.num_kv_heads, w.head_dim, layer_begin, lc, t0, t1, device)
    v = W.kv_values(w.seed, W.KIND_V, uid, w.num_kv_heads, w.head_dim, layer_begin, lc, t0, t1, device)
    return k, v


def pool_bits(pool) -> np.ndarray:
    """Device KV region -> flat uint16 numpy (whole-slab compare)."""
    return pool.slab[: pool.kv_bytes].view(torch.int16).cpu().numpy().view(np.uint16)


def oracle_slab(pool, sentinel=NAN_BITS) -> np.ndarray:
    return oracle.new_slab(dims_of(pool), sentinel)


def oracle_ingest(slab, pool, w, uid, t0, t1, blocks=None):
    """CPU side of an ingest of logical tokens [t0, t1) of request uid."""
    if blocks is None:
        blocks, _ = pool.block_table(uid)
    k, v = kv_src(w, uid, t0, t1, "cpu")
    oracle.scatter(slab, dims_of(pool), blocks, t0, bits_of(k), bits_of(v))


def compare_attention(got_bf16: torch.Tensor, want: np.ndarray, max_abs=1e-2, mean_abs=1e-3, rel_rms=3e-2):
    """BASELINE.json bar (max abs <= 1e-2, mean abs <= 1e-3) plus the per-request relative bar of
    SURVEY §8(c) A9: max err / rms(oracle out) <= 3e-2 (beyond each element's own bf16 rounding)."""
    got = bits_to_f64(bits_of(got_bf16))
    assert got.shape == want.shape
    assert np.all(np.isfinite(got)), "non-finite output (unmasked read of a sentinel slot?)"
    err = np.abs(got - want)
    stats = dict(max_abs=float(err.max()), mean_abs=float(err.mean()))
    assert stats["max_abs"] <= max_abs, stats
    assert stats["mean_abs"] <= mean_abs, stats
    # per request row: the error left after allowing each element its own final bf16 rounding (half an ulp
    # <= 2^-8 |want|, DESIGN.md §6 (iv) — an outlier element of a head whose weights concentrate on one
    # token is many times the row rms) must stay below rel_rms x rms(oracle row)
    for r in range(want.shape[0]):
        rms = float(np.sqrt(np.mean(want[r] ** 2)))
        if rms > 0:
            rel = float(np.maximum(err[r] - np.abs(want[r]) * 2.0 ** -8, 0.0).max()) / rms
            assert rel <= rel_rms, (r, rel, stats)
            stats["max_rel_rms"] = max(stats.get("max_rel_rms", 0.0), rel)
    return stats


def oracle_attention(slab, pool, layer, ids, q_bf16: torch.Tensor, scale=None):
    lists, lens = [], []
    for i in ids:
        b, n = pool.block_table(i)
        lists.append(b)
        lens.append(n)
    return oracle.attention(slab, dims_of(pool), layer, pool.cfg.num_q_heads, lists, lens, bits_of(q_bf16), scale=scale)
