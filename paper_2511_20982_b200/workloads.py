"""Seeded synthetic inputs shaped like the paper's workloads — and nothing else.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests; it holds none of
the method's arithmetic (no attention, no scatter, no block allocation): only request-length
laws, bf16 value generation and the table of BASELINE.json configurations.  It imports
neither the CUDA binding nor ``oracle``.

Stand-in statement.  The paper measures on Azure conversation/code traces, BurstGPT and
ShareGPT with LLaMa-3.3-70B-FP8 / OPT-30B / Qwen weights.  None of that is
available here and none of it is reproduced: request lengths are drawn from the laws
BASELINE.json's ``configs`` state (uniform / lognormal / bimodal; cf. the paper's
heavy-tailed ISL, its 100-vs-1900-token mixture, and Table I's
sequence lengths 100-1700 at concurrency 104-248), and q/K/V values are
i.i.d. N(0,1) rounded to bf16.

Value generator (SURVEY §8(d) "D-gen").  A value is a pure function of its LOGICAL position
    (seed, kind in {K,V,q}, request uid, layer, head, token, j)
so that (i) the GPU can fill tens of GB without crossing PCIe while the CPU regenerates any
slice bit-identically, (ii) content does not depend on physical placement, and (iii)
appending tokens [a,b) yields the same bits as ingesting them in one go.
    bits  = splitmix64-style mix of the position (integer only, wrap-around int64)
    value = NORMAL_TABLE[bits >> 48]      65 536 bf16 standard-normal quantiles
The same torch integer ops run on CPU and CUDA, so both sides get identical bf16 bits.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np
import torch

KIND_K, KIND_V, KIND_Q = 0, 1, 2

_GAMMA = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB
_MASK64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int -> the signed 64-bit value with the same bit pattern."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right of an int64 tensor (torch's >> is arithmetic)."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def mix64_t(x: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on an int64 tensor (wrap-around arithmetic)."""
    x = (x ^ _lsr(x, 30)) * _s64(_M1)
    x = (x ^ _lsr(x, 27)) * _s64(_M2)
    return x ^ _lsr(x, 31)


def mix64_i(x: int) -> int:
    """The same finaliser on a Python int (unsigned 64-bit)."""
    x &= _MASK64
    x = ((x ^ (x >> 30)) * _M1) & _MASK64
    x = ((x ^ (x >> 27)) * _M2) & _MASK64
    return x ^ (x >> 31)


_TABLES: dict[str, torch.Tensor] = {}


def normal_table(device="cpu") -> torch.Tensor:
    """65 536 bf16 quantiles of N(0,1): table[i] = bf16(Phi^-1((i + 0.5) / 65536)).

    Always computed on the CPU in fp64 (so every process gets the same bits), then moved."""
    key = str(device)
    if key not in _TABLES:
        if "cpu" not in _TABLES:
            p = (torch.arange(65536, dtype=torch.float64) + 0.5) / 65536.0
            _TABLES["cpu"] = torch.special.ndtri(p).to(torch.float32).to(torch.bfloat16)
        _TABLES[key] = _TABLES["cpu"].to(device)
    return _TABLES[key]


def stream_key(seed: int, kind: int, uid: int) -> int:
    return mix64_i(mix64_i(seed * _GAMMA + kind) + uid)


def _values(key: int, ctr: torch.Tensor) -> torch.Tensor:
    bits = mix64_t(ctr * _s64(_GAMMA) + _s64(key))
    return normal_table(ctr.device)[_lsr(bits, 48)]


def kv_values(seed: int, kind: int, uid: int, num_kv_heads: int, head_dim: int, layer_begin: int,
              layer_count: int, t0: int, t1: int, device="cpu") -> torch.Tensor:
    """bf16 [layer_count][num_kv_heads][t1-t0][head_dim]: K (kind 0) or V (kind 1) of request `uid`,
    logical tokens [t0, t1), layers [layer_begin, layer_begin+layer_count)."""
    assert head_dim <= 256 and t1 <= (1 << 20)
    key = stream_key(seed, kind, uid)
    out = torch.empty((layer_count, num_kv_heads, t1 - t0, head_dim), dtype=torch.bfloat16, device=device)
    t = torch.arange(t0, t1, dtype=torch.int64, device=device).view(1, -1, 1)
    j = torch.arange(head_dim, dtype=torch.int64, device=device).view(1, 1, -1)
    h = torch.arange(num_kv_heads, dtype=torch.int64, device=device).view(-1, 1, 1)
    for ll in range(layer_count):  # one layer at a time bounds the int64 temporaries
        row = (layer_begin + ll) * num_kv_heads + h
        ctr = ((row << 20) | t) << 8 | j
        out[ll] = _values(key, ctr)
    return out


def stream_keys(seed: int, kind: int, uids) -> np.ndarray:
    """Vectorised stream_key: int64 bit patterns of stream_key(seed, kind, uid) for each uid."""
    def mix(x):
        x = (x ^ (x >> np.uint64(30))) * np.uint64(_M1)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(_M2)
        return x ^ (x >> np.uint64(31))
    with np.errstate(over="ignore"):
        base = np.uint64(mix64_i(seed * _GAMMA + kind))
        return mix(base + np.asarray(uids, dtype=np.int64).astype(np.uint64)).astype(np.int64)


def kv_values_at(seed: int, kind: int, uids, positions, num_kv_heads: int, head_dim: int, layer_begin: int,
                 layer_count: int, device="cpu") -> torch.Tensor:
    """bf16 [layer_count][B][num_kv_heads][head_dim]: for request i, the K/V row of logical token
    positions[i] — element [ll][i][h][j] == kv_values(seed, kind, uids[i], ..., t, t+1)[ll][h][0][j]
    with t = positions[i].  One call serves a whole decode batch's appended tokens."""
    keys = torch.from_numpy(stream_keys(seed, kind, uids)).to(device).view(1, -1, 1, 1)
    t = torch.as_tensor(np.asarray(positions, dtype=np.int64), device=device).view(1, -1, 1, 1)
    assert int(t.max()) < (1 << 20) and head_dim <= 256
    ll = torch.arange(layer_begin, layer_begin + layer_count, dtype=torch.int64, device=device).view(-1, 1, 1, 1)
    h = torch.arange(num_kv_heads, dtype=torch.int64, device=device).view(1, 1, -1, 1)
    j = torch.arange(head_dim, dtype=torch.int64, device=device).view(1, 1, 1, -1)
    ctr = (((ll * num_kv_heads + h) << 20) | t) << 8 | j
    bits = mix64_t(ctr * _s64(_GAMMA) + keys)
    return normal_table(device)[_lsr(bits, 48)]


def q_values(seed: int, step: int, layer: int, batch: int, num_q_heads: int, head_dim: int,
             device="cpu") -> torch.Tensor:
    """bf16 [batch][num_q_heads][head_dim] query of decode step `step`, layer `layer`."""
    key = stream_key(seed, KIND_Q, (step << 16) | layer)
    ctr = torch.arange(batch * num_q_heads * head_dim, dtype=torch.int64, device=device)
    return _values(key, ctr).view(batch, num_q_heads, head_dim)


# ---------------------------------------------------------------------------------------------
# request-length laws (BASELINE.json `configs`)
# ---------------------------------------------------------------------------------------------

def lengths_fixed(values):
    vals = [int(v) for v in values]
    return lambda rng, n: np.array([vals[i % len(vals)] for i in range(n)], dtype=np.int64)


def lengths_uniform(lo, hi):
    return lambda rng, n: rng.integers(lo, hi + 1, size=n, dtype=np.int64)


def lengths_lognormal(median, sigma, lo, hi):
    def f(rng, n):
        z = rng.standard_normal(n)
        return np.clip(np.rint(np.exp(np.log(median) + sigma * z)), lo, hi).astype(np.int64)
    return f


def lengths_bimodal(p_long, short, long):
    def f(rng, n):
        is_long = rng.random(n) < p_long
        s = rng.integers(short[0], short[1] + 1, size=n, dtype=np.int64)
        l = rng.integers(long[0], long[1] + 1, size=n, dtype=np.int64)
        return np.where(is_long, l, s)
    return f


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json configuration (or a scaled-down copy of one for the parity tests)."""

    name: str
    num_layers: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    batch: int
    length_law: object = field(repr=False)
    seed: int
    block_size: int = 16
    ingest_per_step: int = 0      # prefill-completed requests handed over per decode step
    decode_steps: int = 1         # timed decode steps in the bench
    pool_slack: float = 1.25      # pool blocks = slack x expected resident blocks
    pool_hbm_frac: float = 0.0    # >0: size the pool to this fraction of device memory (config 5)
    fragmented: bool = False      # config 4: interleaved slice-wise ingest on a permuted pool
    max_len: int = 0              # upper bound of the length law (for max_blocks_per_request)

    def rng(self, salt: int = 0) -> np.random.Generator:
        return np.random.Generator(np.random.PCG64([self.seed, salt]))

    def draw_lengths(self, n: int | None = None, salt: int = 0) -> np.ndarray:
        return self.length_law(self.rng(salt), self.batch if n is None else n)

    @property
    def group(self) -> int:
        return self.num_q_heads // self.num_kv_heads

    def kv_bytes_per_token(self, layers: int | None = None) -> int:
        return 2 * (self.num_layers if layers is None else layers) * self.num_kv_heads * self.head_dim * 2

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


# ---------------------------------------------------------------------------------------------
# byte accounting (SURVEY §8(d) "algorithmic bytes") — counting only, shared by bench.py's CUDA arm, its
# oracle-timing arm and the engine; lives here so that the oracle arm never imports the CUDA binding
# ---------------------------------------------------------------------------------------------

def kv_token_bytes_layer(w: Workload, fp8: bool = False) -> int:
    """Pool bytes of one token in one layer: K and V rows of every kv head — bf16, or e4m3 codes plus the
    two fp32 row scales (FP8 pool, NEXT-2)."""
    return w.num_kv_heads * ((2 * w.head_dim + 8) if fp8 else (2 * w.head_dim * 2))


def attention_bytes(w: Workload, lens, fp8: bool = False) -> int:
    """Algorithmic bytes of one layer's decode attention: every resident K and V element once, q in and
    out once, the block_table once per request, seq_lens."""
    lens = np.asarray(lens, dtype=np.int64)
    kv = int(lens.sum()) * kv_token_bytes_layer(w, fp8)
    qo = 2 * len(lens) * w.num_q_heads * w.head_dim * 2
    bt = 4 * int(((lens + w.block_size - 1) // w.block_size).sum()) + 4 * len(lens)
    return kv + qo + bt


CONFIGS: dict[str, Workload] = {
    # configs[0] tiny correctness case
    "cfg1_tiny": Workload("cfg1_tiny", 1, 8, 2, 64, 4, lengths_fixed([17, 64, 130, 255]), 2098201,
                          max_len=255 + 64),
    # configs[1] 7B-MHA-shaped single-layer decode, 64 steps appending one token per request
    "cfg2_7b_mha": Workload("cfg2_7b_mha", 1, 32, 32, 128, 64, lengths_uniform(512, 2048), 2098202,
                            decode_steps=64, max_len=2048 + 64 + 16),
    # configs[2] 8B-GQA-shaped decode under concurrency, 16 newly prefilled requests per step
    "cfg3_8b_gqa": Workload("cfg3_8b_gqa", 32, 32, 8, 128, 256, lengths_lognormal(1024, 0.8, 128, 8192),
                            2098203, ingest_per_step=16, decode_steps=32, max_len=8192 + 256),
    # configs[3] 70B-shaped long-context decode, fragmented block_table
    "cfg4_70b_long": Workload("cfg4_70b_long", 1, 64, 8, 128, 128, lengths_uniform(4096, 32768), 2098204,
                              decode_steps=16, fragmented=True, max_len=32768 + 64),
    # configs[4] mixed-length high-concurrency stress, pool ~60 % of HBM, bursts of 64
    "cfg5_stress": Workload("cfg5_stress", 8, 32, 8, 128, 512,
                            lengths_bimodal(0.2, (64, 256), (8192, 16384)), 2098205,
                            ingest_per_step=64, decode_steps=16, pool_hbm_frac=0.60, max_len=16384 + 256),
}
