"""ORACLE — test infrastructure only.

A plain fp64 CPU statement (plain C, ``kv_oracle.c``) of what the D-instance KV path computes,
written from the paper before any kernel.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package; it imports
nothing from ``paper_2511_20982_b200`` and shares no code with the CUDA path.

This module is argument marshalling (numpy <-> C) only; every number comes from kv_oracle.c.
bf16 tensors cross this boundary as ``numpy.uint16`` bit patterns.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kv_oracle.c")
_LIB = os.path.join(_HERE, "libkv_oracle.so")


def build(force: bool = False) -> str:
    """Compile kv_oracle.c with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.run(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra", "-ffp-contract=off",
             "-o", tmp, _SRC, "-lm"],
            check=True,
        )
        os.replace(tmp, _LIB)
    return _LIB


class _Dims(ctypes.Structure):
    _fields_ = [
        ("num_layers", ctypes.c_int32),
        ("num_kv_heads", ctypes.c_int32),
        ("head_dim", ctypes.c_int32),
        ("block_size", ctypes.c_int32),
        ("num_blocks", ctypes.c_int64),
    ]


@dataclass(frozen=True)
class Dims:
    """Pool geometry as the oracle sees it (see include/kv_pool.h, "Slab layout")."""

    num_layers: int
    num_kv_heads: int
    head_dim: int
    block_size: int
    num_blocks: int

    @property
    def kv_elems(self) -> int:
        return self.num_layers * self.num_blocks * self.num_kv_heads * 2 * self.block_size * self.head_dim

    @property
    def fp8_tile_bytes(self) -> int:
        """FP8 pool: K8[16][d] | V8[16][d] | sc[16][2] fp32 per (layer, block, kv head)."""
        return 32 * self.head_dim + 128

    @property
    def fp8_bytes(self) -> int:
        return self.num_layers * self.num_blocks * self.num_kv_heads * self.fp8_tile_bytes

    def shape(self):
        return (self.num_layers, self.num_blocks, self.num_kv_heads, 2, self.block_size, self.head_dim)

    def _c(self) -> _Dims:
        return _Dims(self.num_layers, self.num_kv_heads, self.head_dim, self.block_size, self.num_blocks)


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P = ctypes.c_void_p
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_scatter.restype = None
        lib.oracle_scatter.argtypes = [P, ctypes.POINTER(_Dims), P, ctypes.c_int32, ctypes.c_int32, P, P,
                                       ctypes.c_int32, ctypes.c_int32]
        lib.oracle_gather.restype = None
        lib.oracle_gather.argtypes = [P, ctypes.POINTER(_Dims), P, ctypes.c_int32, P, P]
        lib.oracle_attention.restype = ctypes.c_int
        lib.oracle_attention.argtypes = [P, ctypes.POINTER(_Dims), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                         P, P, P, P, ctypes.c_double, P, P]
        lib.oracle_attention_varq.restype = ctypes.c_int
        lib.oracle_attention_varq.argtypes = [P, ctypes.POINTER(_Dims), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                              P, P, P, P, P, P, ctypes.c_double, P, P]
        D = ctypes.c_double
        lib.oracle_capacity.restype = None
        lib.oracle_capacity.argtypes = [D] * 10 + [P]
        lib.oracle_pd_ratio.restype = D
        lib.oracle_pd_ratio.argtypes = [D] * 4
        lib.oracle_e4m3_decode_table.restype = None
        lib.oracle_e4m3_decode_table.argtypes = [P]
        lib.oracle_e4m3_encode_many.restype = None
        lib.oracle_e4m3_encode_many.argtypes = [P, ctypes.c_int64, P]
        lib.oracle_scatter_fp8.restype = None
        lib.oracle_scatter_fp8.argtypes = [P, ctypes.POINTER(_Dims), P, ctypes.c_int32, ctypes.c_int32, P, P,
                                           ctypes.c_int32, ctypes.c_int32]
        lib.oracle_dequant_fp8.restype = None
        lib.oracle_dequant_fp8.argtypes = [P, ctypes.POINTER(_Dims), ctypes.c_int32, P, ctypes.c_int32, P, P]
        lib.oracle_attention_fp8.restype = ctypes.c_int
        lib.oracle_attention_fp8.argtypes = [P, ctypes.POINTER(_Dims), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                             P, P, P, P, ctypes.c_double, P, P]
        lib.oracle_attention_varq_fp8.restype = ctypes.c_int
        lib.oracle_attention_varq_fp8.argtypes = [P, ctypes.POINTER(_Dims), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                                  P, P, P, P, P, P, ctypes.c_double, P, P]
        lib.oracle_transfer.restype = None
        lib.oracle_transfer.argtypes = [P, ctypes.POINTER(_Dims), P, P, ctypes.POINTER(_Dims), P, ctypes.c_int32,
                                        ctypes.c_int32, ctypes.c_int32]
        lib.oracle_transfer_fp8.restype = None
        lib.oracle_transfer_fp8.argtypes = lib.oracle_transfer.argtypes
        lib.oracle_gather_fp8.restype = None
        lib.oracle_gather_fp8.argtypes = [P, ctypes.POINTER(_Dims), P, ctypes.c_int32, P, P, P, P]
        lib.oracle_chunk.restype = None
        lib.oracle_chunk.argtypes = [P, ctypes.POINTER(_Dims), ctypes.c_int32, ctypes.c_int32, P, ctypes.c_int32,
                                     ctypes.c_int32, P, ctypes.c_double, P, P, P]
        lib.oracle_combine.restype = None
        lib.oracle_combine.argtypes = [ctypes.c_int32, ctypes.c_int32, P, P, P, P]
        _lib = lib
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _u16(a, name) -> np.ndarray:
    a = np.asarray(a)
    if a.dtype != np.uint16:
        raise TypeError(f"{name}: expected uint16 bf16 bit patterns, got {a.dtype}")
    return np.ascontiguousarray(a)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def new_slab(dims: Dims, fill: int = 0) -> np.ndarray:
    """A host KV region, flat uint16, pre-filled with a 16-bit sentinel pattern."""
    return np.full(dims.kv_elems, fill, dtype=np.uint16)


def scatter(kv: np.ndarray, dims: Dims, blocks, start_pos: int, k_src, v_src, layer_begin: int = 0) -> None:
    """In place: kv <- request tokens.  k_src/v_src: uint16 [layer_count][Hkv][n][d]."""
    assert kv.dtype == np.uint16 and kv.flags.c_contiguous and kv.size == dims.kv_elems
    k_src, v_src = _u16(k_src, "k_src"), _u16(v_src, "v_src")
    layer_count, hkv, n, d = k_src.shape
    assert v_src.shape == k_src.shape and hkv == dims.num_kv_heads and d == dims.head_dim
    assert 0 <= layer_begin and layer_begin + layer_count <= dims.num_layers
    blocks = np.ascontiguousarray(blocks, dtype=np.int32)
    assert (start_pos + n + dims.block_size - 1) // dims.block_size <= blocks.size
    assert blocks.size == 0 or (0 <= blocks.min() and blocks.max() < dims.num_blocks)
    c = dims._c()
    _load().oracle_scatter(_ptr(kv), ctypes.byref(c), _ptr(blocks), start_pos, n, _ptr(k_src), _ptr(v_src),
                           layer_begin, layer_count)


def gather(kv: np.ndarray, dims: Dims, blocks, length: int):
    """Returns (k, v) uint16 [L][Hkv][length][d]."""
    assert kv.dtype == np.uint16 and kv.flags.c_contiguous and kv.size == dims.kv_elems
    blocks = np.ascontiguousarray(blocks, dtype=np.int32)
    assert (length + dims.block_size - 1) // dims.block_size <= blocks.size
    shape = (dims.num_layers, dims.num_kv_heads, length, dims.head_dim)
    k = np.empty(shape, dtype=np.uint16)
    v = np.empty(shape, dtype=np.uint16)
    c = dims._c()
    _load().oracle_gather(_ptr(kv), ctypes.byref(c), _ptr(blocks), length, _ptr(k), _ptr(v))
    return k, v


def attention(kv: np.ndarray, dims: Dims, layer: int, num_q_heads: int, block_lists, seq_lens, q,
              scale: float | None = None, return_wsum: bool = False):
    """Decode attention by the definition.  q: uint16 [B][Hq][d].  Returns float64 [B][Hq][d]."""
    assert kv.dtype == np.uint16 and kv.flags.c_contiguous and kv.size == dims.kv_elems
    q = _u16(q, "q")
    batch = q.shape[0]
    assert q.shape == (batch, num_q_heads, dims.head_dim)
    assert num_q_heads % dims.num_kv_heads == 0 and 0 <= layer < dims.num_layers
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    assert seq_lens.shape == (batch,) and len(block_lists) == batch
    lists = [np.ascontiguousarray(b, dtype=np.int32) for b in block_lists]
    for b, n in zip(lists, seq_lens):
        assert (int(n) + dims.block_size - 1) // dims.block_size <= b.size
        assert b.size == 0 or (0 <= b.min() and b.max() < dims.num_blocks)
    off = np.zeros(batch + 1, dtype=np.int64)
    off[1:] = np.cumsum([b.size for b in lists])
    bt = np.concatenate(lists) if lists else np.zeros(0, np.int32)
    bt = np.ascontiguousarray(bt, dtype=np.int32)
    if scale is None:
        scale = 1.0 / float(np.sqrt(np.float64(dims.head_dim)))
    out = np.empty((batch, num_q_heads, dims.head_dim), dtype=np.float64)
    wsum = np.empty((batch, num_q_heads), dtype=np.float64)
    c = dims._c()
    rc = _load().oracle_attention(_ptr(kv), ctypes.byref(c), layer, num_q_heads, batch, _ptr(bt), _ptr(off),
                                  _ptr(seq_lens), _ptr(q), float(scale), _ptr(out), _ptr(wsum))
    if rc != 0:
        raise ValueError(f"oracle_attention failed ({rc}): empty context or out of memory")
    return (out, wsum) if return_wsum else out


def attention_varq(kv: np.ndarray, dims: Dims, layer: int, num_q_heads: int, block_lists, seq_lens, q_lens, q,
                   scale: float | None = None, return_wsum: bool = False):
    """Variable-q-length causal attention (in-place prefill rows + decode rows in one batch).
    q: uint16 [sum(q_lens)][Hq][d], request r's query tokens are its LAST q_lens[r] tokens.
    Returns float64 [sum(q_lens)][Hq][d]."""
    assert kv.dtype == np.uint16 and kv.flags.c_contiguous and kv.size == dims.kv_elems
    q = _u16(q, "q")
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    q_lens = np.ascontiguousarray(q_lens, dtype=np.int32)
    batch = seq_lens.size
    total_q = int(q_lens.sum())
    assert q_lens.shape == (batch,) and len(block_lists) == batch
    assert q.shape == (total_q, num_q_heads, dims.head_dim)
    assert num_q_heads % dims.num_kv_heads == 0 and 0 <= layer < dims.num_layers
    lists = [np.ascontiguousarray(b, dtype=np.int32) for b in block_lists]
    for b, n in zip(lists, seq_lens):
        assert (int(n) + dims.block_size - 1) // dims.block_size <= b.size
        assert b.size == 0 or (0 <= b.min() and b.max() < dims.num_blocks)
    off = np.zeros(batch + 1, dtype=np.int64)
    off[1:] = np.cumsum([b.size for b in lists])
    q_off = np.zeros(batch + 1, dtype=np.int64)
    q_off[1:] = np.cumsum(q_lens)
    bt = np.ascontiguousarray(np.concatenate(lists) if lists else np.zeros(0, np.int32), dtype=np.int32)
    if scale is None:
        scale = 1.0 / float(np.sqrt(np.float64(dims.head_dim)))
    out = np.empty((total_q, num_q_heads, dims.head_dim), dtype=np.float64)
    wsum = np.empty((total_q, num_q_heads), dtype=np.float64)
    c = dims._c()
    rc = _load().oracle_attention_varq(_ptr(kv), ctypes.byref(c), layer, num_q_heads, batch, _ptr(bt), _ptr(off),
                                       _ptr(seq_lens), _ptr(q_lens), _ptr(q_off), _ptr(q), float(scale), _ptr(out),
                                       _ptr(wsum))
    if rc != 0:
        raise ValueError(f"oracle_attention_varq failed ({rc}): q_len outside [1, seq_len] or out of memory")
    return (out, wsum) if return_wsum else out


def chunk(kv: np.ndarray, dims: Dims, layer: int, kv_head: int, blocks, t0: int, t1: int, qv, scale: float):
    """(m, l, O) of tokens [t0, t1) for one query vector qv (uint16 [d])."""
    qv = _u16(qv, "qv")
    blocks = np.ascontiguousarray(blocks, dtype=np.int32)
    m = ctypes.c_double()
    l = ctypes.c_double()
    O = np.empty(dims.head_dim, dtype=np.float64)
    c = dims._c()
    _load().oracle_chunk(_ptr(kv), ctypes.byref(c), layer, kv_head, _ptr(blocks), t0, t1, _ptr(qv), float(scale),
                         ctypes.byref(m), ctypes.byref(l), _ptr(O))
    return m.value, l.value, O


def combine(m, l, O) -> np.ndarray:
    m = np.ascontiguousarray(m, dtype=np.float64)
    l = np.ascontiguousarray(l, dtype=np.float64)
    O = np.ascontiguousarray(O, dtype=np.float64)
    n, d = O.shape
    out = np.empty(d, dtype=np.float64)
    _load().oracle_combine(n, d, _ptr(m), _ptr(l), _ptr(O), _ptr(out))
    return out


def capacity(M_gpu, M_prime, M_model, TP, BW, alpha, t_d_slo, ISL, OSL, M_token):
    """(V_mem, V_BW, cc_d) by Eq. 11-13 as printed."""
    out = np.empty(3, dtype=np.float64)
    _load().oracle_capacity(float(M_gpu), float(M_prime), float(M_model), float(TP), float(BW), float(alpha),
                            float(t_d_slo), float(ISL), float(OSL), float(M_token), _ptr(out))
    return tuple(float(x) for x in out)


def pd_ratio(cc_d, t_p, t_d, OSL) -> float:
    """n_p / n_d by Eq. 14."""
    return float(_load().oracle_pd_ratio(float(cc_d), float(t_p), float(t_d), float(OSL)))


# ---- NEXT-2: FP8 (e4m3) KV pool -------------------------------------------------------------

def e4m3_decode_table() -> np.ndarray:
    out = np.empty(256, dtype=np.float64)
    _load().oracle_e4m3_decode_table(_ptr(out))
    return out


def e4m3_encode(y) -> np.ndarray:
    """float32 array -> e4m3 codes (uint8), round-to-nearest-even, saturating at +-448."""
    y = np.ascontiguousarray(y, dtype=np.float32)
    out = np.empty(y.shape, dtype=np.uint8)
    _load().oracle_e4m3_encode_many(_ptr(y), y.size, _ptr(out))
    return out


def new_slab_fp8(dims: Dims, fill: int = 0) -> np.ndarray:
    """A host FP8 KV region, flat uint8, pre-filled with a byte pattern."""
    return np.full(dims.fp8_bytes, fill, dtype=np.uint8)


def scatter_fp8(kv8: np.ndarray, dims: Dims, blocks, start_pos: int, k_src, v_src, layer_begin: int = 0) -> None:
    """In place: quantising scatter of bf16 rows (uint16 [layer_count][Hkv][n][d]) into the FP8 pool."""
    assert kv8.dtype == np.uint8 and kv8.flags.c_contiguous and kv8.size == dims.fp8_bytes and dims.block_size == 16
    k_src, v_src = _u16(k_src, "k_src"), _u16(v_src, "v_src")
    layer_count, hkv, n, d = k_src.shape
    assert v_src.shape == k_src.shape and hkv == dims.num_kv_heads and d == dims.head_dim
    assert 0 <= layer_begin and layer_begin + layer_count <= dims.num_layers
    blocks = np.ascontiguousarray(blocks, dtype=np.int32)
    assert (start_pos + n + dims.block_size - 1) // dims.block_size <= blocks.size
    assert blocks.size == 0 or (0 <= blocks.min() and blocks.max() < dims.num_blocks)
    c = dims._c()
    _load().oracle_scatter_fp8(_ptr(kv8), ctypes.byref(c), _ptr(blocks), start_pos, n, _ptr(k_src), _ptr(v_src),
                               layer_begin, layer_count)


def dequant_fp8(kv8: np.ndarray, dims: Dims, layer: int, blocks, length: int):
    """Dequantised (k, v) float64 [Hkv][length][d] of one request's layer."""
    assert kv8.dtype == np.uint8 and kv8.size == dims.fp8_bytes
    blocks = np.ascontiguousarray(blocks, dtype=np.int32)
    k = np.empty((dims.num_kv_heads, length, dims.head_dim), dtype=np.float64)
    v = np.empty_like(k)
    c = dims._c()
    _load().oracle_dequant_fp8(_ptr(kv8), ctypes.byref(c), layer, _ptr(blocks), length, _ptr(k), _ptr(v))
    return k, v


def attention_fp8(kv8: np.ndarray, dims: Dims, layer: int, num_q_heads: int, block_lists, seq_lens, q,
                  scale: float | None = None, return_wsum: bool = False):
    """Decode attention over an FP8 pool (definition on the dequantised values).  q: uint16 [B][Hq][d]."""
    assert kv8.dtype == np.uint8 and kv8.flags.c_contiguous and kv8.size == dims.fp8_bytes
    q = _u16(q, "q")
    batch = q.shape[0]
    assert q.shape == (batch, num_q_heads, dims.head_dim)
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    lists = [np.ascontiguousarray(b, dtype=np.int32) for b in block_lists]
    for b, n in zip(lists, seq_lens):
        assert (int(n) + dims.block_size - 1) // dims.block_size <= b.size
        assert b.size == 0 or (0 <= b.min() and b.max() < dims.num_blocks)
    off = np.zeros(batch + 1, dtype=np.int64)
    off[1:] = np.cumsum([b.size for b in lists])
    bt = np.ascontiguousarray(np.concatenate(lists) if lists else np.zeros(0, np.int32), dtype=np.int32)
    if scale is None:
        scale = 1.0 / float(np.sqrt(np.float64(dims.head_dim)))
    out = np.empty((batch, num_q_heads, dims.head_dim), dtype=np.float64)
    wsum = np.empty((batch, num_q_heads), dtype=np.float64)
    c = dims._c()
    rc = _load().oracle_attention_fp8(_ptr(kv8), ctypes.byref(c), layer, num_q_heads, batch, _ptr(bt), _ptr(off),
                                      _ptr(seq_lens), _ptr(q), float(scale), _ptr(out), _ptr(wsum))
    if rc != 0:
        raise ValueError(f"oracle_attention_fp8 failed ({rc})")
    return (out, wsum) if return_wsum else out


def attention_varq_fp8(kv8: np.ndarray, dims: Dims, layer: int, num_q_heads: int, block_lists, seq_lens, q_lens, q,
                       scale: float | None = None, return_wsum: bool = False):
    """attention_varq over an FP8 pool (causal definition on the dequantised values)."""
    assert kv8.dtype == np.uint8 and kv8.flags.c_contiguous and kv8.size == dims.fp8_bytes
    q = _u16(q, "q")
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    q_lens = np.ascontiguousarray(q_lens, dtype=np.int32)
    batch = seq_lens.size
    total_q = int(q_lens.sum())
    assert q.shape == (total_q, num_q_heads, dims.head_dim) and len(block_lists) == batch
    lists = [np.ascontiguousarray(b, dtype=np.int32) for b in block_lists]
    for b, n in zip(lists, seq_lens):
        assert (int(n) + dims.block_size - 1) // dims.block_size <= b.size
        assert b.size == 0 or (0 <= b.min() and b.max() < dims.num_blocks)
    off = np.zeros(batch + 1, dtype=np.int64)
    off[1:] = np.cumsum([b.size for b in lists])
    q_off = np.zeros(batch + 1, dtype=np.int64)
    q_off[1:] = np.cumsum(q_lens)
    bt = np.ascontiguousarray(np.concatenate(lists) if lists else np.zeros(0, np.int32), dtype=np.int32)
    if scale is None:
        scale = 1.0 / float(np.sqrt(np.float64(dims.head_dim)))
    out = np.empty((total_q, num_q_heads, dims.head_dim), dtype=np.float64)
    wsum = np.empty((total_q, num_q_heads), dtype=np.float64)
    c = dims._c()
    rc = _load().oracle_attention_varq_fp8(_ptr(kv8), ctypes.byref(c), layer, num_q_heads, batch, _ptr(bt), _ptr(off),
                                           _ptr(seq_lens), _ptr(q_lens), _ptr(q_off), _ptr(q), float(scale), _ptr(out),
                                           _ptr(wsum))
    if rc != 0:
        raise ValueError(f"oracle_attention_varq_fp8 failed ({rc})")
    return (out, wsum) if return_wsum else out


# ---- NEXT-4: producer -> consumer transfer, FP8 gather ---------------------------------------

def _same_geometry(a: Dims, b: Dims) -> bool:
    return (a.num_layers, a.num_kv_heads, a.head_dim, a.block_size) == (b.num_layers, b.num_kv_heads, b.head_dim, b.block_size)


def transfer(src_kv: np.ndarray, src_dims: Dims, src_blocks, dst_kv: np.ndarray, dst_dims: Dims, dst_blocks,
             length: int, layer_begin: int = 0, layer_count: int | None = None) -> None:
    """In place on dst_kv: tokens [0, length) of a request move from pool A (src) to pool B (dst), each side
    addressed through its own block list.  bf16 pools (uint16 slabs)."""
    assert src_kv.dtype == np.uint16 and src_kv.size == src_dims.kv_elems
    assert dst_kv.dtype == np.uint16 and dst_kv.flags.c_contiguous and dst_kv.size == dst_dims.kv_elems
    assert _same_geometry(src_dims, dst_dims)
    lc = src_dims.num_layers - layer_begin if layer_count is None else layer_count
    assert 0 <= layer_begin and lc >= 0 and layer_begin + lc <= src_dims.num_layers
    sb = np.ascontiguousarray(src_blocks, dtype=np.int32)
    db = np.ascontiguousarray(dst_blocks, dtype=np.int32)
    nb = (length + src_dims.block_size - 1) // src_dims.block_size
    assert nb <= sb.size and nb <= db.size
    assert nb == 0 or (0 <= sb[:nb].min() and sb[:nb].max() < src_dims.num_blocks)
    assert nb == 0 or (0 <= db[:nb].min() and db[:nb].max() < dst_dims.num_blocks)
    cs, cd = src_dims._c(), dst_dims._c()
    _load().oracle_transfer(_ptr(np.ascontiguousarray(src_kv)), ctypes.byref(cs), _ptr(sb), _ptr(dst_kv),
                            ctypes.byref(cd), _ptr(db), length, layer_begin, lc)


def transfer_fp8(src_kv8: np.ndarray, src_dims: Dims, src_blocks, dst_kv8: np.ndarray, dst_dims: Dims, dst_blocks,
                 length: int, layer_begin: int = 0, layer_count: int | None = None) -> None:
    """transfer() between two FP8 pools (uint8 slabs): codes and row scales move verbatim."""
    assert src_kv8.dtype == np.uint8 and src_kv8.size == src_dims.fp8_bytes and src_dims.block_size == 16
    assert dst_kv8.dtype == np.uint8 and dst_kv8.flags.c_contiguous and dst_kv8.size == dst_dims.fp8_bytes
    assert _same_geometry(src_dims, dst_dims)
    lc = src_dims.num_layers - layer_begin if layer_count is None else layer_count
    assert 0 <= layer_begin and lc >= 0 and layer_begin + lc <= src_dims.num_layers
    sb = np.ascontiguousarray(src_blocks, dtype=np.int32)
    db = np.ascontiguousarray(dst_blocks, dtype=np.int32)
    nb = (length + 15) // 16
    assert nb <= sb.size and nb <= db.size
    assert nb == 0 or (0 <= sb[:nb].min() and sb[:nb].max() < src_dims.num_blocks)
    assert nb == 0 or (0 <= db[:nb].min() and db[:nb].max() < dst_dims.num_blocks)
    cs, cd = src_dims._c(), dst_dims._c()
    _load().oracle_transfer_fp8(_ptr(np.ascontiguousarray(src_kv8)), ctypes.byref(cs), _ptr(sb), _ptr(dst_kv8),
                                ctypes.byref(cd), _ptr(db), length, layer_begin, lc)


def gather_fp8(kv8: np.ndarray, dims: Dims, blocks, length: int):
    """Stored codes and scales of tokens [0, length), all layers:
    (k_codes uint8 [L][Hkv][length][d], k_scales float32 [L][Hkv][length], v_codes, v_scales)."""
    assert kv8.dtype == np.uint8 and kv8.flags.c_contiguous and kv8.size == dims.fp8_bytes and dims.block_size == 16
    blocks = np.ascontiguousarray(blocks, dtype=np.int32)
    assert (length + 15) // 16 <= blocks.size
    shape = (dims.num_layers, dims.num_kv_heads, length, dims.head_dim)
    kc, vc = np.empty(shape, dtype=np.uint8), np.empty(shape, dtype=np.uint8)
    ks, vs = np.empty(shape[:3], dtype=np.float32), np.empty(shape[:3], dtype=np.float32)
    c = dims._c()
    _load().oracle_gather_fp8(_ptr(kv8), ctypes.byref(c), _ptr(blocks), length, _ptr(kc), _ptr(ks), _ptr(vc), _ptr(vs))
    return kc, ks, vc, vs
