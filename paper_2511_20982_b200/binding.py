"""Thin ctypes binding of include/kv_pool.h — argument marshalling only.

Every function has the name and meaning of its C counterpart; device tensors are passed as
their ``data_ptr()``.  ``KVPool`` bundles a pool handle with the torch slab it lives in.  There
is no fallback of any kind: a missing ``csrc/libkvpool.so`` raises ImportError at import.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(_HERE, "csrc", "libkvpool.so")

if not os.path.exists(lib_path):
    raise ImportError(
        f"{lib_path} is missing: build it with `python -m paper_2511_20982_b200.build` "
        "(nvcc, sm_100a).  There is no CPU or PyTorch fallback for this path.")

from . import build as _build

if _build.stale():
    raise ImportError(
        f"{lib_path} was not built from the sources in this tree (source hash mismatch): rebuild it with "
        "`python -m paper_2511_20982_b200.build --force`.  A stale library is refused rather than loaded.")

lib = ctypes.CDLL(lib_path)

KV_OK = 0
KV_ERR_INVALID, KV_ERR_NO_BLOCKS, KV_ERR_UNKNOWN_REQUEST, KV_ERR_TOO_LONG = -1, -2, -3, -4
KV_ERR_TOO_MANY_REQUESTS, KV_ERR_CUDA, KV_ERR_NO_DEVICE, KV_ERR_UNSUPPORTED = -5, -6, -7, -8
KV_ERR_SCRATCH_LIMIT = -9
KV_STATIC_MAX_PARTIALS = 4096
KV_DTYPE_BF16, KV_DTYPE_FP8_E4M3 = 0, 1


class _Config(ctypes.Structure):
    _fields_ = [
        ("num_layers", ctypes.c_int32), ("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32),
        ("head_dim", ctypes.c_int32), ("block_size", ctypes.c_int32), ("num_blocks", ctypes.c_int64),
        ("max_requests", ctypes.c_int32), ("max_blocks_per_request", ctypes.c_int32),
        ("alloc_seed", ctypes.c_uint64), ("device_base", ctypes.c_void_p), ("device_bytes", ctypes.c_int64),
        ("kv_dtype", ctypes.c_int32),
    ]


_P = ctypes.c_void_p
_i32, _i64 = ctypes.c_int32, ctypes.c_int64
_CFG = ctypes.POINTER(_Config)
_SIGS = {
    "kv_pool_kv_bytes": (_i64, [_CFG]),
    "kv_pool_required_bytes": (_i64, [_CFG]),
    "kv_pool_create": (_i32, [_CFG, ctypes.POINTER(_P)]),
    "kv_pool_destroy": (_i32, [_P]),
    "kv_reserve": (_i32, [_P, _i32, _P, _P]),
    "kv_ingest": (_i32, [_P, _i32, _P, _P, _P, _P, _i32, _i32, _P]),
    "paged_decode_attention": (_i32, [_P, _i32, _i32, _P, _P, _P, ctypes.c_float, _P]),
    "paged_decode_attention_static": (_i32, [_P, _i32, _i32, _P, _P, _P, ctypes.c_float, _P]),
    "kv_static_scratch_bytes": (_i64, []),
    "paged_decode_step": (_i32, [_P, _i32, _i32, _P, _P, _P, _P, _P, ctypes.c_float, _P]),
    "paged_decode_step_host": (_i32, [_P, _i32, _i32, _P, _P, _P, _P, _P, ctypes.c_float, _P, _i64, _P]),
    "paged_decode_step_layers": (_i32, [_P, _i32, _i32, _i32, _P, _P, _P, _P, _P, _i64, _i64, ctypes.c_float, _i32, _P]),
    "paged_varlen_attention": (_i32, [_P, _i32, _i32, _P, _P, _P, _P, ctypes.c_float, _P]),
    "paged_varlen_step": (_i32, [_P, _i32, _i32, _P, _P, _P, _P, _P, _P, ctypes.c_float, _i32, _P]),
    "kv_free": (_i32, [_P, _i32, _P]),
    "kv_block_table": (_i32, [_P, _i64, _P, _i32, ctypes.POINTER(_i32), ctypes.POINTER(_i32)]),
    "kv_pool_stats": (_i32, [_P, ctypes.POINTER(_i64), ctypes.POINTER(_i64), ctypes.POINTER(_i32),
                             ctypes.POINTER(_i64)]),
    "kv_gather": (_i32, [_P, _i64, _P, _P, _P]),
    "kv_gather_bytes": (_i64, [_CFG, _i32]),
    "kv_transfer": (_i32, [_P, _P, _i32, _P, _P, _i32, _i32, _P]),
    "kv_plan_decode": (_i32, [_P, _i32, _P, _P, _i32, ctypes.POINTER(_i32), ctypes.POINTER(_i32)]),
    "kv_ingest_host": (_i32, [_P, _i32, _P, _P, _P, _P, _i32, _i32, _P, _i64, _P]),
    "paged_decode_attention_host": (_i32, [_P, _i32, _i32, _P, _P, _P, ctypes.c_float, _P, _i64, _P]),
    "kv_capacity": (_i32, [_P, _P]),
    "kv_optimal_pd_ratio": (_i32, [ctypes.c_double] * 4 + [ctypes.POINTER(ctypes.c_double)]),
    "kv_token_bytes": (_i64, [_CFG]),
    "kv_launch_count": (_i64, [_P]),
    "kv_pool_counter": (_i64, [_P, ctypes.c_char_p]),
    "kv_profile_read": (_i32, [_P, _i32, ctypes.POINTER(_i64), ctypes.POINTER(ctypes.c_double)]),
    "kv_profile_reset": (_i32, [_P]),
    "kv_pool_set_option": (_i32, [_P, ctypes.c_char_p, _i64]),
    "kv_last_cuda_error": (_i32, [_P]),
    "kv_strerror": (ctypes.c_char_p, [_i32]),
    "kv_version": (ctypes.c_char_p, []),
}
EXPORTS = tuple(_SIGS)
for _name, (_res, _args) in _SIGS.items():
    _f = getattr(lib, _name)  # AttributeError here = the .so does not export what the header declares
    _f.restype, _f.argtypes = _res, _args


class KVError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {kv_strerror(status)} ({status})")


def _check(status: int, where: str) -> None:
    if status != KV_OK:
        raise KVError(status, where)


@dataclass
class PoolConfig:
    num_layers: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    num_blocks: int
    max_requests: int
    max_blocks_per_request: int
    block_size: int = 16
    alloc_seed: int = 0
    kv_dtype: int = KV_DTYPE_BF16

    def _c(self, device_base: int = 0, device_bytes: int = 0) -> _Config:
        return _Config(self.num_layers, self.num_q_heads, self.num_kv_heads, self.head_dim, self.block_size,
                       self.num_blocks, self.max_requests, self.max_blocks_per_request, self.alloc_seed,
                       device_base or None, device_bytes, self.kv_dtype)


def _ids(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int64)


def _i32s(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptrs(a) -> np.ndarray:
    """list of tensors / ints, or an integer array of addresses -> uint64 array of addresses."""
    if isinstance(a, np.ndarray):
        return np.ascontiguousarray(a, dtype=np.uint64)
    return np.ascontiguousarray([x if isinstance(x, int) else x.data_ptr() for x in a], dtype=np.uint64)


def _np(a: np.ndarray):
    return a.ctypes.data_as(_P)


def kv_strerror(status: int) -> str:
    return lib.kv_strerror(status).decode()


def kv_version() -> str:
    return lib.kv_version().decode()


def kv_pool_kv_bytes(cfg: PoolConfig) -> int:
    c = cfg._c()
    n = lib.kv_pool_kv_bytes(ctypes.byref(c))
    if n < 0:
        raise KVError(int(n), "kv_pool_kv_bytes")
    return int(n)


def kv_pool_required_bytes(cfg: PoolConfig) -> int:
    c = cfg._c()
    n = lib.kv_pool_required_bytes(ctypes.byref(c))
    if n < 0:
        raise KVError(int(n), "kv_pool_required_bytes")
    return int(n)


def kv_pool_create(cfg: PoolConfig, device_base: int = 0, device_bytes: int = 0) -> int:
    c = cfg._c(device_base, device_bytes)
    h = _P()
    _check(lib.kv_pool_create(ctypes.byref(c), ctypes.byref(h)), "kv_pool_create")
    return h.value


def kv_pool_destroy(handle: int) -> None:
    _check(lib.kv_pool_destroy(handle), "kv_pool_destroy")


def kv_reserve(handle: int, req_ids, n_tokens) -> None:
    ids, n = _ids(req_ids), _i32s(n_tokens)
    assert ids.shape == n.shape
    _check(lib.kv_reserve(handle, ids.size, _np(ids), _np(n)), "kv_reserve")


def kv_ingest(handle: int, req_ids, n_tokens, k_src, v_src, layer_begin: int = 0, layer_count: int = 1,
              stream: int = 0) -> None:
    ids, n, kp, vp = _ids(req_ids), _i32s(n_tokens), _ptrs(k_src), _ptrs(v_src)
    assert ids.shape == n.shape == kp.shape == vp.shape
    _check(lib.kv_ingest(handle, ids.size, _np(ids), _np(n), _np(kp), _np(vp), layer_begin, layer_count,
                         stream or None), "kv_ingest")


def paged_decode_attention(handle: int, layer: int, req_ids, q_ptr: int, out_ptr: int, sm_scale: float = 0.0,
                           stream: int = 0) -> None:
    ids = _ids(req_ids)
    _check(lib.paged_decode_attention(handle, layer, ids.size, _np(ids), q_ptr, out_ptr, sm_scale, stream or None),
           "paged_decode_attention")


def paged_decode_attention_static(handle: int, layer: int, req_ids, q_ptr: int, out_ptr: int, sm_scale: float = 0.0,
                                  stream: int = 0) -> None:
    """paged_decode_attention with its split-KV workspace in the library's static device array (allocates nothing)."""
    ids = _ids(req_ids)
    _check(lib.paged_decode_attention_static(handle, layer, ids.size, _np(ids), q_ptr, out_ptr, sm_scale,
                                             stream or None), "paged_decode_attention_static")


def kv_static_scratch_bytes() -> int:
    return int(lib.kv_static_scratch_bytes())


def paged_decode_step(handle: int, layer: int, req_ids, q_ptr: int, k_new_ptr: int, v_new_ptr: int, out_ptr: int,
                      sm_scale: float = 0.0, stream: int = 0) -> None:
    """Fused a3 + a4 + a5 (after kv_reserve(req_ids, ones) for this step)."""
    ids = _ids(req_ids)
    _check(lib.paged_decode_step(handle, layer, ids.size, _np(ids), q_ptr, k_new_ptr, v_new_ptr, out_ptr, sm_scale,
                                 stream or None), "paged_decode_step")


KV_STEP_RESERVE = 1


def paged_decode_step_layers(handle: int, layer_begin: int, layer_count: int, req_ids, q_ptr: int, k_new_ptr: int,
                             v_new_ptr: int, out_ptr: int, q_layer_stride_bytes: int, kv_layer_stride_bytes: int,
                             sm_scale: float = 0.0, flags: int = 0, stream: int = 0) -> None:
    """One decode step's (append +) attention for layer_count layers in one call; k_new_ptr = 0: no append."""
    ids = _ids(req_ids)
    _check(lib.paged_decode_step_layers(handle, layer_begin, layer_count, ids.size, _np(ids), q_ptr, k_new_ptr or None,
                                        v_new_ptr or None, out_ptr, q_layer_stride_bytes, kv_layer_stride_bytes,
                                        sm_scale, flags, stream or None), "paged_decode_step_layers")


def paged_decode_step_host(handle: int, layer: int, req_ids, q_host_ptr: int, k_new_host_ptr: int,
                           v_new_host_ptr: int, out_host_ptr: int, sm_scale: float, staging_ptr: int,
                           staging_bytes: int, stream: int = 0) -> None:
    ids = _ids(req_ids)
    _check(lib.paged_decode_step_host(handle, layer, ids.size, _np(ids), q_host_ptr, k_new_host_ptr, v_new_host_ptr,
                                      out_host_ptr, sm_scale, staging_ptr, staging_bytes, stream or None),
           "paged_decode_step_host")


def kv_ingest_host(handle: int, req_ids, n_tokens, k_src, v_src, layer_begin: int, layer_count: int,
                   staging_ptr: int, staging_bytes: int, stream: int = 0) -> None:
    """k_src / v_src: HOST addresses (pinned tensors or ints)."""
    ids, n, kp, vp = _ids(req_ids), _i32s(n_tokens), _ptrs(k_src), _ptrs(v_src)
    assert ids.shape == n.shape == kp.shape == vp.shape
    _check(lib.kv_ingest_host(handle, ids.size, _np(ids), _np(n), _np(kp), _np(vp), layer_begin, layer_count,
                              staging_ptr, staging_bytes, stream or None), "kv_ingest_host")


def paged_decode_attention_host(handle: int, layer: int, req_ids, q_host_ptr: int, out_host_ptr: int,
                                sm_scale: float, staging_ptr: int, staging_bytes: int, stream: int = 0) -> None:
    ids = _ids(req_ids)
    _check(lib.paged_decode_attention_host(handle, layer, ids.size, _np(ids), q_host_ptr, out_host_ptr, sm_scale,
                                           staging_ptr, staging_bytes, stream or None),
           "paged_decode_attention_host")


def paged_varlen_attention(handle: int, layer: int, req_ids, q_lens, q_ptr: int, out_ptr: int, sm_scale: float = 0.0,
                           stream: int = 0) -> None:
    """Variable-q-length causal attention: request i's last q_lens[i] tokens are its query tokens."""
    ids, ql = _ids(req_ids), _i32s(q_lens)
    assert ids.shape == ql.shape
    _check(lib.paged_varlen_attention(handle, layer, ids.size, _np(ids), _np(ql), q_ptr, out_ptr, sm_scale,
                                      stream or None), "paged_varlen_attention")


KERNEL_KINDS = {"attn": 0, "combine": 1, "ingest": 2, "gather": 3, "varq": 4, "transfer": 5}


def paged_varlen_step(handle: int, layer: int, req_ids, q_lens, q_ptr: int, k_new_ptrs, v_new_ptrs, out_ptr: int,
                      sm_scale: float = 0.0, flags: int = 0, stream: int = 0) -> None:
    """(a1,) a2 of this layer's new rows, then the variable-q attention; k_new_ptrs / v_new_ptrs: one device pointer
    per request ([Hkv][q_len][d] bf16)."""
    ids, ql, kp, vp = _ids(req_ids), _i32s(q_lens), _ptrs(k_new_ptrs), _ptrs(v_new_ptrs)
    assert ids.size == ql.size == kp.size == vp.size
    _check(lib.paged_varlen_step(handle, layer, ids.size, _np(ids), _np(ql), q_ptr, _np(kp), _np(vp), out_ptr, sm_scale,
                                 flags, stream or None), "paged_varlen_step")


def kv_profile_read(handle: int, kind: int):
    """(launches, total milliseconds) of kernel `kind` since the last reset (needs option profile=1)."""
    n, ms = _i64(), ctypes.c_double()
    _check(lib.kv_profile_read(handle, kind, ctypes.byref(n), ctypes.byref(ms)), "kv_profile_read")
    return int(n.value), float(ms.value)


def kv_profile_reset(handle: int) -> None:
    _check(lib.kv_profile_reset(handle), "kv_profile_reset")


def kv_free(handle: int, req_ids) -> None:
    ids = _ids(req_ids)
    _check(lib.kv_free(handle, ids.size, _np(ids)), "kv_free")


def kv_block_table(handle: int, req_id: int):
    nb, ln = _i32(), _i32()
    _check(lib.kv_block_table(handle, req_id, None, 0, ctypes.byref(nb), ctypes.byref(ln)), "kv_block_table")
    out = np.empty(nb.value, dtype=np.int32)
    _check(lib.kv_block_table(handle, req_id, _np(out), out.size, ctypes.byref(nb), ctypes.byref(ln)),
           "kv_block_table")
    return out, ln.value


def kv_pool_stats(handle: int) -> dict:
    t, f, r, hw = _i64(), _i64(), _i32(), _i64()
    _check(lib.kv_pool_stats(handle, ctypes.byref(t), ctypes.byref(f), ctypes.byref(r), ctypes.byref(hw)),
           "kv_pool_stats")
    return {"blocks_total": t.value, "blocks_free": f.value, "live_requests": r.value, "blocks_high_water": hw.value}


def kv_gather(handle: int, req_id: int, k_dst_ptr: int, v_dst_ptr: int, stream: int = 0) -> None:
    _check(lib.kv_gather(handle, req_id, k_dst_ptr, v_dst_ptr, stream or None), "kv_gather")


def kv_gather_bytes(cfg: PoolConfig, n_tokens: int) -> int:
    c = cfg._c()
    n = lib.kv_gather_bytes(ctypes.byref(c), n_tokens)
    if n < 0:
        raise KVError(int(n), "kv_gather_bytes")
    return int(n)


def kv_transfer(dst_handle: int, src_handle: int, dst_req_ids, src_req_ids, layer_begin: int = 0, layer_count: int = 1,
                stream: int = 0) -> None:
    """NEXT-4: requests src_req_ids of the producer pool become requests dst_req_ids of the consumer pool."""
    d, s_ = _ids(dst_req_ids), _ids(src_req_ids)
    assert d.shape == s_.shape
    _check(lib.kv_transfer(dst_handle, src_handle, d.size, _np(d), _np(s_), layer_begin, layer_count, stream or None),
           "kv_transfer")


def kv_plan_decode(handle: int, req_ids):
    """Returns (items int32 [n][5] = (batch_idx, kv_head, blk_begin, n_blocks, partial_idx), chunk_blocks)."""
    ids = _ids(req_ids)
    n, ch = _i32(), _i32()
    _check(lib.kv_plan_decode(handle, ids.size, _np(ids), None, 0, ctypes.byref(n), ctypes.byref(ch)),
           "kv_plan_decode")
    items = np.empty((n.value, 5), dtype=np.int32)
    _check(lib.kv_plan_decode(handle, ids.size, _np(ids), _np(items), n.value, ctypes.byref(n), ctypes.byref(ch)),
           "kv_plan_decode")
    return items, ch.value


class _CapacityModel(ctypes.Structure):
    _fields_ = [("m_gpu", ctypes.c_double), ("m_reserved", ctypes.c_double), ("m_model", ctypes.c_double),
                ("tp", ctypes.c_int32), ("bw", ctypes.c_double), ("alpha", ctypes.c_double),
                ("t_d_slo", ctypes.c_double), ("isl", ctypes.c_double), ("osl", ctypes.c_double),
                ("m_token", ctypes.c_double)]


class _Capacity(ctypes.Structure):
    _fields_ = [("v_mem", ctypes.c_double), ("v_bw", ctypes.c_double), ("cc_d", ctypes.c_double),
                ("bandwidth_bound", ctypes.c_int32)]


def kv_capacity(m_gpu, m_reserved, m_model, tp, bw, alpha, t_d_slo, isl, osl, m_token) -> dict:
    """Eq. 11-13: {v_mem, v_bw, cc_d, bandwidth_bound}."""
    m = _CapacityModel(m_gpu, m_reserved, m_model, tp, bw, alpha, t_d_slo, isl, osl, m_token)
    r = _Capacity()
    _check(lib.kv_capacity(ctypes.byref(m), ctypes.byref(r)), "kv_capacity")
    return {"v_mem": r.v_mem, "v_bw": r.v_bw, "cc_d": r.cc_d, "bandwidth_bound": bool(r.bandwidth_bound)}


def kv_optimal_pd_ratio(cc_d, t_p, t_d, osl) -> float:
    """Eq. 14: n_p / n_d = cc_d * t_p / (t_d * OSL)."""
    r = ctypes.c_double()
    _check(lib.kv_optimal_pd_ratio(cc_d, t_p, t_d, osl, ctypes.byref(r)), "kv_optimal_pd_ratio")
    return float(r.value)


def kv_token_bytes(cfg: PoolConfig) -> int:
    c = cfg._c()
    n = lib.kv_token_bytes(ctypes.byref(c))
    if n < 0:
        raise KVError(int(n), "kv_token_bytes")
    return int(n)


def kv_launch_count(handle: int) -> int:
    return int(lib.kv_launch_count(handle))


def kv_pool_counter(handle: int, name: str) -> int:
    n = int(lib.kv_pool_counter(handle, name.encode()))
    if n < 0:
        raise KVError(n, f"kv_pool_counter({name})")
    return n


def kv_pool_set_option(handle: int, key: str, value: int) -> None:
    _check(lib.kv_pool_set_option(handle, key.encode(), value), f"kv_pool_set_option({key})")


def kv_last_cuda_error(handle: int) -> int:
    return int(lib.kv_last_cuda_error(handle))


class KVPool:
    """A pool handle plus the torch uint8 slab it lives in (PyTorch = device memory and streams only)."""

    def __init__(self, cfg: PoolConfig, device=None, fill_byte: int | None = None):
        import torch

        self.cfg = cfg
        self.kv_bytes = kv_pool_kv_bytes(cfg)
        if device is None:  # host-only pool: allocator + planner, no kernels
            self.slab = None
            self.handle = kv_pool_create(cfg)
        else:
            nbytes = kv_pool_required_bytes(cfg)
            self.slab = torch.empty(nbytes, dtype=torch.uint8, device=device)
            if fill_byte is not None:
                self.slab[: self.kv_bytes].fill_(fill_byte)
            self.handle = kv_pool_create(cfg, self.slab.data_ptr(), nbytes)

    def kv_region(self):
        """The KV region as a bf16 tensor [L][num_blocks][Hkv][2][block_size][head_dim] (a view)."""
        import torch

        c = self.cfg
        return self.slab[: self.kv_bytes].view(torch.bfloat16).view(
            c.num_layers, c.num_blocks, c.num_kv_heads, 2, c.block_size, c.head_dim)

    @staticmethod
    def _stream(stream) -> int:
        if stream is None:
            import torch
            return torch.cuda.current_stream().cuda_stream
        return stream if isinstance(stream, int) else stream.cuda_stream

    def reserve(self, req_ids, n_tokens):
        kv_reserve(self.handle, req_ids, n_tokens)

    def ingest(self, req_ids, k_src, v_src, layer_begin=0, layer_count=None, stream=None):
        """k_src[i], v_src[i]: bf16 CUDA tensors [layer_count][Hkv][n_i][d], contiguous."""
        lc = self.cfg.num_layers - layer_begin if layer_count is None else layer_count
        n = [int(k.shape[2]) for k in k_src]
        for k, v in zip(k_src, v_src):
            assert k.is_contiguous() and v.is_contiguous() and k.shape == v.shape and k.shape[0] == lc
        kv_ingest(self.handle, req_ids, n, k_src, v_src, layer_begin, lc, self._stream(stream))

    def attention(self, layer, req_ids, q, out=None, sm_scale=0.0, stream=None):
        import torch

        assert q.is_contiguous() and q.dtype == torch.bfloat16
        if out is None:
            out = torch.empty_like(q)
        paged_decode_attention(self.handle, layer, req_ids, q.data_ptr(), out.data_ptr(), sm_scale, self._stream(stream))
        return out

    def decode_attention_static(self, layer, req_ids, q, out=None, sm_scale=0.0, stream=None):
        """decode_attention through paged_decode_attention_static: split-KV workspace in the library's static
        device array, no allocation inside the call (``out`` given).  KV_ERR_SCRATCH_LIMIT beyond
        KV_STATIC_MAX_PARTIALS partial slots."""
        import torch

        assert q.is_contiguous() and q.dtype == torch.bfloat16
        if out is None:
            out = torch.empty_like(q)
        paged_decode_attention_static(self.handle, layer, req_ids, q.data_ptr(), out.data_ptr(), sm_scale,
                                      self._stream(stream))
        return out

    def decode_step(self, layer, req_ids, q, k_new, v_new, out=None, sm_scale=0.0, stream=None):
        """Fused append + attention for one layer; k_new / v_new: bf16 [batch][Hkv][d].  The caller has
        reserved the step's token with ``reserve(req_ids, ones)``."""
        import torch

        assert q.is_contiguous() and k_new.is_contiguous() and v_new.is_contiguous()
        if out is None:
            out = torch.empty_like(q)
        paged_decode_step(self.handle, layer, req_ids, q.data_ptr(), k_new.data_ptr(), v_new.data_ptr(),
                          out.data_ptr(), sm_scale, self._stream(stream))
        return out

    def varlen_attention(self, layer, req_ids, q_lens, q, out=None, sm_scale=0.0, stream=None):
        """q: bf16 [sum(q_lens)][Hq][d]; decode rows have q_len 1, in-place prefill rows their prompt length."""
        import torch

        assert q.is_contiguous() and q.dtype == torch.bfloat16 and q.shape[0] == int(sum(int(x) for x in q_lens))
        if out is None:
            out = torch.empty_like(q)
        paged_varlen_attention(self.handle, layer, req_ids, q_lens, q.data_ptr(), out.data_ptr(), sm_scale,
                               self._stream(stream))
        return out

    def varlen_step(self, layer, req_ids, q_lens, q, k_new, v_new, out=None, sm_scale=0.0, reserve=False, stream=None):
        """k_new[i], v_new[i]: bf16 [Hkv][q_lens[i]][d] of THIS layer; q: bf16 [sum(q_lens)][Hq][d]."""
        import torch

        assert q.is_contiguous() and q.dtype == torch.bfloat16 and all(t.is_contiguous() for t in list(k_new) + list(v_new))
        if out is None:
            out = torch.empty_like(q)
        paged_varlen_step(self.handle, layer, req_ids, q_lens, q.data_ptr(), [t.data_ptr() for t in k_new],
                          [t.data_ptr() for t in v_new], out.data_ptr(), sm_scale, KV_STEP_RESERVE if reserve else 0,
                          self._stream(stream))
        return out

    def gather(self, req_id, stream=None, src_kv_heads=None):
        """bf16 pool: (k, v) bf16 [L][H][n][d].  FP8 pool: (k_codes u8 [L][H][n][d], k_scales f32 [L][H][n],
        v_codes, v_scales) — views of the two buffers kv_gather fills.  H = src_kv_heads or the pool's kv heads."""
        import torch

        _, n = kv_block_table(self.handle, req_id)
        c = self.cfg
        H = src_kv_heads or c.num_kv_heads
        dev = self.slab.device
        if c.kv_dtype == KV_DTYPE_BF16:
            k = torch.empty((c.num_layers, H, n, c.head_dim), dtype=torch.bfloat16, device=dev)
            v = torch.empty_like(k)
            kv_gather(self.handle, req_id, k.data_ptr(), v.data_ptr(), self._stream(stream))
            return k, v
        rows = c.num_layers * H * n
        codes = (rows * c.head_dim + 15) // 16 * 16
        kb = torch.empty(codes + 4 * rows, dtype=torch.uint8, device=dev)
        vb = torch.empty_like(kb)
        kv_gather(self.handle, req_id, kb.data_ptr(), vb.data_ptr(), self._stream(stream))
        split = lambda b: (b[: rows * c.head_dim].view(c.num_layers, H, n, c.head_dim),
                           b[codes:].view(torch.float32).view(c.num_layers, H, n))
        return (*split(kb), *split(vb))

    def transfer_from(self, src: "KVPool", dst_req_ids, src_req_ids, layer_begin=0, layer_count=None, stream=None):
        """NEXT-4: pull requests out of the producer pool `src` into this pool, block to block."""
        lc = self.cfg.num_layers - layer_begin if layer_count is None else layer_count
        kv_transfer(self.handle, src.handle, dst_req_ids, src_req_ids, layer_begin, lc, self._stream(stream))

    def free(self, req_ids):
        kv_free(self.handle, req_ids)

    def profile(self) -> dict:
        """{kernel: (launches, total ms)} since the last profile_reset() (option profile=1)."""
        return {k: kv_profile_read(self.handle, i) for k, i in KERNEL_KINDS.items()}

    def profile_reset(self):
        kv_profile_reset(self.handle)

    def block_table(self, req_id):
        return kv_block_table(self.handle, req_id)

    def stats(self):
        return kv_pool_stats(self.handle)

    def plan(self, req_ids):
        return kv_plan_decode(self.handle, req_ids)

    def set_option(self, key, value):
        kv_pool_set_option(self.handle, key, value)

    @property
    def launches(self) -> int:
        return kv_launch_count(self.handle)

    def counter(self, name: str) -> int:
        return kv_pool_counter(self.handle, name)

    def close(self):
        if getattr(self, "handle", None):
            kv_pool_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
