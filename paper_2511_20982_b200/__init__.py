"""B200-native D-instance KV data path (arxiv 2511.20982, DOPD): paged KV pool, KV ingest,
split-KV paged decode attention + LSE combine, behind the C-ABI of ``include/kv_pool.h``.

``paper_2511_20982_b200.workloads`` (seeded synthetic inputs) imports without the native
library.  Everything else is the thin ctypes binding in ``binding`` and is loaded on first
use; it raises ``ImportError`` loudly if ``csrc/libkvpool.so`` has not been built — there is
no CPU or PyTorch fallback for any step of the path.
"""
from __future__ import annotations

_BINDING_NAMES = (
    "KVPool", "KVError", "PoolConfig", "lib", "lib_path",
    "kv_pool_create", "kv_pool_destroy", "kv_pool_kv_bytes", "kv_pool_required_bytes", "kv_reserve",
    "kv_ingest", "paged_decode_attention", "kv_free", "kv_block_table", "kv_pool_stats", "kv_gather",
    "kv_plan_decode", "kv_launch_count", "paged_decode_step", "paged_decode_step_layers", "kv_transfer", "kv_gather_bytes", "kv_token_bytes", "kv_capacity", "kv_optimal_pd_ratio", "paged_varlen_attention", "paged_decode_step_host", "kv_ingest_host", "paged_decode_attention_host", "kv_profile_read", "kv_profile_reset", "kv_pool_set_option", "kv_last_cuda_error", "kv_strerror", "paged_decode_attention_static", "kv_static_scratch_bytes", "paged_varlen_step",
    "kv_version",
)


def __getattr__(name):
    if name in _BINDING_NAMES or name == "binding":
        import importlib
        _b = importlib.import_module(__name__ + ".binding")  # raises ImportError if the .so is missing
        return _b if name == "binding" else getattr(_b, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
