"""paper_2606_09150_b200 — B200-native sparse causal chunk attention of Ultra Flash (arxiv/paper_2606_09150).

The product is the C-ABI library `libuf.so` (include/uf.h; CUDA sources in `csrc/`, built in-tree
by `build.py` for sm_100a).  This package is its thin ctypes binding: same call names, argument
marshalling only.  No CPU fallback exists; importing works without a GPU, every device call fails
loudly (UFError) without one.
"""
from .binding import (  # noqa: F401
    LIB_PATH, SYMBOLS, UFError, load_library, uf_ctx_create, uf_ctx_destroy, uf_ctx_device_bytes,
    uf_attn_redone_items, uf_ctx_launch_count, uf_ctx_reset, uf_get_cache_block, uf_get_pooled_k, uf_get_slot_map, uf_kv_append,
    uf_last_error, uf_query_topk, uf_select_blocks, uf_set_attn_impl, uf_sparse_attn_fwd, uf_version,
)
from .build import build  # noqa: F401

__all__ = [
    "LIB_PATH", "SYMBOLS", "UFError", "build", "load_library", "uf_ctx_create", "uf_ctx_destroy",
    "uf_attn_redone_items", "uf_ctx_device_bytes", "uf_ctx_launch_count", "uf_ctx_reset", "uf_get_cache_block", "uf_get_pooled_k",
    "uf_get_slot_map", "uf_kv_append", "uf_last_error", "uf_query_topk", "uf_select_blocks", "uf_set_attn_impl",
    "uf_sparse_attn_fwd", "uf_version",
]
