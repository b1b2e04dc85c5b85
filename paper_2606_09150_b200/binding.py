"""ctypes binding of include/uf.h — argument marshalling only.

Every function has the name and the arguments of the C call it wraps; tensors are passed as
objects with `.data_ptr()` (torch tensors) or as raw integer addresses.  Nothing of the method is
computed here: pooling, scoring, top-k, cache policy and attention all run inside libuf.so.
There is no fallback: if the library is missing or a call fails, `UFError` is raised.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_float, c_int32, c_int64, c_void_p

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libuf.so")

UF_OK, UF_ERR_INVALID_ARG, UF_ERR_STATE, UF_ERR_CAPACITY, UF_ERR_UNSUPPORTED, UF_ERR_CUDA = range(6)
UF_MAX_CAPACITY_CHUNKS = 16
_ERR_NAMES = {1: "UF_ERR_INVALID_ARG", 2: "UF_ERR_STATE", 3: "UF_ERR_CAPACITY", 4: "UF_ERR_UNSUPPORTED",
              5: "UF_ERR_CUDA"}

# every symbol include/uf.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "uf_ctx_create", "uf_ctx_destroy", "uf_ctx_reset", "uf_kv_append", "uf_query_topk", "uf_select_blocks",
    "uf_sparse_attn_fwd", "uf_set_attn_impl", "uf_get_slot_map", "uf_get_cache_block", "uf_get_pooled_k",
    "uf_attn_redone_items", "uf_ctx_device_bytes", "uf_ctx_launch_count", "uf_last_error", "uf_version",
    "uf_next_window", "uf_get_select_usage", "uf_qkv_rope_append", "uf_set_pooled_q_reuse",
    "uf_ctx_set_tiling", "uf_query_budget_paper", "uf_select_blocks_paper", "uf_tile_tokens", "uf_untile_tokens",
]


class UFError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class uf_config(Structure):
    _fields_ = [(n, c_int32) for n in ("n_heads", "head_dim", "block", "chunk_tokens_max", "capacity_chunks",
                                       "sink_blocks", "k_min", "device")]


class uf_tiling(Structure):
    _fields_ = [(n, c_int32) for n in ("frames", "grid_h", "grid_w", "bt", "bh", "bw", "window")]


UF_WIN_FIXED, UF_WIN_POSITION, UF_WIN_MEMORY, UF_WIN_CONTENT = range(4)


class uf_rope_spec(Structure):
    _fields_ = [("cos_tab", c_void_p), ("sin_tab", c_void_p), ("gq", c_void_p), ("gk", c_void_p), ("eps", c_double),
                ("max_pos", c_int32), ("t0", c_int32), ("grid_h", c_int32), ("grid_w", c_int32),
                ("dim_t", c_int32), ("dim_h", c_int32), ("dim_w", c_int32)]


class uf_window_policy(Structure):
    _fields_ = [("kind", c_int32), ("warm_chunks", c_int32), ("compact_window", c_int32),
                ("min_share_permille", c_int32), ("budget_bytes", c_int64)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libuf.so (built in-tree by paper_2606_09150_b200.build); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise UFError(UF_ERR_UNSUPPORTED, f"{LIB_PATH} not built: run `python -m paper_2606_09150_b200.build` "
                                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    P = c_void_p
    lib.uf_ctx_create.argtypes = [POINTER(uf_config), POINTER(P)]
    lib.uf_ctx_destroy.argtypes = [P]
    lib.uf_ctx_reset.argtypes = [P, P]
    lib.uf_kv_append.argtypes = [P, P, P, c_int32, c_int64, c_int64, c_int32, P]
    lib.uf_query_topk.argtypes = [P, c_int32, c_int32, POINTER(c_int32), POINTER(c_int32)]
    lib.uf_select_blocks.argtypes = [P, P, c_int32, c_int64, c_int64, c_int32, c_int32, P, P, P]
    lib.uf_sparse_attn_fwd.argtypes = [P, P, P, P, c_int32, c_int64, c_int64, c_float, P]
    lib.uf_set_attn_impl.argtypes = [P, c_int32]
    lib.uf_get_slot_map.argtypes = [P, POINTER(c_int32), POINTER(c_int32), POINTER(c_int32)]
    lib.uf_get_cache_block.argtypes = [P, c_int32, c_int32, P, P, P]
    lib.uf_get_pooled_k.argtypes = [P, c_int32, c_int32, POINTER(c_double), P]
    lib.uf_ctx_device_bytes.argtypes = [P]
    lib.uf_ctx_device_bytes.restype = c_int64
    lib.uf_attn_redone_items.argtypes = [P, POINTER(c_int32), P]
    lib.uf_ctx_launch_count.argtypes = [P]
    lib.uf_ctx_launch_count.restype = c_int64
    lib.uf_last_error.argtypes = [P]
    lib.uf_last_error.restype = c_char_p
    lib.uf_ctx_set_tiling.argtypes = [P, POINTER(uf_tiling)]
    lib.uf_query_budget_paper.argtypes = [P, c_int32, c_int32, POINTER(c_int32), POINTER(c_int32)]
    lib.uf_select_blocks_paper.argtypes = [P, P, c_int32, c_int64, c_int64, c_int32, c_int32, P, c_int32, P, P]
    lib.uf_tile_tokens.argtypes = [P, P, P, c_int64, c_int64, c_int64, c_int64, P]
    lib.uf_untile_tokens.argtypes = [P, P, P, c_int64, c_int64, c_int64, c_int64, P]
    lib.uf_qkv_rope_append.argtypes = [P, P, P, P, P, c_int32, c_int64, c_int64, c_int64, c_int64,
                                       POINTER(uf_rope_spec), c_int32, P]
    lib.uf_set_pooled_q_reuse.argtypes = [P, c_int32]
    lib.uf_next_window.argtypes = [P, POINTER(uf_window_policy), POINTER(c_int32), P]
    lib.uf_get_select_usage.argtypes = [P, POINTER(c_int64), POINTER(c_int32), POINTER(c_int32), P]
    lib.uf_version.argtypes = []
    lib.uf_version.restype = c_char_p
    for name in SYMBOLS:
        if getattr(lib, name).restype is ctypes.c_int:
            getattr(lib, name).restype = c_int32
    _lib = lib
    return lib


def _ptr(x) -> c_void_p:
    if x is None:
        return c_void_p(0)
    if hasattr(x, "data_ptr"):
        return c_void_p(x.data_ptr())
    if hasattr(x, "ctypes"):                       # numpy array (host pointers of the getters)
        return c_void_p(x.ctypes.data)
    return c_void_p(int(x))


def _stream(s) -> c_void_p:
    if s is None:
        return c_void_p(0)
    if hasattr(s, "cuda_stream"):
        return c_void_p(s.cuda_stream)
    return c_void_p(int(s))


def _check(ctx, code: int):
    if code != UF_OK:
        msg = load_library().uf_last_error(ctx)
        raise UFError(code, msg.decode() if msg else "")


def uf_version() -> str:
    return load_library().uf_version().decode()


def uf_ctx_create(n_heads: int, head_dim: int, block: int, chunk_tokens_max: int, capacity_chunks: int,
                  sink_blocks: int = 1, k_min: int = 4, device: int = 0) -> c_void_p:
    lib = load_library()
    cfg = uf_config(n_heads, head_dim, block, chunk_tokens_max, capacity_chunks, sink_blocks, k_min, device)
    out = c_void_p(0)
    _check(None, lib.uf_ctx_create(byref(cfg), byref(out)))
    return out


def uf_ctx_destroy(ctx) -> None:
    _check(None, load_library().uf_ctx_destroy(ctx))


def uf_ctx_reset(ctx, stream=None) -> None:
    _check(ctx, load_library().uf_ctx_reset(ctx, _stream(stream)))


def uf_kv_append(ctx, k, v, n_tokens: int, tok_stride: int, head_stride: int, window_chunks: int = 0,
                 stream=None) -> None:
    _check(ctx, load_library().uf_kv_append(ctx, _ptr(k), _ptr(v), n_tokens, tok_stride, head_stride,
                                            window_chunks, _stream(stream)))


def uf_query_topk(ctx, topk_count: int = -1, topk_percent: int = -1) -> tuple[int, int]:
    """-> (|CAND|, k')"""
    n_cand, k_eff = c_int32(0), c_int32(0)
    _check(ctx, load_library().uf_query_topk(ctx, topk_count, topk_percent, byref(n_cand), byref(k_eff)))
    return n_cand.value, k_eff.value


def uf_select_blocks(ctx, q, n_tokens: int, tok_stride: int, head_stride: int, topk_count: int = -1,
                     topk_percent: int = -1, idx_out=None, cnt_out=None, stream=None) -> None:
    _check(ctx, load_library().uf_select_blocks(ctx, _ptr(q), n_tokens, tok_stride, head_stride, topk_count,
                                                topk_percent, _ptr(idx_out), _ptr(cnt_out), _stream(stream)))


def uf_qkv_rope_append(ctx, q_in, k_in, v_in, q_out, n_tokens: int, in_tok_stride: int, in_head_stride: int,
                       out_tok_stride: int, out_head_stride: int, cos_tab, sin_tab, gq, gk, max_pos: int, t0: int,
                       grid_h: int, grid_w: int, dims=(44, 42, 42), eps: float = 1e-6, window_chunks: int = 0,
                       stream=None) -> None:
    rs = uf_rope_spec(_ptr(cos_tab), _ptr(sin_tab), _ptr(gq), _ptr(gk), eps, max_pos, t0, grid_h, grid_w, *dims)
    _check(ctx, load_library().uf_qkv_rope_append(ctx, _ptr(q_in), _ptr(k_in), _ptr(v_in), _ptr(q_out), n_tokens,
                                                  in_tok_stride, in_head_stride, out_tok_stride, out_head_stride,
                                                  byref(rs), window_chunks, _stream(stream)))


def uf_set_pooled_q_reuse(ctx, on: bool) -> None:
    _check(ctx, load_library().uf_set_pooled_q_reuse(ctx, 1 if on else 0))


def uf_next_window(ctx, kind: int, warm_chunks: int = 0, compact_window: int = 1, min_share_permille: int = 0,
                   budget_bytes: int = 0, stream=None) -> int:
    """-> window_chunks for the next uf_kv_append"""
    p = uf_window_policy(kind, warm_chunks, compact_window, min_share_permille, budget_bytes)
    w = c_int32(0)
    _check(ctx, load_library().uf_next_window(ctx, byref(p), byref(w), _stream(stream)))
    return int(w.value)


def uf_get_select_usage(ctx, stream=None) -> tuple[list[int], list[int]]:
    """-> (kept top-k blocks per listed chunk, the chunks' ids), ascending chunk id"""
    kept = (c_int64 * UF_MAX_CAPACITY_CHUNKS)()
    ids = (c_int32 * UF_MAX_CAPACITY_CHUNKS)()
    n = c_int32(0)
    _check(ctx, load_library().uf_get_select_usage(ctx, kept, ids, byref(n), _stream(stream)))
    return list(kept[:n.value]), list(ids[:n.value])


def uf_ctx_set_tiling(ctx, frames: int, grid_h: int, grid_w: int, bt: int = 2, bh: int = 8, bw: int = 8,
                      window: int = 9) -> None:
    t = uf_tiling(frames, grid_h, grid_w, bt, bh, bw, window)
    _check(ctx, load_library().uf_ctx_set_tiling(ctx, byref(t)))


def uf_query_budget_paper(ctx, topk_count: int = -1, rho_permille: int = 1000) -> tuple[int, int]:
    """-> (N_blocks in the causal mask, k')"""
    n_blocks, k_eff = c_int32(0), c_int32(0)
    _check(ctx, load_library().uf_query_budget_paper(ctx, topk_count, rho_permille, byref(n_blocks), byref(k_eff)))
    return n_blocks.value, k_eff.value


def uf_select_blocks_paper(ctx, q, n_tokens: int, tok_stride: int, head_stride: int, topk_count: int = -1,
                           rho_permille: int = 1000, idx_out=None, idx_stride: int = 0, cnt_out=None,
                           stream=None) -> None:
    _check(ctx, load_library().uf_select_blocks_paper(ctx, _ptr(q), n_tokens, tok_stride, head_stride, topk_count,
                                                      rho_permille, _ptr(idx_out), idx_stride, _ptr(cnt_out),
                                                      _stream(stream)))


def uf_tile_tokens(ctx, raster, tiled, raster_tok_stride: int, raster_head_stride: int, tiled_tok_stride: int,
                   tiled_head_stride: int, stream=None) -> None:
    _check(ctx, load_library().uf_tile_tokens(ctx, _ptr(raster), _ptr(tiled), raster_tok_stride, raster_head_stride,
                                              tiled_tok_stride, tiled_head_stride, _stream(stream)))


def uf_untile_tokens(ctx, tiled, raster, tiled_tok_stride: int, tiled_head_stride: int, raster_tok_stride: int,
                     raster_head_stride: int, stream=None) -> None:
    _check(ctx, load_library().uf_untile_tokens(ctx, _ptr(tiled), _ptr(raster), tiled_tok_stride, tiled_head_stride,
                                                raster_tok_stride, raster_head_stride, _stream(stream)))


def uf_sparse_attn_fwd(ctx, q, o, lse, n_tokens: int, tok_stride: int, head_stride: int,
                       softmax_scale: float = 0.0, stream=None) -> None:
    _check(ctx, load_library().uf_sparse_attn_fwd(ctx, _ptr(q), _ptr(o), _ptr(lse), n_tokens, tok_stride,
                                                  head_stride, softmax_scale, _stream(stream)))


def uf_set_attn_impl(ctx, impl: int) -> None:
    _check(ctx, load_library().uf_set_attn_impl(ctx, impl))


def uf_get_slot_map(ctx, capacity_chunks: int) -> tuple[list[int], int, int]:
    """-> (slot -> chunk id or -1, number resident, newest chunk id)"""
    arr = (c_int32 * UF_MAX_CAPACITY_CHUNKS)()
    n_res, newest = c_int32(0), c_int32(0)
    _check(ctx, load_library().uf_get_slot_map(ctx, arr, byref(n_res), byref(newest)))
    return list(arr[:capacity_chunks]), n_res.value, newest.value


def uf_get_cache_block(ctx, global_block: int, head: int, k_out, v_out, stream=None) -> None:
    """k_out, v_out: host buffers (numpy uint16 [B, d]) or None."""
    _check(ctx, load_library().uf_get_cache_block(ctx, global_block, head, _ptr(k_out), _ptr(v_out),
                                                  _stream(stream)))


def uf_get_pooled_k(ctx, global_block: int, head: int, out, stream=None) -> None:
    """out: host buffer, numpy float64 [d]."""
    _check(ctx, load_library().uf_get_pooled_k(ctx, global_block, head,
                                               ctypes.cast(_ptr(out), POINTER(c_double)), _stream(stream)))


def uf_ctx_device_bytes(ctx) -> int:
    return load_library().uf_ctx_device_bytes(ctx)


def uf_attn_redone_items(ctx, stream=None) -> int:
    n = c_int32(0)
    _check(ctx, load_library().uf_attn_redone_items(ctx, byref(n), _stream(stream)))
    return int(n.value)


def uf_ctx_launch_count(ctx) -> int:
    return load_library().uf_ctx_launch_count(ctx)


def uf_last_error(ctx=None) -> str:
    msg = load_library().uf_last_error(ctx)
    return msg.decode() if msg else ""


__all__ = ["LIB_PATH", "SYMBOLS", "UFError", "load_library", "uf_config", "uf_tiling", "uf_window_policy", "uf_rope_spec",
           "UF_WIN_FIXED", "UF_WIN_POSITION", "UF_WIN_MEMORY", "UF_WIN_CONTENT"] + SYMBOLS
