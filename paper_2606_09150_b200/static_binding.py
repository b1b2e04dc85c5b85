"""ctypes binding of include/uf_static.h — argument marshalling only.

`uf_select_blocks_static` is the one call of the library that allocates no device memory: block pooling, Eq. 4 scores
and top-k on the caller's Q and K, with the pooled tables in a fixed 16 MiB `static __device__` array inside libuf.so.
It exists for hosts that cannot cudaMalloc (plug-ins under a no-allocation contract, processes whose GPU memory another
allocator owns, loops that cannot take cudaMalloc's device-wide synchronisation).  See the header for the size limits
and for what calls that overlap on one GPU do to each other (they race on the array).
"""
from __future__ import annotations

from ctypes import c_char_p, c_int32, c_int64, c_void_p

from .binding import UFError, _ptr, _stream, load_library

UF_STATIC_SCRATCH_BYTES = 16 * 1024 * 1024
UF_STATIC_MAX_KEY_BLOCKS = 4096

# every symbol include/uf_static.h declares
STATIC_SYMBOLS = ["uf_select_blocks_static", "uf_static_last_error"]

_ready = False


def _lib():
    global _ready
    lib = load_library()
    if not _ready:
        P = c_void_p
        lib.uf_select_blocks_static.argtypes = [c_int32, P, c_int32, c_int64, c_int64, P, c_int32, c_int64, c_int64,
                                                c_int32, c_int32, c_int32, c_int32, P, P]
        lib.uf_select_blocks_static.restype = c_int32
        lib.uf_static_last_error.argtypes = []
        lib.uf_static_last_error.restype = c_char_p
        _ready = True
    return lib


def uf_static_last_error() -> str:
    msg = _lib().uf_static_last_error()
    return msg.decode() if msg else ""


def uf_select_blocks_static(device: int, q, n_q_tokens: int, q_tok_stride: int, q_head_stride: int,
                            k, n_k_tokens: int, k_tok_stride: int, k_head_stride: int,
                            n_heads: int, head_dim: int, block: int, topk_count: int, idx_out, stream=None) -> None:
    """idx_out: device int32 [n_heads, ceil(n_q_tokens / block), min(topk_count, ceil(n_k_tokens / block))]."""
    lib = _lib()
    code = lib.uf_select_blocks_static(device, _ptr(q), n_q_tokens, q_tok_stride, q_head_stride,
                                       _ptr(k), n_k_tokens, k_tok_stride, k_head_stride,
                                       n_heads, head_dim, block, topk_count, _ptr(idx_out), _stream(stream))
    if code != 0:
        raise UFError(code, uf_static_last_error())


__all__ = ["STATIC_SYMBOLS", "UF_STATIC_SCRATCH_BYTES", "UF_STATIC_MAX_KEY_BLOCKS"] + STATIC_SYMBOLS
