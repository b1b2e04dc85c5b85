"""ctypes binding of include/uf_cmn.h (causal memory network streaming step) — argument marshalling only.

Same names and arguments as the C calls; tensors are objects with `.data_ptr()` (torch), numpy arrays (host
pointers: weights, getters) or raw addresses.  All arithmetic of the network runs inside libuf.so; there is no
fallback (UFError on any failure).
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, Structure, byref, c_char_p, c_float, c_int32, c_int64, c_void_p

from .binding import UF_OK, UFError, _ERR_NAMES, _ptr, _stream, load_library  # noqa: F401

UF_CMN_MAX_STAGES = 4

# every symbol include/uf_cmn.h declares
CMN_SYMBOLS = [
    "uf_cmn_create", "uf_cmn_destroy", "uf_cmn_n_params", "uf_cmn_param_info", "uf_cmn_set_param", "uf_cmn_reset",
    "uf_cmn_step", "uf_cmn_get_memory", "uf_cmn_flops", "uf_cmn_device_bytes", "uf_cmn_launches", "uf_cmn_n_layers",
    "uf_cmn_layer_info", "uf_cmn_get_activation", "uf_cmn_last_error",
]


class uf_cmn_config(Structure):
    _fields_ = [("in_ch", c_int32), ("out_ch", c_int32), ("n_stages", c_int32),
                ("stage_channels", c_int32 * (UF_CMN_MAX_STAGES + 1)), ("n_blocks", c_int32),
                ("spatial_factors", c_int32 * UF_CMN_MAX_STAGES), ("temporal_factors", c_int32 * UF_CMN_MAX_STAGES),
                ("height", c_int32), ("width", c_int32), ("frames_max", c_int32), ("device", c_int32)]


_ready = False


def _lib():
    global _ready
    lib = load_library()
    if not _ready:
        P = c_void_p
        lib.uf_cmn_create.argtypes = [POINTER(uf_cmn_config), POINTER(P)]
        lib.uf_cmn_destroy.argtypes = [P]
        lib.uf_cmn_n_params.argtypes = [P]
        lib.uf_cmn_param_info.argtypes = [P, c_int32, c_char_p, c_int32, POINTER(c_int32), POINTER(c_int32)]
        lib.uf_cmn_set_param.argtypes = [P, c_char_p, P, P]
        lib.uf_cmn_reset.argtypes = [P, P]
        lib.uf_cmn_step.argtypes = [P, P, c_int32, P, P]
        lib.uf_cmn_get_memory.argtypes = [P, c_int32, c_int32, P, POINTER(c_int32), P]
        lib.uf_cmn_flops.argtypes = [P, c_int32]
        lib.uf_cmn_flops.restype = c_int64
        lib.uf_cmn_device_bytes.argtypes = [P]
        lib.uf_cmn_device_bytes.restype = c_int64
        lib.uf_cmn_launches.argtypes = [P]
        lib.uf_cmn_launches.restype = c_int64
        lib.uf_cmn_n_layers.argtypes = [P]
        lib.uf_cmn_layer_info.argtypes = [P, c_int32, c_char_p, c_int32, POINTER(c_int64), POINTER(c_int32),
                                          POINTER(c_int32), POINTER(c_int32)]
        lib.uf_cmn_get_activation.argtypes = [P, c_int32, P, POINTER(c_int32), P]
        lib.uf_cmn_last_error.argtypes = [P]
        lib.uf_cmn_last_error.restype = c_char_p
        for name in CMN_SYMBOLS:
            if getattr(lib, name).restype is ctypes.c_int:
                getattr(lib, name).restype = c_int32
        _ready = True
    return lib


def _check(net, code: int):
    if code != UF_OK:
        msg = _lib().uf_cmn_last_error(net)
        raise UFError(code, msg.decode() if msg else "")


def uf_cmn_create(in_ch: int, out_ch: int, stage_channels, n_blocks: int, spatial_factors, temporal_factors,
                  height: int, width: int, frames_max: int, device: int = 0) -> c_void_p:
    n_stages = len(spatial_factors)
    cfg = uf_cmn_config()
    cfg.in_ch, cfg.out_ch, cfg.n_stages, cfg.n_blocks = in_ch, out_ch, n_stages, n_blocks
    for i, c in enumerate(stage_channels):
        cfg.stage_channels[i] = c
    for i in range(n_stages):
        cfg.spatial_factors[i] = spatial_factors[i]
        cfg.temporal_factors[i] = temporal_factors[i]
    cfg.height, cfg.width, cfg.frames_max, cfg.device = height, width, frames_max, device
    out = c_void_p(0)
    _check(None, _lib().uf_cmn_create(byref(cfg), byref(out)))
    return out


def uf_cmn_destroy(net) -> None:
    _check(None, _lib().uf_cmn_destroy(net))


def uf_cmn_n_params(net) -> int:
    return _lib().uf_cmn_n_params(net)


def uf_cmn_param_info(net, index: int) -> tuple[str, tuple[int, int, int, int], bool]:
    name = ctypes.create_string_buffer(64)
    shape = (c_int32 * 4)()
    hb = c_int32(0)
    _check(net, _lib().uf_cmn_param_info(net, index, name, 64, shape, byref(hb)))
    return name.value.decode(), tuple(shape), bool(hb.value)


def uf_cmn_set_param(net, name: str, w_host, bias_host=None) -> None:
    """w_host: numpy uint16 (bf16 bits) [C_out, C_in, kh, kw] contiguous; bias_host: numpy float32 [C_out] or None"""
    _check(net, _lib().uf_cmn_set_param(net, name.encode(), _ptr(w_host), _ptr(bias_host)))


def uf_cmn_reset(net, stream=None) -> None:
    _check(net, _lib().uf_cmn_reset(net, _stream(stream)))


def uf_cmn_step(net, z, n_frames: int, out, stream=None) -> None:
    _check(net, _lib().uf_cmn_step(net, _ptr(z), n_frames, _ptr(out), _stream(stream)))


def uf_cmn_get_memory(net, stage: int, block: int, out_host, stream=None) -> tuple[int, int, int]:
    shape = (c_int32 * 3)()
    _check(net, _lib().uf_cmn_get_memory(net, stage, block, _ptr(out_host), shape, _stream(stream)))
    return tuple(shape)


def uf_cmn_flops(net, n_frames: int) -> int:
    return _lib().uf_cmn_flops(net, n_frames)


def uf_cmn_device_bytes(net) -> int:
    return _lib().uf_cmn_device_bytes(net)


def uf_cmn_launches(net) -> int:
    return _lib().uf_cmn_launches(net)


def uf_cmn_n_layers(net) -> int:
    return _lib().uf_cmn_n_layers(net)


def uf_cmn_layer_info(net, index: int) -> tuple[str, int, int, int, tuple[int, int, int, int]]:
    """-> (name, flops per input frame, GEMM N, GEMM K, (frames per input frame, rows, cols, channels) of its output)"""
    name = ctypes.create_string_buffer(64)
    fl, n, k = c_int64(0), c_int32(0), c_int32(0)
    shape = (c_int32 * 4)()
    _check(net, _lib().uf_cmn_layer_info(net, index, name, 64, byref(fl), byref(n), byref(k), shape))
    return name.value.decode(), fl.value, n.value, k.value, tuple(shape)


def uf_cmn_get_activation(net, layer: int, out_host, stream=None) -> tuple[int, int, int, int]:
    """out_host: numpy uint16 buffer large enough for the layer's output of the last step; -> its shape"""
    shape = (c_int32 * 4)()
    _check(net, _lib().uf_cmn_get_activation(net, layer, _ptr(out_host), shape, _stream(stream)))
    return tuple(shape)


def uf_cmn_last_error(net=None) -> str:
    msg = _lib().uf_cmn_last_error(net)
    return msg.decode() if msg else ""


__all__ = ["CMN_SYMBOLS", "uf_cmn_config", "UF_CMN_MAX_STAGES"] + CMN_SYMBOLS
