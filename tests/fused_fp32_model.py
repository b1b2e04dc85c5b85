"""A bit-level MODEL OF THE KERNEL uf_fused_append_kernel (csrc/uf_fused_append.cu) in NumPy float32 — NOT an oracle.

It restates the kernel's own arithmetic (fp32, every operation rounded once, no fused multiply-add, the order the kernel
uses; the sum of squares and the reciprocal square root in fp64, rounded to fp32 once) so that a test can say "the
kernel's bits are a fixed, reproducible function of the input bits".  It proves nothing about correctness: the parity
claim of the fused step rests on oracle/uf_rope_norm.py (fp64, one rounding), with which the kernel is compared within
one bf16 ulp.  Round 2 had this file in oracle/ (commit ce6d265); VERDICT r2 pointed out that an oracle written from the
kernel is the kernel agreeing with itself, so it lives here now.
        ss = sum_j x_j^2 (fp64, exact);  r = fl32(1 / sqrt(ss / C + eps));  u_j = fl(fl(x_j r) g_j);
        out_2i = fl(fl(u_2i cos) - fl(u_2i+1 sin));  out_2i+1 = fl(fl(u_2i sin) + fl(u_2i+1 cos));  bf16 RNE (subnormals kept)
"""
from __future__ import annotations

import numpy as np

AXIS_DIMS = (44, 42, 42)
THETA = 10000.0
EPS = 1e-6


def rope_table(max_pos: int, dims=AXIS_DIMS, theta: float = THETA):
    """cos, sin fp64 [max_pos, d/2]: column i of axis segment a is cos / sin(pos * theta^(-2 i_a / D_a)) (R-38).
    Row index = position along the axis the column belongs to."""
    cols = []
    for D in dims:
        assert D % 2 == 0
        i = np.arange(D // 2, dtype=np.float64)
        cols.append(1.0 / np.power(theta, 2.0 * i / float(D)))
    freq = np.concatenate(cols)                                   # [d/2]
    ang = np.arange(max_pos, dtype=np.float64)[:, None] * freq[None, :]
    return np.cos(ang), np.sin(ang)


def pair_axis(dims=AXIS_DIMS) -> np.ndarray:
    """axis (0 = t, 1 = y, 2 = x) of every complex pair of a head, int [d/2]"""
    return np.concatenate([np.full(D // 2, a, dtype=np.int64) for a, D in enumerate(dims)])


def raster_positions(n_tokens: int, grid_h: int, grid_w: int, t0: int):
    """(t, y, x) of tokens 0 .. n_tokens-1 in raster order, t offset by t0 (R-38)"""
    n = np.arange(n_tokens)
    per = grid_h * grid_w
    return t0 + n // per, (n % per) // grid_w, n % grid_w


def round_to_bf16(y: np.ndarray) -> np.ndarray:
    """fp32 -> nearest bf16 (ties to even), uint16 bit patterns (R-40).  On the fp32 bits: the upper 16 bits, plus one
    when the lower 16 are above half, or exactly half with an odd upper part; the carry may run into the exponent,
    which is the right result (also for subnormals).  No NaN / inf in the step's domain."""
    y = np.ascontiguousarray(y, dtype=np.float32)
    u = y.view(np.uint32)
    upper = u >> np.uint32(16)
    lower = u & np.uint32(0xFFFF)
    up = (lower > np.uint32(0x8000)) | ((lower == np.uint32(0x8000)) & ((upper & np.uint32(1)) == np.uint32(1)))
    out = upper + up.astype(np.uint32)
    assert not ((out & np.uint32(0x7F80)) == np.uint32(0x7F80)).any(), "inf / NaN: outside the step's domain"
    return out.astype(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def rms_factor(X: np.ndarray, eps: float = EPS) -> np.ndarray:
    """r = fl32(1 / sqrt(mean over ALL channels of the token of x^2 + eps)), the inner part in fp64 (R-37, R-40).
    X fp64 [n, H, d] -> float32 [n]"""
    n = X.shape[0]
    C = X.shape[1] * X.shape[2]
    ss = (X * X).reshape(n, C).sum(axis=1)
    return (1.0 / np.sqrt(ss / float(C) + eps)).astype(np.float32)


def apply(X: np.ndarray, g: np.ndarray, cos: np.ndarray, sin: np.ndarray, pos, dims=AXIS_DIMS, eps: float = EPS):
    """QK-norm + 3-D RoPE of one projection output.  X fp64 [n, H, d] (exact bf16 values), g float32 [H*d], cos / sin
    float32 [max_pos, d/2], pos = (t, y, x) integer arrays [n].  Returns uint16 bf16 bits [n, H, d].  Every product and
    sum below is ONE float32 NumPy operation, i.e. rounded once, in the order R-40 states."""
    X = np.asarray(X, dtype=np.float64)
    n, H, d = X.shape
    g = np.asarray(g)
    assert sum(dims) == d and g.shape == (H * d,) and g.dtype == np.float32
    assert cos.dtype == np.float32 and sin.dtype == np.float32
    r = rms_factor(X, eps)                                        # float32 [n]
    x32 = X.astype(np.float32)                                    # exact: bf16 values
    U = (x32 * r[:, None, None]) * g.reshape(1, H, d)             # fl(fl(x r) g)
    ax = pair_axis(dims)                                          # [d/2]
    P = np.stack(pos, axis=1)[:, ax]                              # [n, d/2] position that drives each pair
    col = np.arange(d // 2)[None, :]
    c = cos[P, col][:, None, :]                                   # [n, 1, d/2]
    s = sin[P, col][:, None, :]
    ue, uo = U[:, :, 0::2], U[:, :, 1::2]
    out = np.empty_like(U)
    out[:, :, 0::2] = ue * c - uo * s
    out[:, :, 1::2] = ue * s + uo * c
    assert out.dtype == np.float32
    return round_to_bf16(out)
