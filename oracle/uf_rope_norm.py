"""CPU oracle for the step in front of the hot path: QK-norm + 3-D RoPE of the QKV projection output
(SURVEY.md section 8(f) NEXT-2), whose results feed kv_append / select_blocks / sparse_attn of oracle/uf_oracle.py.

*** TEST INFRASTRUCTURE — NOT A PRODUCT PATH *** (same rules as oracle/uf_oracle.py).

What the paper fixes: "The SR model follows the Wan2.1 architecture ... 12 heads (head dim 128); patch size
(1,2,2); 3D RoPE with axis dims (44,42,42)".  Everything else is that public architecture, restated (readings
R-37 ... R-40 in DESIGN.md):

  R-37  QK-norm: q and k (not v) are RMS-normalised over the WHOLE hidden vector (all H*d channels of a token)
        with a learned per-channel weight g, before the split into heads:
            y = x / sqrt(mean(x^2) + eps) * g,  eps = 1e-6.
  R-38  3-D RoPE: the d channels of every head are consecutive pairs (2i, 2i+1), i = 0 .. d/2-1, treated as
        complex numbers.  The first dim_t/2 pairs rotate with the token's temporal position t, the next dim_h/2
        with its row y, the last dim_w/2 with its column x ((dim_t, dim_h, dim_w) = (44, 42, 42)).  Pair i of
        an axis segment of dim D has frequency theta^(-2i/D), theta = 10000:
            (a + ib) -> (a + ib) * exp(i * pos * theta^(-2i/D)).
        Positions: t counts latent frames from the start of the stream (chunk c starts at t0 = c * F), y, x are the
        token-grid coordinates; tokens arrive in raster (t, y, x) order.
  R-39  The cos / sin tables are MODEL STATE (the architecture precomputes them once, in fp32), i.e. an input of the
        step like the norm weights: `apply` takes them as arguments.  `rope_table` is the definition they must
        satisfy (to fp32 rounding).
  R-40  Arithmetic and rounding.  Inputs are bf16; the result is rounded to bf16 because the cache and the attention
        kernel hold bf16.  That rounding decides cache bytes and, through pooling, block indices, so both sides take
        it in the SAME precision, the kernel's: fp32 with every operation rounded once (IEEE, no fused multiply-add),
        in this order (fl = round to fp32):
            ss = sum_j x_j^2   in fp64 (each x_j^2 is exact; the sum is exact, hence order-free, as long as the
                               squares of one token span fewer than 2^37 — else its last bit may depend on the order),
            r  = fl(1 / sqrt(ss / C + eps))          (the fp64 operations /, +, sqrt, / rounded once each, then fl),
            u_j = fl(fl(x_j * r) * g_j),
            out_2i = fl(fl(u_2i * cos) - fl(u_2i+1 * sin));   out_2i+1 = fl(fl(u_2i * sin) + fl(u_2i+1 * cos)),
            result = bf16(out)   round to nearest even (IEEE, subnormals kept).
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
