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
  R-39  The cos / sin tables are MODEL STATE (the architecture precomputes them once and stores them in fp32), i.e. an
        input of the step like the norm weights: `apply` takes them as arguments and uses the values it is given
        (fp32 table entries are exact in fp64).  `rope_table` is the definition they must satisfy.
  R-40  Arithmetic and rounding.  Inputs are bf16; the result is rounded to bf16 (round to nearest even; results
        whose magnitude is below the smallest normal bf16, 2^-126, become signed zero) because the cache and the
        attention kernel hold bf16.  This file is the DEFINITION: fp64 throughout (BASELINE.json north_star: "NumPy in
        fp64"), ONE rounding to bf16 at the end, every operation before it rounded once in fp64, in this order (no
        fused multiply-add).  The CUDA kernel computes in fp32 and is compared with this file within one bf16 ulp
        (tests/test_gpu_fused_append.py); what follows the rounding (pooling, indices, attention) is then checked
        bit-exactly by feeding the kernel's OWN bf16 bits to oracle/uf_oracle.py (teacher forcing), because a
        last-bit difference in a cached K legitimately moves a pooled mean.  Nothing in this file is taken from the
        kernel's arithmetic (history: 2725cb1 wrote it, ce6d265 replaced it by a float32 mirror of the kernel, round 3
        restored it; the mirror lives on as tests/fused_fp32_model.py, a model of the kernel, not an oracle):
            ss = sum_j x_j^2  (each x_j^2 is exact in fp64; the sum is exact, hence order-free, as long as the
                               squares of one token span fewer than 2^37),
            m = ss / C;  r = 1 / sqrt(m + eps);  u_j = (x_j * r) * g_j;
            out_2i = u_2i * cos - u_2i+1 * sin;   out_2i+1 = u_2i * sin + u_2i+1 * cos.
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
    """fp64 -> nearest bf16 (ties to even), returned as uint16 bit patterns; |y| < 2^-126 -> signed zero (R-40).
    Done on the fp64 bits: keep sign, re-bias the exponent (1023 -> 127), keep the top 7 mantissa bits and round on
    the 45 bits below them."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    u = y.view(np.uint64)
    sign = ((u >> np.uint64(63)) & np.uint64(1)).astype(np.uint64)
    mag = u & np.uint64(0x7FFFFFFFFFFFFFFF)
    keep = mag >> np.uint64(45)                                   # exponent (11 bits) + top 7 mantissa bits
    rest = mag & np.uint64((1 << 45) - 1)
    half = np.uint64(1 << 44)
    up = (rest > half) | ((rest == half) & ((keep & np.uint64(1)) == np.uint64(1)))
    keep = keep + up.astype(np.uint64)                            # a carry into the exponent is the right result
    bias = np.uint64((1023 - 127) << 7)
    small = keep < bias + np.uint64(1 << 7)                       # below 2^-126 after rounding: flush
    out = np.where(small, np.uint64(0), keep - bias)
    assert not (out >= np.uint64(0x7F80)).any(), "overflow to inf / NaN: outside the step's domain"
    return ((sign << np.uint64(15)) | out).astype(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def rms_factor(X: np.ndarray, eps: float = EPS) -> np.ndarray:
    """r = 1 / sqrt(mean over ALL channels of the token of x^2 + eps) (R-37).  X fp64 [n, H, d] -> [n]"""
    n = X.shape[0]
    C = X.shape[1] * X.shape[2]
    ss = (X * X).reshape(n, C).sum(axis=1)
    return 1.0 / np.sqrt(ss / float(C) + eps)


def apply_unrounded(X: np.ndarray, g: np.ndarray, cos: np.ndarray, sin: np.ndarray, pos, dims=AXIS_DIMS,
                    eps: float = EPS) -> np.ndarray:
    """QK-norm + 3-D RoPE of one projection output, BEFORE the rounding to bf16.  X fp64 [n, H, d] (exact bf16 values),
    g [H*d], cos / sin [max_pos, d/2] (any float dtype: used as fp64), pos = (t, y, x) integer arrays [n].
    Returns fp64 [n, H, d]."""
    X = np.asarray(X, dtype=np.float64)
    cos, sin = np.asarray(cos, dtype=np.float64), np.asarray(sin, dtype=np.float64)
    n, H, d = X.shape
    assert sum(dims) == d and g.shape == (H * d,)
    r = rms_factor(X, eps)
    U = (X * r[:, None, None]) * np.asarray(g, dtype=np.float64).reshape(1, H, d)
    ax = pair_axis(dims)                                          # [d/2]
    P = np.stack(pos, axis=1)[:, ax]                              # [n, d/2] position that drives each pair
    col = np.arange(d // 2)[None, :]
    c = cos[P, col][:, None, :]                                   # [n, 1, d/2]
    s = sin[P, col][:, None, :]
    ue, uo = U[:, :, 0::2], U[:, :, 1::2]
    out = np.empty_like(U)
    out[:, :, 0::2] = ue * c - uo * s
    out[:, :, 1::2] = ue * s + uo * c
    return out


def apply(X: np.ndarray, g: np.ndarray, cos: np.ndarray, sin: np.ndarray, pos, dims=AXIS_DIMS, eps: float = EPS):
    """`apply_unrounded` followed by the ONE rounding to bf16 (R-40).  Returns uint16 bf16 bits [n, H, d]."""
    return round_to_bf16(apply_unrounded(X, g, cos, sin, pos, dims, eps))
