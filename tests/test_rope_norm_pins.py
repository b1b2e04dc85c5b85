"""Pins for oracle/uf_rope_norm.py (NEXT-2: QK-norm + 3-D RoPE) against the mathematics: complex exponentials computed
another way, rotation invariants, the relative-position property, closed forms of RMS normalisation, and the bf16
rounding against the storage-format converter and hand-worked ties.  CPU only."""
import numpy as np
import pytest

import uf_workloads as wl
from oracle import uf_rope_norm as rn


def bf16(x):
    return wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))).astype(np.float64)


def test_rope_table_is_exp_i_pos_freq_and_matches_the_model_state_generator():
    """cos + i sin == exp(i pos theta^(-2i/D)) via complex powers; segment sizes 22 / 21 / 21; frequency 1 at i = 0 of
    every axis; the table the workload generator hands to both sides satisfies the same definition."""
    cos, sin = rn.rope_table(50)
    assert cos.shape == sin.shape == (50, 64)
    ax = rn.pair_axis()
    assert (np.bincount(ax) == [22, 21, 21]).all() and (np.diff(ax) >= 0).all()
    for seg_start, D in ((0, 44), (22, 42), (43, 42)):
        for i in (0, 1, D // 2 - 1):
            base = np.exp(1j * 10000.0 ** (-2.0 * i / D))                 # rotation per unit position
            z = base ** np.arange(50)
            assert np.allclose(cos[:, seg_start + i], z.real, atol=1e-12) and np.allclose(sin[:, seg_start + i], z.imag, atol=1e-12)
        assert np.allclose(cos[:, seg_start], np.cos(np.arange(50))) and np.allclose(sin[:, seg_start], np.sin(np.arange(50)))
    c2, s2 = wl.rope_tables(50)
    # the model-state tables are fp32: half an fp32 ulp of a number <= 1, plus the last bit of the fp64 frequency
    assert c2.dtype == s2.dtype == np.float32
    tol = 2.0 ** -25 + 50 * 2.0 ** -51
    assert np.allclose(c2, cos, rtol=0, atol=tol) and np.allclose(s2, sin, rtol=0, atol=tol)


def _setup(seed, n=12, H=2, d=128, gh=3, gw=4, t0=5):
    rng = np.random.default_rng(seed)
    X = bf16(rng.standard_normal((n, H, d)))
    g = (1.0 + 0.1 * rng.standard_normal(H * d)).astype(np.float32)
    cos, sin = (t.astype(np.float32) for t in rn.rope_table(64))
    pos = rn.raster_positions(n, gh, gw, t0)
    return X, g, cos, sin, pos


def test_position_zero_is_identity_and_norm_closed_forms():
    """pos = (0,0,0) -> no rotation: the result is bf16(x * r * g); g = 1, eps = 0 -> every token has mean square 1;
    a constant vector c -> c / |c| * g; scaling x by 4 (exact) changes nothing when eps = 0."""
    X, g, cos, sin, _ = _setup(1)
    zero = (np.zeros(12, int),) * 3
    out = rn.bf16_bits_to_f64(rn.apply(X, g, cos, sin, zero))
    r = 1.0 / np.sqrt((X ** 2).reshape(12, -1).mean(axis=1) + 1e-6)
    want = X * r[:, None, None] * g.astype(np.float64).reshape(1, 2, 128)
    assert (np.abs(out - want) <= np.abs(want) * (2.0 ** -8 + 2.0 ** -21)).all()
    ones = np.ones(256, dtype=np.float32)
    y = rn.rms_factor(X, eps=0.0).astype(np.float64)[:, None, None] * X
    assert np.allclose((y ** 2).reshape(12, -1).mean(axis=1), 1.0, atol=1e-6)
    Cst = np.full((3, 2, 128), -2.5)
    zero3 = (np.zeros(3, int),) * 3
    assert np.array_equal(rn.apply(Cst, ones, cos, sin, zero3, eps=0.0), rn.round_to_bf16(np.full((3, 2, 128), -1.0)))
    assert np.array_equal(rn.apply(4.0 * X, g, cos, sin, zero, eps=0.0), rn.apply(X, g, cos, sin, zero, eps=0.0))


def _apply_exact(X, g, cos, sin, pos, eps=1e-6):
    """the same step WITHOUT the final rounding, written with complex numbers (independent formulation)"""
    n, H, d = X.shape
    r = 1.0 / np.sqrt((X ** 2).reshape(n, -1).mean(axis=1) + eps)
    U = X * r[:, None, None] * np.asarray(g, dtype=np.float64).reshape(1, H, d)
    cos, sin = cos.astype(np.float64), sin.astype(np.float64)
    Z = U[:, :, 0::2] + 1j * U[:, :, 1::2]
    ax = rn.pair_axis()
    P = np.stack(pos, axis=1)[:, ax]
    rot = (cos + 1j * sin)[P, np.arange(d // 2)[None, :]]
    Z = Z * rot[:, None, :]
    out = np.empty_like(U)
    out[:, :, 0::2], out[:, :, 1::2] = Z.real, Z.imag
    return out


def test_rotation_preserves_pair_norms_and_axes_are_separate():
    """|out pair| == |u pair| (a rotation); changing t alone changes only channels [0, 44), y only [44, 86),
    x only [86, 128) of every head; the rounded result is within half a bf16 ulp of the complex formulation."""
    X, g, cos, sin, pos = _setup(2)
    cos64, sin64 = rn.rope_table(64)                          # the definition, unrounded
    ex = _apply_exact(X, g, cos64, sin64, pos)
    base = _apply_exact(X, g, cos64, sin64, (0 * pos[0], 0 * pos[1], 0 * pos[2]))
    n2 = lambda A: A[:, :, 0::2] ** 2 + A[:, :, 1::2] ** 2  # noqa: E731
    assert np.allclose(n2(ex), n2(base), rtol=1e-13)
    got = rn.bf16_bits_to_f64(rn.apply(X, g, cos, sin, pos))
    # half a bf16 ulp + the fp32 arithmetic before it (5 roundings of 2^-24, two of them on terms that may cancel)
    assert (np.abs(got - ex) <= np.abs(ex) * 2.0 ** -8 + 8 * 2.0 ** -24 * np.abs(base).max()).all()
    for a, (lo, hi) in enumerate(((0, 44), (44, 86), (86, 128))):
        p2 = list(pos)
        p2[a] = pos[a] + 3
        d = rn.apply(X, g, cos, sin, tuple(p2)) != rn.apply(X, g, cos, sin, pos)
        assert d[:, :, lo:hi].any() and not d[:, :, :lo].any() and not d[:, :, hi:].any()


def test_relative_position_property():
    """<rope(q, p1), rope(k, p2)> depends only on p1 - p2 per axis: shifting both tokens by the same (dt, dy, dx)
    leaves the dot product unchanged (checked on the unrounded complex formulation AND, within bf16 rounding, on
    the oracle's output)."""
    rng = np.random.default_rng(3)
    q = bf16(rng.standard_normal((1, 1, 128)))
    k = bf16(rng.standard_normal((1, 1, 128)))
    g = np.ones(128, dtype=np.float32)
    cos, sin = (t.astype(np.float32) for t in rn.rope_table(64))
    def dot(pq, pk, f):
        a = f(q, g, cos, sin, tuple(np.array([v]) for v in pq))
        b = f(k, g, cos, sin, tuple(np.array([v]) for v in pk))
        return float((a * b).sum())
    ex = lambda *a: _apply_exact(*a)  # noqa: E731
    orc = lambda *a: rn.bf16_bits_to_f64(rn.apply(*a))  # noqa: E731
    d0 = dot((7, 3, 9), (2, 5, 1), ex)
    assert abs(dot((7 + 11, 3 + 4, 9 + 20), (2 + 11, 5 + 4, 1 + 20), ex) - d0) < 1e-4      # fp32 tables
    assert abs(dot((8, 3, 9), (2, 5, 1), ex) - d0) > 1e-3                   # a different offset does change it
    assert abs(dot((18, 7, 29), (13, 9, 21), orc) - dot((7, 3, 9), (2, 5, 1), orc)) < 0.15


def test_round_to_bf16_is_rne_with_ties_and_subnormals():
    """fp32 -> bf16 against the storage-format converter on random values over 40 binades, hand-worked ties (to even,
    both signs), carries into the exponent, and subnormals."""
    rng = np.random.default_rng(4)
    x = (rng.standard_normal(5000) * np.exp(rng.uniform(-20, 20, 5000))).astype(np.float32)
    assert np.array_equal(rn.round_to_bf16(x), wl.f32_to_bf16_bits(x))
    f = np.float32
    cases = [(f(1.0) + f(2.0 ** -8), 0x3F80), (f(1.0) + f(3 * 2.0 ** -8), 0x3F82), (f(1.0 + 2.0 ** -8 + 2.0 ** -20), 0x3F81),
             (-(f(1.0) + f(2.0 ** -8)), 0xBF80), (f(0.0), 0x0000), (f(-0.0), 0x8000), (f(1.9999999), 0x4000),
             (f(2.0 ** -126), 0x0080), (f(2.0 ** -127), 0x0040), (f(2.0 ** -133), 0x0001), (f(2.0 ** -134), 0x0000),
             (f(3 * 2.0 ** -134), 0x0002)]
    for v, bits in cases:
        got = int(rn.round_to_bf16(np.array([v], dtype=np.float32))[0])
        assert got == bits, (float(v), hex(got), hex(bits))
