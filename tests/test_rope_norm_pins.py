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
    g = (1.0 + 0.1 * rng.standard_normal(H * d)).astype(np.float32).astype(np.float64)
    cos, sin = rn.rope_table(64)
    pos = rn.raster_positions(n, gh, gw, t0)
    return X, g, cos, sin, pos


def test_position_zero_is_identity_and_norm_closed_forms():
    """pos = (0,0,0) -> no rotation: the result is bf16(x * r * g); g = 1, eps = 0 -> every token has mean square 1;
    a constant vector c -> c / |c| * g; scaling x by 4 (exact) changes nothing when eps = 0."""
    X, g, cos, sin, _ = _setup(1)
    zero = (np.zeros(12, int),) * 3
    out = rn.bf16_bits_to_f64(rn.apply(X, g, cos, sin, zero))
    r = 1.0 / np.sqrt((X ** 2).reshape(12, -1).mean(axis=1) + 1e-6)
    want = X * r[:, None, None] * g.reshape(1, 2, 128)
    assert np.abs(out - want).max() <= np.abs(want).max() * 2.0 ** -8
    assert np.array_equal(rn.apply(X, g, cos, sin, zero), rn.round_to_bf16(want))
    ones = np.ones(256)
    y = rn.rms_factor(X, eps=0.0)[:, None, None] * X
    assert np.allclose((y ** 2).reshape(12, -1).mean(axis=1), 1.0, atol=1e-14)
    Cst = np.full((3, 2, 128), -2.5)
    zero3 = (np.zeros(3, int),) * 3
    assert np.array_equal(rn.apply(Cst, ones, cos, sin, zero3, eps=0.0), rn.round_to_bf16(np.full((3, 2, 128), -1.0)))
    assert np.array_equal(rn.apply(4.0 * X, g, cos, sin, zero, eps=0.0), rn.apply(X, g, cos, sin, zero, eps=0.0))


def _apply_exact(X, g, cos, sin, pos, eps=1e-6):
    """the same step WITHOUT the final rounding, written with complex numbers (independent formulation)"""
    n, H, d = X.shape
    r = 1.0 / np.sqrt((X ** 2).reshape(n, -1).mean(axis=1) + eps)
    U = X * r[:, None, None] * g.reshape(1, H, d)
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
    ex = _apply_exact(X, g, cos, sin, pos)
    base = _apply_exact(X, g, cos, sin, (0 * pos[0], 0 * pos[1], 0 * pos[2]))
    n2 = lambda A: A[:, :, 0::2] ** 2 + A[:, :, 1::2] ** 2  # noqa: E731
    assert np.allclose(n2(ex), n2(base), rtol=1e-13)
    got = rn.bf16_bits_to_f64(rn.apply(X, g, cos, sin, pos))
    assert (np.abs(got - ex) <= np.abs(ex) * 2.0 ** -8 + 1e-40).all()
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
    g = np.ones(128)
    cos, sin = rn.rope_table(64)
    def dot(pq, pk, f):
        a = f(q, g, cos, sin, tuple(np.array([v]) for v in pq))
        b = f(k, g, cos, sin, tuple(np.array([v]) for v in pk))
        return float((a * b).sum())
    ex = lambda *a: _apply_exact(*a)  # noqa: E731
    orc = lambda *a: rn.bf16_bits_to_f64(rn.apply(*a))  # noqa: E731
    d0 = dot((7, 3, 9), (2, 5, 1), ex)
    assert abs(dot((7 + 11, 3 + 4, 9 + 20), (2 + 11, 5 + 4, 1 + 20), ex) - d0) < 1e-12
    assert abs(dot((8, 3, 9), (2, 5, 1), ex) - d0) > 1e-3                   # a different offset does change it
    assert abs(dot((18, 7, 29), (13, 9, 21), orc) - dot((7, 3, 9), (2, 5, 1), orc)) < 0.15


def test_round_to_bf16_is_rne_with_ties_and_flush():
    """Against the storage-format converter on fp32 values, on hand-worked ties, on a value where rounding first to
    fp32 and then to bf16 would go the other way (double rounding), and on the flush threshold."""
    rng = np.random.default_rng(4)
    x = (rng.standard_normal(5000) * np.exp(rng.uniform(-20, 20, 5000))).astype(np.float32)
    assert np.array_equal(rn.round_to_bf16(x.astype(np.float64)), wl.f32_to_bf16_bits(x))
    cases = [(1.0 + 2.0 ** -8, 0x3F80), (1.0 + 3 * 2.0 ** -8, 0x3F82), (1.0 + 2.0 ** -8 + 2.0 ** -40, 0x3F81),
             (-(1.0 + 2.0 ** -8), 0xBF80), (0.0, 0x0000), (-0.0, 0x8000),
             # 1 + 2^-8 - 2^-30 is BELOW the tie: bf16 1.0; via fp32 first it would become the tie 1 + 2^-8 -> still 1.0;
             # 1 + 2^-8 + 2^-30 is ABOVE the tie: bf16 1 + 2^-7, while fp32-then-bf16 gives the tie -> 1.0 (wrong)
             (1.0 + 2.0 ** -8 + 2.0 ** -30, 0x3F81),
             (1.9999999, 0x4000), (2.0 ** -126, 0x0080), (2.0 ** -127, 0x0000), (-(2.0 ** -126) * 0.9999, 0x8080),
             ((2.0 ** -126) * 0.99, 0x0000)]
    for v, bits in cases:
        assert int(rn.round_to_bf16(np.array([v]))[0]) == bits, (v, hex(int(rn.round_to_bf16(np.array([v]))[0])), hex(bits))


def test_float32_model_of_the_kernel_is_within_one_ulp_of_the_fp64_oracle():
    """The tolerance the GPU test uses (uf_harness.fused_bits_check), exercised on the CPU: a float32 evaluation in the
    kernel's operation order (tests/fused_fp32_model.py — a model of the kernel, not an oracle) stays within one bf16 ulp
    of this oracle and is bit-equal on >= 99 % of the elements; a wrong sign in the rotation, a swapped cos / sin or a
    norm over the head instead of the token is far outside it."""
    import fused_fp32_model as fm
    import uf_harness as hz
    w = wl.scaled(wl.CONFIGS["1k"], "rn_model", n_heads=3, frames_per_chunk=2, grid_h=9, grid_w=14, capacity_chunks=2)
    Qb, _, _ = wl.make_chunk(w, 1)
    X = hz.bits_to_f64(Qb)
    cos, sin = wl.rope_tables(64)
    gq, _ = wl.norm_weights(w)
    pos = rn.raster_positions(X.shape[0], w.grid_h, w.grid_w, 7)
    y = rn.apply_unrounded(X, gq, cos, sin, pos)
    assert np.array_equal(rn.round_to_bf16(y), rn.apply(X, gq, cos, sin, pos))
    eq = hz.fused_bits_check(fm.apply(X, gq, cos, sin, pos), y, "fp32 model")
    assert eq > 0.999
    for wrong in (rn.round_to_bf16(rn.apply_unrounded(X, gq, cos, -sin, pos)),          # rotation the other way
                  rn.round_to_bf16(rn.apply_unrounded(X, gq, sin, cos, pos)),           # tables swapped
                  rn.round_to_bf16(y * 1.01)):                                          # a 1 % scale error
        with pytest.raises(AssertionError):
            hz.fused_bits_check(wrong, y, "wrong")
